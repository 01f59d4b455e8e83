"""Shared helpers of the parity tests: run the CUDA library through its binding, compare with the oracle."""
from __future__ import annotations

from typing import Dict, Optional

import numpy as np

import workloads as W

FLOAT_RTOL = 1e-6  # north_star: "Projected positions and weights must match within 1e-6 relative"


def _np(t, dtype=None):
    a = t.detach().cpu().numpy()
    return a if dtype is None else a.view(dtype)


def library_result(ctx, with_tables: bool = True) -> Dict:
    """everything the latest build produced, as numpy arrays"""
    b = ctx.get_batch(-1, -1)
    out = {"n_survivors": b["count"]}
    for k in ("E", "x", "y", "u", "v", "w", "wt", "xp", "yp"):
        out[k] = None if b[k] is None else _np(b[k])
    out["src_index"] = _np(b["src_index"], np.uint32)
    if with_tables:
        c, o = ctx.get_tables()
        out["counts"], out["offsets"] = _np(c, np.uint32), _np(o, np.uint32)
    out["stats"] = ctx.get_stats()
    return out


def run_library(workload: W.Workload, records: np.ndarray, beam: Optional[Dict], chunk: int = 0, mem: str = "device",
                flags: int = 0, ctx=None, max_records: Optional[int] = None):
    """load `records` in chunks of `chunk` (0 = one chunk) from `mem` in {"device","pinned","pageable"} and build"""
    import torch

    import paper_1302_1861_b200 as P

    n = len(records)
    own = ctx is None
    if own:
        ctx = P.PslContext(workload.grid, workload.geometry, workload.mode, max_records=max_records or max(n, 1),
                           flags=flags)
    raw = np.ascontiguousarray(records).view(np.uint8).reshape(-1)
    step = chunk or max(n, 1)
    for first in range(0, n, step):
        piece = raw[first * 28:min(n, first + step) * 28]
        if mem == "device":
            ctx.load_chunk(torch.from_numpy(piece.copy()).cuda())
        elif mem == "pinned":
            ctx.load_chunk(torch.from_numpy(piece.copy()).pin_memory())
        else:
            ctx.load_chunk(piece.copy())
    ctx.build_batches(beam)
    return ctx


def assert_matches_oracle(lib: Dict, orc: Dict, index_only: bool = False, proj: bool = False):
    """bit-exact for every integer / index / copied field; floats within FLOAT_RTOL (and, as the arithmetic
    contract predicts, bit-equal)."""
    assert lib["n_survivors"] == orc["n_survivors"]
    assert np.array_equal(lib["counts"], orc["counts"])
    assert np.array_equal(lib["offsets"], orc["offsets"])
    assert np.array_equal(lib["src_index"], orc["src_index"])
    for f in ("E", "x", "y", "u", "v"):
        assert np.array_equal(lib[f].view(np.uint32), orc[f].view(np.uint32)), f
    fl = ["wt"] if index_only else ["w", "wt"]
    if proj and not index_only:
        fl += ["xp", "yp"]
    for f in fl:
        a, b = lib[f], orc[{"xp": "xm", "yp": "ym"}.get(f, f)]
        assert np.allclose(a, b, rtol=FLOAT_RTOL, atol=0.0), f
        assert np.array_equal(a.view(np.uint32), b.view(np.uint32)), f + " (bit-equality diagnostic)"
    ls, os_ = lib["stats"], orc["stats"]
    for k in ("n_in", "n_invalid", "n_outside_grid", "n_roi_skipped", "n_jaw_rejected", "n_zero_weight",
              "n_survivors"):
        assert ls[k] == os_[k], k
    for k in ("sum_wt_in", "sum_wt_indexed", "sum_wt_out"):
        if index_only and k == "sum_wt_out":
            continue
        assert abs(ls[k] - os_[k]) <= 1e-9 * max(1.0, abs(os_[k])), k


def dirty(records: np.ndarray, seed: int) -> np.ndarray:
    """sprinkle invalid / out-of-grid records and non-unit weights over generator output"""
    r = records.copy()
    n = len(r)
    rng = np.random.default_rng(seed)
    idx = rng.choice(n, size=max(8, n // 40), replace=False)
    q = len(idx) // 8
    r["type"][idx[:q]] = 5
    r["type"][idx[q:2 * q]] = -1
    r["E"][idx[2 * q:3 * q]] = np.nan
    r["E"][idx[3 * q:4 * q]] = -0.5
    r["x"][idx[4 * q:5 * q]] = 20.0
    r["y"][idx[5 * q:6 * q]] = -np.inf
    r["u"][idx[6 * q:7 * q]] = 1.0
    r["wt"][idx[7 * q:]] = np.inf
    r["wt"][~np.isin(np.arange(n), idx)] = rng.uniform(0.25, 2.0, n - len(idx)).astype(np.float32)
    return r
