"""ctypes wrapper around oracle/psl_oracle.c -- TEST INFRASTRUCTURE ONLY.

Only tests/, ``__graft_entry__.smoke()`` and bench.py's ``cpu_baseline`` / ``--impl reference``
legs may import this.  It does not import, and is not imported by, ``paper_1302_1861_b200``.
It marshals the neutral dicts of ``workloads`` (grid / geometry / beam) into the oracle's own
C structs; argument marshalling only -- every step of the definition runs in psl_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "psl_oracle.c")
_LIB = os.path.join(_HERE, "libpsl_oracle.so")

RECORD_DTYPE = np.dtype(
    [("type", "<i4"), ("E", "<f4"), ("x", "<f4"), ("y", "<f4"), ("u", "<f4"), ("v", "<f4"), ("wt", "<f4")]
)

SURVIVOR, INVALID, OUTSIDE_GRID, ROI_SKIPPED, JAW_REJECTED, ZERO_WEIGHT = range(6)
FLAG_DROP_ZERO_WEIGHT = 2

#: the flags every oracle build uses; -ffp-contract=off is what makes each line one rounding
CFLAGS = ["-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-Wall", "-Wextra"]


class _Config(C.Structure):
    _fields_ = [
        ("n_types", C.c_int32), ("ebin_mode", C.c_int32), ("n_ebins", C.c_int32),
        ("e_min", C.c_float), ("e_max", C.c_float), ("e_edges", C.c_void_p),
        ("n_xbins", C.c_int32), ("n_ybins", C.c_int32),
        ("x_min", C.c_float), ("y_min", C.c_float), ("dx", C.c_float), ("dy", C.c_float),
        ("z_src", C.c_float), ("z_plane", C.c_float), ("z_jaw_x", C.c_float), ("z_jaw_y", C.c_float),
        ("z_map", C.c_float), ("z_iso", C.c_float),
        ("flags", C.c_uint32),
    ]


class _Beam(C.Structure):
    _fields_ = [
        ("has_jaws", C.c_int32),
        ("jaw_x1", C.c_float), ("jaw_x2", C.c_float), ("jaw_y1", C.c_float), ("jaw_y2", C.c_float),
        ("fluence", C.c_void_p), ("map_nx", C.c_int32), ("map_ny", C.c_int32),
        ("map_x0", C.c_float), ("map_y0", C.c_float), ("map_dx", C.c_float), ("map_dy", C.c_float),
        ("has_roi", C.c_int32),
        ("roi_x1", C.c_float), ("roi_x2", C.c_float), ("roi_y1", C.c_float), ("roi_y2", C.c_float),
        ("mu_weight", C.c_float),
        ("gantry_deg", C.c_float), ("coll_deg", C.c_float), ("couch_deg", C.c_float),
    ]


class _Plan(C.Structure):
    _fields_ = [("n_simulate", C.c_uint64), ("seed", C.c_uint64), ("rr_group", C.c_uint32), ("apr", C.c_uint32),
                ("phantom_lo", C.c_float * 3), ("phantom_hi", C.c_float * 3)]


class _EmitStats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("n_list", "n_jaw_rejected", "n_zero_weight", "n_missed", "n_launched")] + \
               [("sum_wt", C.c_double)]


class _Stats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in
                ("n_in", "n_invalid", "n_outside_grid", "n_roi_skipped", "n_jaw_rejected", "n_zero_weight",
                 "n_survivors")] + [(n, C.c_double) for n in ("sum_wt_in", "sum_wt_indexed", "sum_wt_out")]


def build_lib(force: bool = False) -> str:
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if force or stale:
        subprocess.run(["gcc", *CFLAGS, "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"], check=True)
    return _LIB


_lib = None


def use_library(path: Optional[str]) -> None:
    """Load the oracle from another shared object (tests/test_oracle_mutations.py builds deliberately wrong copies
    of psl_oracle.c to check that the pins catch them); None goes back to the real one."""
    global _lib, _override
    _override = path
    _lib = None


_override = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_override or build_lib())
        lib.orc_build.restype = C.c_uint64
        lib.orc_n_keys.restype = C.c_uint32
        lib.orc_bin_width.restype = C.c_float
        lib.orc_jaw_edge.restype = C.c_float
        lib.orc_jaw_edge.argtypes = [C.c_float] * 4
        lib.orc_q.restype = C.c_float
        lib.orc_q.argtypes = [C.c_float, C.c_float]
        lib.orc_w.restype = C.c_float
        lib.orc_w.argtypes = [C.c_float, C.c_float]
        lib.orc_fluence_at.restype = C.c_float
        lib.orc_fluence_at.argtypes = [C.c_void_p, C.c_float, C.c_float]
        lib.orc_mix64.restype = C.c_uint64
        lib.orc_mix64.argtypes = [C.c_uint64]
        lib.orc_rng32.restype = C.c_uint32
        lib.orc_rng32.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64]
        lib.orc_plan_total.restype = C.c_uint64
        lib.orc_sample_batch.restype = C.c_uint64
        lib.orc_emit.restype = C.c_uint64
        lib.orc_flush_schedule.restype = C.c_uint64
        lib.orc_surface.restype = C.c_int
        lib.orc_record_bytes.restype = C.c_uint32
        assert lib.orc_record_bytes() == 28
        _lib = lib
    return _lib


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else C.c_void_p(a.ctypes.data)


class Oracle:
    """The definition, bound to one grid + geometry (+ flags)."""

    def __init__(self, grid: Dict, geometry: Dict, flags: int = 0):
        self.lib = _load()
        g = grid
        self._edges = None
        if g["ebin_mode"] == 1:
            self._edges = np.ascontiguousarray(g["e_edges"], dtype=np.float32)
            assert self._edges.shape[0] == g["n_ebins"] + 1
        self.cfg = _Config(
            g["n_types"], g["ebin_mode"], g["n_ebins"], g["e_min"], g["e_max"],
            None if self._edges is None else self._edges.ctypes.data,
            g["n_xbins"], g["n_ybins"], g["x_min"], g["y_min"], g["dx"], g["dy"],
            geometry["z_src"], geometry["z_plane"], geometry["z_jaw_x"], geometry["z_jaw_y"],
            geometry["z_map"], geometry["z_iso"], flags,
        )
        self.n_keys = int(self.lib.orc_n_keys(C.byref(self.cfg)))
        self._keep = []

    # -- marshalling ----------------------------------------------------------------------
    def beam(self, b: Optional[Dict]):
        if b is None:
            return None
        fl = None
        nx = ny = 0
        if b.get("fluence") is not None:
            fl = np.ascontiguousarray(b["fluence"], dtype=np.float32)
            ny, nx = fl.shape
            self._keep.append(fl)
        j = b.get("jaws")
        r = b.get("roi")
        return _Beam(
            0 if j is None else 1, *(j if j is not None else (0, 0, 0, 0)),
            None if fl is None else fl.ctypes.data, nx, ny,
            b.get("map_x0", 0.0), b.get("map_y0", 0.0), b.get("map_dx", 1.0), b.get("map_dy", 1.0),
            0 if r is None else 1, *(r if r is not None else (0, 0, 0, 0)),
            b.get("mu_weight", 1.0), b.get("gantry_deg", 0.0), b.get("coll_deg", 0.0), b.get("couch_deg", 0.0),
        )

    @staticmethod
    def _rec(records: np.ndarray) -> np.ndarray:
        assert records.dtype == RECORD_DTYPE
        return np.ascontiguousarray(records)

    # -- scalar steps, array forms ---------------------------------------------------------
    def energy_bins(self, E: np.ndarray) -> np.ndarray:
        E = np.ascontiguousarray(E, dtype=np.float32)
        out = np.empty(E.shape[0], dtype=np.int32)
        self.lib.orc_energy_bins(C.byref(self.cfg), _ptr(E), C.c_uint64(E.shape[0]), _ptr(out))
        return out

    def axis_bins(self, x: np.ndarray, origin: float, d: float, nbins: int) -> np.ndarray:
        """bin index per coordinate, -1 outside; used for position bins and map pixels alike"""
        x = np.ascontiguousarray(x, dtype=np.float32)
        out = np.empty(x.shape[0], dtype=np.int32)
        self.lib.orc_axis_bins(_ptr(x), C.c_uint64(x.shape[0]), C.c_float(origin), C.c_float(d), C.c_int32(nbins),
                               _ptr(out))
        return out

    def bin_width(self) -> float:
        return float(self.lib.orc_bin_width(C.byref(self.cfg)))

    def w(self, u: float, v: float) -> float:
        return float(self.lib.orc_w(u, v))

    def q(self, u: float, v: float) -> float:
        return float(self.lib.orc_q(u, v))

    def jaw_edge(self, edge_iso: float, z_jaw: float) -> float:
        return float(self.lib.orc_jaw_edge(edge_iso, z_jaw, self.cfg.z_src, self.cfg.z_iso))

    def jaw_points(self, records: np.ndarray):
        rec = self._rec(records)
        n = rec.shape[0]
        xj = np.empty(n, dtype=np.float32)
        yj = np.empty(n, dtype=np.float32)
        self.lib.orc_jaw_points(C.byref(self.cfg), _ptr(rec), C.c_uint64(n), _ptr(xj), _ptr(yj))
        return xj, yj

    def fluence_at(self, beam: Dict, xm: float, ym: float) -> float:
        b = self.beam(beam)
        return float(self.lib.orc_fluence_at(C.byref(b), xm, ym))

    def roi_bins(self, beam: Dict):
        """(rx0, rx1, ry0, ry1), inclusive; empty selection has rx0 > rx1 or ry0 > ry1"""
        b = self.beam(beam)
        out = (C.c_int32 * 4)()
        self.lib.orc_roi_bins(C.byref(self.cfg), C.byref(b), out)
        return tuple(int(v) for v in out)

    def roi_from_jaws(self, beam: Dict, margin: float):
        b = self.beam(beam)
        out = (C.c_float * 4)()
        rc = self.lib.orc_roi_from_jaws(C.byref(self.cfg), C.byref(b), C.c_float(margin), out)
        return int(rc), tuple(float(v) for v in out)

    def classify(self, records: np.ndarray, beam: Optional[Dict]):
        rec = self._rec(records)
        n = rec.shape[0]
        cls = np.empty(n, dtype=np.uint8)
        keys = np.empty(n, dtype=np.uint32)
        b = self.beam(beam)
        self.lib.orc_classify_all(C.byref(self.cfg), None if b is None else C.byref(b), _ptr(rec), C.c_uint64(n),
                                  _ptr(cls), _ptr(keys))
        return cls, keys

    # -- the whole result -------------------------------------------------------------------
    def build(self, records: np.ndarray, beam: Optional[Dict] = None, want_classes: bool = False) -> Dict:
        """filter, then stable sort by key.  beam=None: method 1 / the PSL index itself."""
        rec = self._rec(records)
        n = rec.shape[0]
        K = self.n_keys
        counts = np.empty(K, dtype=np.uint32)
        offsets = np.empty(K + 1, dtype=np.uint32)
        cap = max(n, 1)
        f = {k: np.empty(cap, dtype=np.float32) for k in ("E", "x", "y", "u", "v", "w", "wt", "xm", "ym")}
        src = np.empty(cap, dtype=np.uint32)
        cls = np.empty(cap, dtype=np.uint8) if want_classes else None
        keys = np.empty(cap, dtype=np.uint32) if want_classes else None
        st = _Stats()
        b = self.beam(beam)
        ns = self.lib.orc_build(
            C.byref(self.cfg), None if b is None else C.byref(b), _ptr(rec), C.c_uint64(n), _ptr(counts),
            _ptr(offsets), *[_ptr(f[k]) for k in ("E", "x", "y", "u", "v", "w", "wt", "xm", "ym")], _ptr(src),
            _ptr(cls), _ptr(keys), C.byref(st),
        )
        ns = int(ns)
        out = {k: v[:ns] for k, v in f.items()}
        out.update(
            counts=counts, offsets=offsets, src_index=src[:ns], n_survivors=ns,
            stats={name: getattr(st, name) for name, _ in _Stats._fields_},
        )
        if want_classes:
            out.update(classes=cls[:n], keys=keys[:n])
        return out

    # -- sampling layer, field transform, APR, capacity-N emission ------------------
    def _beams(self, beams):
        arr = (_Beam * len(beams))(*[self.beam(b) for b in beams])
        return arr

    @staticmethod
    def plan(n_simulate: int, seed: int = 1, rr_group: int = 4, phantom=((-15.0, -15.0, -15.0), (15.0, 15.0, 15.0))):
        p = _Plan(n_simulate, seed, rr_group, 0)
        p.phantom_lo[:] = phantom[0]
        p.phantom_hi[:] = phantom[1]
        return p

    def mix64(self, z: int) -> int:
        return int(self.lib.orc_mix64(C.c_uint64(z & (2 ** 64 - 1))))

    def rng32(self, seed: int, a: int, b: int) -> int:
        return int(self.lib.orc_rng32(C.c_uint64(seed), C.c_uint64(a), C.c_uint64(b)))

    def plan_total(self, beams, counts: np.ndarray) -> int:
        counts = np.ascontiguousarray(counts, dtype=np.uint32)
        return int(self.lib.orc_plan_total(C.byref(self.cfg), self._beams(beams), C.c_uint32(len(beams)), _ptr(counts)))

    def plan_budgets(self, beams, counts: np.ndarray, n_simulate: int):
        """(budget[K], mask[K]): particles to simulate from PSL k for each field that selects it; the fields"""
        counts = np.ascontiguousarray(counts, dtype=np.uint32)
        budget = np.empty(self.n_keys, np.uint32)
        mask = np.empty(self.n_keys, np.uint32)
        self.lib.orc_plan_budgets(C.byref(self.cfg), self._beams(beams), C.c_uint32(len(beams)), _ptr(counts),
                                  C.c_uint64(n_simulate), _ptr(budget), _ptr(mask))
        return budget, mask

    def sample_batch(self, beams, counts, offsets, plan, t: int, ie: int, cap: int):
        counts = np.ascontiguousarray(counts, dtype=np.uint32)
        offsets = np.ascontiguousarray(offsets, dtype=np.uint32)
        slot = np.empty(max(cap, 1), np.uint32)
        beam = np.empty(max(cap, 1), np.uint8)
        n = int(self.lib.orc_sample_batch(C.byref(self.cfg), self._beams(beams), C.c_uint32(len(beams)), _ptr(counts),
                                          _ptr(offsets), C.byref(plan), C.c_int32(t), C.c_int32(ie), _ptr(slot),
                                          _ptr(beam), C.c_uint64(cap)))
        assert n <= cap, "launch list longer than the capacity given"
        return slot[:n], beam[:n]

    def emit(self, beams, plan, index: Dict, slot: np.ndarray, beam_id: np.ndarray) -> Dict:
        """index: the bare index (build(records, None)); slot / beam_id: a launch list"""
        n = len(slot)
        slot = np.ascontiguousarray(slot, np.uint32)
        beam_id = np.ascontiguousarray(beam_id, np.uint8)
        f = {k: np.empty(max(n, 1), np.float32) for k in ("E", "X", "Y", "Z", "U", "V", "W", "wt")}
        src = np.empty(max(n, 1), np.uint32)
        ob = np.empty(max(n, 1), np.uint8)
        st = _EmitStats()
        m = int(self.lib.orc_emit(
            C.byref(self.cfg), self._beams(beams), C.c_uint32(len(beams)), C.byref(plan),
            *[_ptr(np.ascontiguousarray(index[k])) for k in ("E", "x", "y", "u", "v", "wt")],
            _ptr(np.ascontiguousarray(index["src_index"])), _ptr(slot), _ptr(beam_id), C.c_uint64(n),
            *[_ptr(f[k]) for k in ("E", "X", "Y", "Z", "U", "V", "W", "wt")], _ptr(src), _ptr(ob), C.byref(st)))
        out = {k: v[:m] for k, v in f.items()}
        out.update(src_index=src[:m], beam=ob[:m], n_launched=m,
                   stats={name: getattr(st, name) for name, _ in _EmitStats._fields_})
        return out

    def beam_matrix(self, beam: Dict) -> np.ndarray:
        b = self.beam(beam)
        m = (C.c_float * 9)()
        self.lib.orc_beam_matrix(C.byref(b), m)
        return np.array(m, dtype=np.float32).reshape(3, 3)

    def rotate(self, M: np.ndarray, v) -> np.ndarray:
        m = (C.c_float * 9)(*np.asarray(M, np.float32).reshape(-1))
        a = (C.c_float * 3)(*v)
        o = (C.c_float * 3)()
        self.lib.orc_rotate(m, a, o)
        return np.array(o, dtype=np.float32)

    def surface(self, P, D, lo, hi):
        a, d, l, h, o = [(C.c_float * 3)(*v) for v in (P, D, lo, hi, (0, 0, 0))]
        hit = int(self.lib.orc_surface(a, d, l, h, o))
        return hit, np.array(o, dtype=np.float32)

    def apr_cos_sin(self, r: int):
        c, s_ = C.c_float(), C.c_float()
        self.lib.orc_apr_cos_sin(C.c_uint32(r), C.byref(c), C.byref(s_))
        return c.value, s_.value

    def apr(self, seed: int, records: np.ndarray, first_index: int = 0) -> np.ndarray:
        rec = self._rec(records)
        out = np.empty_like(rec)
        self.lib.orc_apr_all(C.c_uint64(seed), C.c_uint64(first_index), _ptr(rec), C.c_uint64(len(rec)), _ptr(out))
        return out

    def flush_schedule(self, build: Dict, capacity: int):
        """events (key, first slot, count) of the capacity-N emission for a build made with want_classes=True"""
        n = len(build["classes"])
        cap = n // max(capacity, 1) + self.n_keys + 1
        ek, ef, ec = (np.empty(cap, np.uint32) for _ in range(3))
        ne = int(self.lib.orc_flush_schedule(C.c_uint32(self.n_keys), C.c_uint64(n), _ptr(np.ascontiguousarray(build["classes"])),
                                             _ptr(np.ascontiguousarray(build["keys"])),
                                             _ptr(np.ascontiguousarray(build["offsets"])), C.c_uint32(capacity), _ptr(ek),
                                             _ptr(ef), _ptr(ec), C.c_uint64(cap)))
        return ek[:ne], ef[:ne], ec[:ne]
