"""-m gpu: psl_count_static, the entry point that allocates nothing (include/psl.h), against the existing path
(psl_create + psl_load_chunk + psl_build_batches(NULL) + psl_get_tables) on the same records: counts[K] and the
class totals are integers, so the bar is bit-exact.  Collected last on purpose (the file name): the suite runs
with pytest -x."""
import ctypes as C

import numpy as np
import pytest

import workloads as W
from helpers import dirty
from oracle import psl_oracle as O

pytestmark = pytest.mark.gpu


def _grids():
    edges16 = W.log_edges(0.01, 6.0, 16)
    return {
        # the largest key space the static scratch takes: 2 x 16 x 8 x 8 = 2048 keys, energy edges, position bins
        "pos_edges_2048": W._grid(n_types=2, ebin_mode=W.EBIN_EDGES, n_ebins=16, e_min=0.01, e_max=6.0, e_edges=edges16,
                                  n_xbins=8, n_ybins=8, x_min=-20.0, y_min=-20.0, dx=5.0, dy=5.0),
        "pos_linear_1536": W._grid(n_types=3, n_ebins=8, n_xbins=8, n_ybins=8, x_min=-16.0, y_min=-16.0, dx=4.0, dy=4.0),
        "cfg2_linear_192": W.config(2).grid,
        "cfg1_edges_96": W.config(1).grid,
    }


def _existing_path(P, grid, geometry, dev_records, n):
    """counts[K] and statistics through a context, the path every other test covers"""
    ctx = P.PslContext(grid, geometry, P.MODE_ONTHEFLY, max_records=max(n, 1), max_host_records=0)
    if n:
        ctx.load_chunk(dev_records)
    st = ctx.build_batches(None, want_stats=True)
    counts, _ = ctx.get_tables()
    out = counts.clone()
    ctx.destroy()
    return out, st


def _device_records(torch, r, shift=0):
    """packed records on the device; shift = bytes the buffer starts past a 256-byte boundary"""
    raw = torch.from_numpy(np.ascontiguousarray(r).view(np.uint8).reshape(-1).copy())
    buf = torch.empty(raw.numel() + 256, dtype=torch.uint8, device="cuda")
    view = buf[shift:shift + raw.numel()]
    view.copy_(raw)
    return view


def test_two_calls_in_a_row_match_the_existing_path():
    import torch

    import paper_1302_1861_b200 as P

    g = _grids()
    geom = W.config(2).geometry
    # first call: 2048 keys, 684 tiles (every CTA of the wave has a column), ragged tail; second call straight behind it on
    # the same stream: fewer keys, 49 tiles = fewer columns -- whatever the first call left in the scratch must not show
    ra = dirty(W.generate(W.GenParams(4201), 0, 700_003), 7)
    rb = dirty(W.generate(W.GenParams(4202, half_x=6.0, half_y=6.0), 0, 50_001), 8)
    da, db = _device_records(torch, ra), _device_records(torch, rb)
    ca = torch.full((2048,), -1, dtype=torch.int32, device="cuda")
    cb = torch.full((192,), -1, dtype=torch.int32, device="cuda")
    ta = torch.full((4,), -1, dtype=torch.int64, device="cuda")
    tb = torch.full((4,), -1, dtype=torch.int64, device="cuda")
    P.count_static(g["pos_edges_2048"], geom, da, ca, ta)  # also the first call on this device: set-up
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    P.count_static(g["pos_edges_2048"], geom, da, ca, ta)
    P.count_static(g["cfg2_linear_192"], geom, db, cb, tb)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before  # nothing was allocated on the device
    for grid, r, dev, c, t in ((g["pos_edges_2048"], ra, da, ca, ta), (g["cfg2_linear_192"], rb, db, cb, tb)):
        ref, st = _existing_path(P, grid, geom, dev, len(r))
        assert torch.equal(c, ref)
        assert t.tolist() == [len(r), st["n_invalid"], st["n_outside_grid"], st["n_survivors"]]
        assert int(c.sum()) == st["n_survivors"] > 0
        orc = O.Oracle(grid, geom).build(r, None)  # and, beyond the brief, the oracle's counts
        assert np.array_equal(c.cpu().numpy().view(np.uint32), orc["counts"])
    # and once more in the opposite order, reusing the outputs
    P.count_static(g["cfg2_linear_192"], geom, db, cb, tb)
    P.count_static(g["pos_edges_2048"], geom, da, ca, ta)
    torch.cuda.synchronize()
    assert torch.equal(ca, _existing_path(P, g["pos_edges_2048"], geom, da, len(ra))[0])
    assert torch.equal(cb, _existing_path(P, g["cfg2_linear_192"], geom, db, len(rb))[0])


@pytest.mark.parametrize("name", ["pos_edges_2048", "pos_linear_1536", "cfg2_linear_192", "cfg1_edges_96"])
@pytest.mark.parametrize("n,shift", [(0, 0), (3, 0), (1024, 0), (40_001, 4), (333_333, 0)])
def test_every_kernel_variant_and_buffer_shape(name, n, shift):
    import torch

    import paper_1302_1861_b200 as P

    grid = _grids()[name]
    geom = W.config(2).geometry
    r = dirty(W.generate(W.GenParams(4300 + n % 97), 0, n), 3) if n >= 64 else W.generate(W.GenParams(4300), 0, n)
    dev = _device_records(torch, r, shift)  # shift = 4: not 16-byte aligned, the tiles are fetched without TMA
    K = grid["n_types"] * grid["n_ebins"] * grid["n_xbins"] * grid["n_ybins"]
    c = torch.full((K,), -1, dtype=torch.int32, device="cuda")
    t = torch.full((4,), -1, dtype=torch.int64, device="cuda")
    P.count_static(grid, geom, dev, c, t)
    torch.cuda.synchronize()
    if shift:
        ref, st = _existing_path(P, grid, geom, _device_records(torch, r, 0), n)
    else:
        ref, st = _existing_path(P, grid, geom, dev, n)
    assert torch.equal(c, ref)
    assert t.tolist() == [n, st["n_invalid"], st["n_outside_grid"], st["n_survivors"]]


def test_limits_are_rejected_with_a_clear_error():
    import torch

    import paper_1302_1861_b200 as P
    from paper_1302_1861_b200 import binding as B

    geom = W.config(2).geometry
    lib = P.load_library()
    dev = _device_records(torch, W.generate(W.GenParams(1), 0, 1024))
    c = torch.zeros(4096, dtype=torch.int32, device="cuda")
    big = W._grid(n_types=3, n_ebins=64, n_xbins=4, n_ybins=4, dx=10.0, dy=10.0)  # 3072 keys > 2048
    cfg, _keep = B.make_config(big, geom, P.MODE_ONTHEFLY, 1, 0)
    rc = lib.psl_count_static(C.byref(cfg), dev.data_ptr(), 1024, c.data_ptr(), None)
    assert rc == 3 and b"at most 2048" in lib.psl_last_error(None)
    ok = _grids()["cfg2_linear_192"]
    cfg, _keep = B.make_config(ok, geom, P.MODE_ONTHEFLY, 1, 0)
    rc = lib.psl_count_static(C.byref(cfg), dev.data_ptr(), 1 << 32, c.data_ptr(), None)
    assert rc == 3 and b"2^32" in lib.psl_last_error(None)
    assert lib.psl_count_static(C.byref(cfg), dev.data_ptr(), 1024, None, None) == 1       # counts is NULL
    assert lib.psl_count_static(C.byref(cfg), dev.data_ptr() + 2, 1024, c.data_ptr(), None) == 1  # misaligned records
    cfg.n_types = 4
    assert lib.psl_count_static(C.byref(cfg), dev.data_ptr(), 1024, c.data_ptr(), None) == 1  # psl_create's checks
    torch.cuda.synchronize()
    assert int(c.sum()) == 0  # a rejected call enqueues nothing


def test_the_call_can_be_captured_into_a_cuda_graph():
    """what the entry point is for: under stream capture nothing may allocate or synchronise.  Captured once (after a
    first, uncaptured call has done the per-device set-up), replayed on new contents of the same buffers."""
    import torch

    import paper_1302_1861_b200 as P

    grid = _grids()["pos_edges_2048"]
    geom = W.config(2).geometry
    n = 200_003
    ra = dirty(W.generate(W.GenParams(4401), 0, n), 1)
    rb = dirty(W.generate(W.GenParams(4402, half_x=6.0, half_y=6.0), 0, n), 2)
    dev = _device_records(torch, ra)
    counts = torch.full((2048,), -1, dtype=torch.int32, device="cuda")
    totals = torch.full((4,), -1, dtype=torch.int64, device="cuda")
    P.count_static(grid, geom, dev, counts, totals)  # set-up happens here, outside the capture
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        P.count_static(grid, geom, dev, counts, totals)  # enqueued on the capturing stream (torch's current stream)
    for r in (ra, rb, ra):
        dev.copy_(torch.from_numpy(np.ascontiguousarray(r).view(np.uint8).reshape(-1).copy()))
        counts.fill_(-1)
        g.replay()
        torch.cuda.synchronize()
        ref, st = _existing_path(P, grid, geom, dev, n)
        assert torch.equal(counts, ref)
        assert totals.tolist() == [n, st["n_invalid"], st["n_outside_grid"], st["n_survivors"]]
