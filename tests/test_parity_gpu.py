"""-m gpu: the CUDA path (through the C-ABI, via the thin binding) against the CPU oracle, element by element,
on the same seeded inputs.  Bit-exact for counts, offsets, permutation (src_index), survivor set and every
copied field; floats within 1e-6 relative (north_star) -- and, per the arithmetic contract, bit-equal."""
import numpy as np
import pytest

import workloads as W
from helpers import assert_matches_oracle, dirty, library_result, run_library
from oracle import psl_oracle as O

pytestmark = pytest.mark.gpu


def P():
    import paper_1302_1861_b200 as P_

    return P_


def check(w, r, beam, chunk=0, mem="device", flags=0, proj=False):
    ctx = run_library(w, r, beam, chunk=chunk, mem=mem, flags=flags)
    lib = library_result(ctx)
    orc = O.Oracle(w.grid, w.geometry, flags=flags & 2).build(r, beam)
    assert_matches_oracle(lib, orc, proj=proj)
    ctx.destroy()
    return lib


# ---------------------------------------------------------------------------------------------
# ONTHEFLY (methods 1 and 2): configs 1-3
# ---------------------------------------------------------------------------------------------
def test_config1_tiny_open_field_full_size():
    w = W.config(1)
    r = w.records()
    lib = check(w, r, w.beams[0])
    assert 100 < lib["n_survivors"] < 600  # 4x4 field at isocentre = +-1 cm on the 40x40 plane


def test_config1_variants_no_jaws_and_zero_projection_distance():
    w = W.config(1)
    r = w.records()
    check(w, r, None)
    check(w, r, W.make_beam(jaws=(-100, 100, -100, 100), mu_weight=0.25))
    flat = dict(z_src=-100.0, z_plane=0.0, z_jaw_x=0.0, z_jaw_y=0.0, z_map=0.0, z_iso=0.0)
    w0 = W.Workload("cfg1_flat", w.n_records, w.gen, w.mode, w.grid, geometry=flat, beams=w.beams)
    lib = check(w0, r, w.beams[0])
    keep = (r["x"] >= -2) & (r["x"] < 2) & (r["y"] >= -2) & (r["y"] < 2)
    assert lib["n_survivors"] == int(keep.sum())


@pytest.mark.parametrize("mem", ["device", "pinned", "pageable"])
def test_config2_chunked_equals_oracle(mem):
    w = W.config(2, 300_000)
    r = w.records()
    check(w, r, None, chunk=w.chunk_records, mem=mem)


def test_chunking_does_not_change_a_single_byte():
    w = W.config(2, 12_000)
    r = dirty(w.records(), 1)
    ref = library_result(run_library(w, r, None, chunk=0))
    for chunk in (4, 1000, 2048, 4096 + 4, 11_996):
        got = library_result(run_library(w, r, None, chunk=chunk, max_records=len(r)))
        for k in ("counts", "offsets", "src_index", "E", "x", "y", "u", "v", "w", "wt"):
            assert np.array_equal(ref[k].view(np.uint32), got[k].view(np.uint32)), (chunk, k)
        assert ref["stats"] == got["stats"], chunk


def test_config3_jaws_and_fluence_map():
    w = W.config(3, 400_000)
    r = dirty(w.records(), 3)
    lib = check(w, r, w.beams[0], flags=1, proj=True)
    f = lib["n_survivors"] / len(r)
    assert 0.10 < f < 0.16  # (15/40)^2 = 14 %


def test_zero_weight_policy():
    w = W.config(3, 200_000)
    r = w.records()
    m = W.fluence_uniform(5)
    m[:, :80] = 0.0
    beam = W.make_beam(jaws=(-15, 15, -15, 15), fluence=m, mu_weight=0.5)
    kept = check(w, r, beam)
    assert (kept["wt"] == 0).any()
    dropped = check(w, r, beam, flags=2)
    assert dropped["stats"]["n_zero_weight"] == int((kept["wt"] == 0).sum())


def test_two_type_divisions_and_asymmetric_jaws():
    w = W.config(3, 150_000)
    g2 = dict(w.grid, n_types=2, n_ebins=10)
    w2 = W.Workload("two_types", w.n_records, w.gen, w.mode, g2)
    r = dirty(w2.records(), 8)
    check(w2, r, W.make_beam(jaws=(2.0, 14.0, -12.0, -4.0), fluence=W.fluence_uniform(2), mu_weight=1.0 / 3.0))


def test_many_keys_in_one_pass():
    w = W.config(3, 120_000)
    g = dict(w.grid, n_ebins=600)  # 1800 keys: close to the single-pass limit
    w2 = W.Workload("many_keys", w.n_records, w.gen, w.mode, g)
    check(w2, w2.records(), W.make_beam(jaws=(-20, 20, -20, 20)))


@pytest.mark.parametrize("n", [0, 1, 3, 4, 5, 2047, 2048, 2049, 4100])
def test_ragged_and_empty_inputs(n):
    w = W.config(2, max(n, 1))
    r = dirty(w.records(), n)[:n] if n >= 8 else w.records()[:n]
    check(w, r, None)
    w3 = W.config(3, max(n, 1))
    check(w3, w3.records()[:n], w3.beams[0])


def test_everything_rejected():
    w = W.config(3, 10_000)
    r = w.records()
    lib = check(w, r, W.make_beam(jaws=(50, 51, 50, 51)))
    assert lib["n_survivors"] == 0 and lib["stats"]["n_jaw_rejected"] == len(r)
    bad = r.copy()
    bad["type"] = 9
    lib = check(w, bad, None)
    assert lib["stats"]["n_invalid"] == len(r)


def test_rebuild_with_another_beam_and_run_to_run_determinism():
    w = W.config(3, 100_000)
    r = w.records()
    ctx = run_library(w, r, w.beams[0], chunk=30_000)
    a = library_result(ctx)
    ctx.build_batches(W.make_beam(jaws=(-3, 3, -3, 3)))
    b = library_result(ctx)
    assert_matches_oracle(b, O.Oracle(w.grid, w.geometry).build(r, W.make_beam(jaws=(-3, 3, -3, 3))))
    ctx.build_batches(w.beams[0])
    c = library_result(ctx)
    for k in ("counts", "offsets", "src_index", "w", "wt"):
        assert np.array_equal(a[k].view(np.uint32), c[k].view(np.uint32))
    assert a["stats"] == c["stats"]  # including the double sums: fixed-order reductions
    ctx.reset()
    ctx.load_chunk(__import__("torch").from_numpy(r[:5000].view(np.uint8).reshape(-1).copy()).cuda())
    ctx.build_batches(None)
    assert_matches_oracle(library_result(ctx), O.Oracle(w.grid, w.geometry).build(r[:5000], None))
    ctx.destroy()


def test_per_batch_views():
    w = W.config(2, 50_000)
    r = w.records()
    ctx = run_library(w, r, None)
    orc = O.Oracle(w.grid, w.geometry).build(r, None)
    total = 0
    for t in range(3):
        for ie in (0, 5, 17, 63):
            b = ctx.get_batch(t, ie)
            k = t * 64 + ie
            assert b["first"] == orc["offsets"][k] and b["count"] == orc["counts"][k]
            got = b["src_index"].cpu().numpy().view(np.uint32)
            assert np.array_equal(got, orc["src_index"][orc["offsets"][k]:orc["offsets"][k + 1]])
            assert np.array_equal(b["bin_offsets"].cpu().numpy().view(np.uint32), orc["offsets"][k:k + 2])
            total += b["count"]
    assert total > 0
    ctx.destroy()


# ---------------------------------------------------------------------------------------------
# INDEX (method 3, the PSL method): configs 4 and 5
# ---------------------------------------------------------------------------------------------
def index_result(ctx):
    lib = library_result(ctx)
    return lib


def test_config4_index_then_beam():
    w = W.config(4, 500_000)
    r = dirty(w.records(), 4)
    ctx = run_library(w, r, None, chunk=120_000)
    orc = O.Oracle(w.grid, w.geometry)
    assert_matches_oracle(library_result(ctx), orc.build(r, None), index_only=True)
    ctx.build_batches(w.beams[0])
    lib = library_result(ctx)
    assert_matches_oracle(lib, orc.build(r, w.beams[0]))
    assert ctx.roi_bins(w.beams[0]) == (28, 51, 28, 51) == orc.roi_bins(w.beams[0])
    assert lib["stats"]["n_roi_skipped"] > 0.85 * len(r)
    # per-batch view with position-bin offsets
    o = orc.build(r, w.beams[0])
    b = ctx.get_batch(0, 5)
    k0 = 5 * 6400
    assert b["first"] == o["offsets"][k0] and b["count"] == o["offsets"][k0 + 6400] - o["offsets"][k0]
    assert np.array_equal(b["bin_offsets"].cpu().numpy().view(np.uint32), o["offsets"][k0:k0 + 6401])
    ctx.destroy()


def test_index_roi_edge_cases():
    w = W.config(4, 200_000)
    r = w.records()
    ctx = run_library(w, r, None)
    orc = O.Oracle(w.grid, w.geometry)
    beams = [
        W.make_beam(jaws=(-5, 5, -5, 5), roi=(-20, 20, -20, 20)),            # whole plane
        W.make_beam(jaws=(-5, 5, -5, 5)),                                    # no ROI at all
        W.make_beam(jaws=(-5, 5, -5, 5), roi=(3.0, 3.0, -20, 20)),           # zero-width ROI: nothing
        W.make_beam(jaws=(-5, 5, -5, 5), roi=(50, 60, 50, 60)),              # off the plane
        W.make_beam(roi=(-0.5, 0.5, 0.0, 0.5)),                              # ROI only, edges on bin edges
        W.make_beam(jaws=(-40, 40, -40, 40), roi=(-7.3, 2.2, 1.1, 19.9), fluence=W.fluence_uniform(9), mu_weight=0.125),
        W.make_beam(jaws=(1, 9, -9, -1), roi=(-25, 25, -25, 25)),
    ]
    for beam in beams:
        ctx.build_batches(beam)
        if beam["roi"] is not None:
            ls, os_ = ctx.roi_bins(beam), orc.roi_bins(beam)
            empty = lambda s: s[0] > s[1] or s[2] > s[3]  # noqa: E731
            assert ls == os_ or (empty(ls) and empty(os_))
        assert_matches_oracle(library_result(ctx), orc.build(r, beam))
    ctx.destroy()


def test_index_with_drop_zero_weight_and_projection_outputs():
    w = W.config(4, 150_000)
    r = w.records()
    m = W.fluence_uniform(6)
    m[80:, :] = 0.0
    beam = W.make_beam(jaws=(-8, 8, -8, 8), fluence=m, roi=(-6, 6, -6, 6))
    ctx = run_library(w, r, beam, flags=3)
    assert_matches_oracle(library_result(ctx), O.Oracle(w.grid, w.geometry, flags=2).build(r, beam), proj=True)
    ctx.destroy()


@pytest.mark.parametrize("mem", ["pinned", "pageable", "device"])
def test_config5_streamed_imrt_beams(mem):
    w = W.config(5, 700_000)
    r = w.records()
    ctx = run_library(w, r, None, chunk=w.chunk_records, mem=mem)
    orc = O.Oracle(w.grid, w.geometry)
    assert_matches_oracle(library_result(ctx), orc.build(r, None), index_only=True)
    for beam in w.beams:
        ctx.build_batches(beam)
        assert_matches_oracle(library_result(ctx), orc.build(r, beam))
    ctx.destroy()


def test_paper_sized_psl_grid_two_types():
    # 20x20 cm^2, 1-cm bins, 10 energy bins, 2 type divisions = 8000 PSLs
    g = W._grid(n_types=2, n_ebins=10, n_xbins=20, n_ybins=20, x_min=-10.0, y_min=-10.0, dx=1.0, dy=1.0)
    w = W.Workload("paper_psl", 300_000, W.GenParams(77), W.MODE_INDEX, g)
    r = dirty(w.records(), 6)
    beam = W.make_beam(jaws=(-5, 5, -5, 5), roi=(-3.2, 3.2, -3.2, 3.2), fluence=W.fluence_uniform(1))
    ctx = run_library(w, r, None)
    orc = O.Oracle(g, w.geometry)
    assert_matches_oracle(library_result(ctx), orc.build(r, None), index_only=True)
    ctx.build_batches(beam)
    assert_matches_oracle(library_result(ctx), orc.build(r, beam))
    ctx.destroy()


@pytest.mark.parametrize("n", [0, 1, 5, 2049])
def test_index_ragged_and_empty(n):
    w = W.config(4, max(n, 1))
    r = w.records()[:n]
    ctx = run_library(w, r, None)
    orc = O.Oracle(w.grid, w.geometry)
    assert_matches_oracle(library_result(ctx), orc.build(r, None), index_only=True)
    ctx.build_batches(w.beams[0])
    assert_matches_oracle(library_result(ctx), orc.build(r, w.beams[0]))
    ctx.destroy()


# ---------------------------------------------------------------------------------------------
# error behaviour
# ---------------------------------------------------------------------------------------------
def test_error_codes():
    import torch

    p = P()
    w = W.config(4, 10_000)
    r = w.records()
    raw = torch.from_numpy(r.view(np.uint8).reshape(-1).copy()).cuda()
    ctx = p.PslContext(w.grid, w.geometry, w.mode, max_records=10_000, max_beam_records=16)
    with pytest.raises(p.PslError) as e:
        ctx.get_batch(0, 0)
    assert e.value.status_name == "PSL_ERR_STATE"
    ctx.load_chunk(raw)
    with pytest.raises(p.PslError) as e:
        ctx.load_chunk(raw[:28 * 4])
    assert e.value.status_name == "PSL_ERR_CAPACITY"
    ctx.build_batches(None)
    with pytest.raises(p.PslError) as e:
        ctx.load_chunk(raw[:28 * 4])
    assert e.value.status_name == "PSL_ERR_STATE"
    with pytest.raises(p.PslError) as e:
        ctx.build_batches(w.beams[0])  # ROI selects far more than max_beam_records = 16
    assert e.value.status_name == "PSL_ERR_CAPACITY"
    with pytest.raises(p.PslError) as e:
        ctx.get_batch(3, 0)
    assert e.value.status_name == "PSL_ERR_ARG"
    ctx.destroy()
    w2 = W.config(2, 1000)
    ctx = p.PslContext(w2.grid, w2.geometry, w2.mode, max_records=1000)
    ctx.load_chunk(raw[:28 * 6])  # 6 records: not a multiple of 4 -> must be the last chunk
    with pytest.raises(p.PslError) as e:
        ctx.load_chunk(raw[:28 * 4])
    assert e.value.status_name == "PSL_ERR_ARG"
    with pytest.raises(p.PslError) as e:
        ctx.build_batches(W.make_beam(roi=(-1, 1, -1, 1)))  # ROI needs the index
    assert e.value.status_name == "PSL_ERR_ARG"
    ctx.destroy()


# ---------------------------------------------------------------------------------------------
# full size, in the launch configuration bench.py times (config 2: 1e7 records, ten 1e6-record device chunks)
# ---------------------------------------------------------------------------------------------
def test_config2_full_size_element_by_element():
    w = W.config(2)
    r = w.records()
    check(w, r, None, chunk=w.chunk_records, mem="device")


# ---------------------------------------------------------------------------------------------
# kernel-structure cases: stage rings that wrap, tiles that straddle nothing but are ragged, sources TMA cannot
# copy, both ONTHEFLY tile sizes, the INDEX digit split near its limits
# ---------------------------------------------------------------------------------------------
def test_big_tiles_ragged_chunks_and_ring_wraparound():
    """config-2 keys (192 <= 256: the 4096-record-tile scatter); chunks of 3000 records leave a ragged 952-record
    ring stage after every two full ones, and 2.4e6 records give every persistent CTA several big tiles, so ring
    stages and their barriers are reused with both parities."""
    w = W.config(2, 2_400_000)
    r = dirty(w.records(), 7)
    check(w, r, None, chunk=3000 * 40, mem="device")
    w_small = W.config(2, 70_001)
    check(w_small, dirty(w_small.records(), 8), None, chunk=3000, mem="device")


def test_small_tiles_with_a_rejecting_beam_at_scale():
    """a beam with jaws and the survivor compaction switched off (PSL_NO_COMPACT) takes the 1024-record-tile scatter
    (two CTAs per SM), which ranks from the histogram kernel's one byte per record; several tiles per CTA"""
    w = W.config(3, 1_500_000)
    check(w, w.records(), w.beams[0], chunk=500_000, mem="device", flags=P().OUT_PROJ | P().NO_COMPACT, proj=True)


def test_compacted_survivors_at_scale_and_against_the_other_path():
    """a beam with jaws and K <= 256: the histogram kernel compacts the survivors per segment and the scatter reads
    only those (psl_compact.cuh).  Against the oracle, and byte for byte against the path without compaction."""
    w = W.config(3, 1_500_000)
    r = dirty(w.records(), 11)
    a = check(w, r, w.beams[0], chunk=500_000, mem="device", flags=P().OUT_PROJ, proj=True)
    b = library_result(run_library(w, r, w.beams[0], chunk=500_000, mem="device", flags=P().OUT_PROJ | P().NO_COMPACT))
    for k in ("counts", "offsets", "src_index", "E", "x", "y", "u", "v", "w", "wt", "xp", "yp"):
        assert np.array_equal(a[k].view(np.uint32), b[k].view(np.uint32)), k
    assert a["stats"] == b["stats"]


def test_compacted_survivors_when_every_record_survives():
    """jaws wider than the whole phase-space: a rejecting beam that rejects nothing.  Every warp of the histogram
    kernel compacts all 128 of its records, every region is full, and the scatter's 4096-survivor tiles straddle
    the regions of the two histogram CTAs per segment; ragged chunks leave ragged tiles in between."""
    w = W.config(2, 2_400_000)
    r = w.records()
    lib = check(w, r, W.make_beam(jaws=(-20, 20, -20, 20)), chunk=3000 * 40, mem="device")
    assert lib["n_survivors"] == len(r)
    w_small = W.config(2, 70_001)
    check(w_small, dirty(w_small.records(), 9), W.make_beam(jaws=(-20, 20, -20, 20), mu_weight=0.25), chunk=3000, mem="device")


def test_compacted_survivors_sparse_and_with_the_zero_weight_policy():
    """few survivors (config 1: 0.25 %): most segments compact nothing and their scatter CTAs have no tile; and the
    zero-weight policy, which rejects after the fluence lookup"""
    w = W.config(1)
    check(w, dirty(w.records(), 12), w.beams[0], chunk=10_000, mem="device")
    w3 = W.config(3, 600_000)
    m = W.fluence_uniform(6)
    m[40:120, :] = 0.0
    check(w3, w3.records(), W.make_beam(jaws=(-15, 15, -15, 15), fluence=m, mu_weight=0.5), chunk=0, mem="pinned", flags=2)


def test_unaligned_device_source_takes_the_manual_stage_fill():
    """a DEVICE chunk that is only 4-byte aligned cannot be bulk-copied: every stage is fetched by the threads"""
    import torch

    p = P()
    w = W.config(2, 20_000)
    r = w.records()
    raw = np.ascontiguousarray(r).view(np.uint8).reshape(-1)
    buf = torch.empty(len(raw) + 4, dtype=torch.uint8, device="cuda")
    buf[4:].copy_(torch.from_numpy(raw.copy()))
    for grid, beam in ((w.grid, None), (W.config(3, 1).grid, W.config(3, 1).beams[0])):
        ctx = p.PslContext(grid, w.geometry, w.mode, max_records=len(r))
        ctx.load_chunk(buf[4:], p.MEM_DEVICE)
        ctx.build_batches(beam)
        assert_matches_oracle(library_result(ctx), O.Oracle(grid, w.geometry).build(r, beam))
        ctx.destroy()
    w4 = W.config(4, 20_000)
    ctx = p.PslContext(w4.grid, w4.geometry, w4.mode, max_records=len(r))
    r4 = w4.records()
    buf[4:].copy_(torch.from_numpy(np.ascontiguousarray(r4).view(np.uint8).reshape(-1).copy()))
    ctx.load_chunk(buf[4:], p.MEM_DEVICE)
    ctx.build_batches(w4.beams[0])
    assert_matches_oracle(library_result(ctx), O.Oracle(w4.grid, w4.geometry).build(r4, w4.beams[0]))
    ctx.destroy()


def test_index_at_scale_many_segments_then_bare_index_and_beam():
    """3e6 records: every persistent CTA of both INDEX passes owns several tiles; the bare index (SoA view made
    on demand from the keyed records) and a beam build from the same index"""
    w = W.config(4, 3_000_000)
    r = dirty(w.records(), 11)
    ctx = run_library(w, r, None, chunk=1_000_000, mem="device")
    orc = O.Oracle(w.grid, w.geometry)
    assert_matches_oracle(library_result(ctx), orc.build(r, None), index_only=True)
    ctx.build_batches(w.beams[0])
    assert_matches_oracle(library_result(ctx), orc.build(r, w.beams[0]))
    ctx.build_batches(None)  # back to the bare index: the view is still valid
    assert_matches_oracle(library_result(ctx), orc.build(r, None), index_only=True)
    ctx.destroy()


def test_index_digit_split_extremes():
    """few keys (one digit does all the work) and close to the 2048 x 2048 limit"""
    w = W.config(4, 40_000)
    tiny = dict(w.grid, n_ebins=1, n_xbins=2, n_ybins=2, x_min=-20.0, dx=20.0, y_min=-20.0, dy=20.0)  # 12 keys
    wt = W.Workload("idx_tiny", w.n_records, w.gen, w.mode, tiny)
    r = wt.records()
    ctx = run_library(wt, r, None)
    assert_matches_oracle(library_result(ctx), O.Oracle(tiny, w.geometry).build(r, None), index_only=True)
    ctx.destroy()
    huge = dict(w.grid, n_ebins=100, n_xbins=100, n_ybins=100, x_min=-20.0, dx=0.4, y_min=-20.0, dy=0.4)  # 3e6 keys
    wh = W.Workload("idx_huge", w.n_records, w.gen, w.mode, huge)
    beam = W.make_beam(jaws=(-8, 8, -8, 8), roi=(-5, 5, -5, 5))
    ctx = run_library(wh, r, beam)
    assert_matches_oracle(library_result(ctx), O.Oracle(huge, w.geometry).build(r, beam))
    ctx.destroy()


def test_config3_full_size_element_by_element():
    """config 3 as bench.py times it: 5e7 records, jaws 30x30 at isocentre, 160x160 fluence map, one device chunk"""
    w = W.config(3)
    r = w.records()
    check(w, r, w.beams[0], mem="device")


def test_config4_full_size_index_and_beam():
    """config 4 as bench.py times it: 2e8 records -> PSL index over 1 228 800 keys -> the 10x10 beam with its ROI.
    The whole index (counts, offsets, permutation, copied fields) and the beam's batches against the oracle."""
    w = W.config(4)
    r = w.records()
    orc = O.Oracle(w.grid, w.geometry)
    ctx = run_library(w, r, None, mem="device")
    assert_matches_oracle(library_result(ctx), orc.build(r, None), index_only=True)
    ctx.build_batches(w.beams[0])
    assert_matches_oracle(library_result(ctx), orc.build(r, w.beams[0]))
    ctx.destroy()


def test_hundreds_of_small_chunks_and_index_determinism():
    """295 chunks of 68 records and 13 chunks of ~5000: INDEX pass A walks one span per chunk inside ONE launch (ring
    stage and barrier-parity bookkeeping runs on across spans); ONTHEFLY gets tiles of 68 records.  Then the INDEX
    build twice: bit-identical outputs and statistics from run to run."""
    w4 = W.config(4, 20_060)
    r4 = dirty(w4.records(), 21)
    orc = O.Oracle(w4.grid, w4.geometry)
    want_idx, want_beam = orc.build(r4, None), orc.build(r4, w4.beams[0])
    outs = []
    for chunk in (68, 5000, 68):
        ctx = run_library(w4, r4, None, chunk=chunk, mem="device")
        a = library_result(ctx)
        assert_matches_oracle(a, want_idx, index_only=True)
        ctx.build_batches(w4.beams[0])
        b = library_result(ctx)
        assert_matches_oracle(b, want_beam)
        outs.append((a, b))
        ctx.destroy()
    for k in ("E", "wt", "src_index", "counts", "offsets"):
        assert np.array_equal(outs[0][0][k].view(np.uint32), outs[2][0][k].view(np.uint32))
        assert np.array_equal(outs[0][1][k].view(np.uint32), outs[2][1][k].view(np.uint32))
    assert outs[0][1]["stats"] == outs[2][1]["stats"]  # including the double sums: fixed reduction order
    w2 = W.config(2, 20_060)
    check(w2, dirty(w2.records(), 22), None, chunk=68, mem="device")
    w3 = W.config(3, 20_060)
    check(w3, w3.records(), w3.beams[0], chunk=68, mem="pinned")


def test_config5_streamed_at_1e8_records_nine_beams():
    """config 5 at a tenth of its size, in the launch configuration bench.py times: 1e8 records in pinned host
    memory, streamed in 268 435 440-byte chunks (9 586 980 records) through the copy stream while the histogram of
    the previous chunk runs, one index, nine IMRT beams -- every beam's batches against the oracle, element by element."""
    import torch

    p = P()
    w = W.config(5, 100_000_000)
    chunk = W.config(5).chunk_records
    n = w.n_records
    host = torch.empty(n * 28, dtype=torch.uint8, pin_memory=True)
    W.generate_into(w.gen, 0, n, host.data_ptr(), threads=8)
    r = host.numpy().view(W.RECORD_DTYPE)
    ctx = p.PslContext(w.grid, w.geometry, w.mode, max_records=n, max_chunks=n // chunk + 2)
    for f in range(0, n, chunk):
        ctx.load_chunk(host[f * 28:min(n, f + chunk) * 28], p.MEM_PINNED)
    orc = O.Oracle(w.grid, w.geometry)
    for beam in w.beams:  # all nine beams against the oracle, element by element
        ctx.build_batches(beam)
        assert_matches_oracle(library_result(ctx), orc.build(r, beam))
    ctx.destroy()


def test_config5_at_its_real_size_through_bench_verify():
    """config 5 as bench.py times it -- 1e9 records (28 GB) streamed from pinned host memory in 105 chunks, one index,
    nine beams -- checked by bench.py --verify: the oracle classifies every record on all host cores and its counts[],
    statistics and sum(counts) = offsets[K] = n_survivors must equal the library's for the index and for every beam"""
    import json
    import os
    import subprocess
    import sys

    import psutil

    if psutil.virtual_memory().available < 70e9:
        pytest.skip("needs about 60 GB of host memory (28 GB pinned input + oracle work arrays)")
    import gc

    import torch

    gc.collect()
    torch.cuda.empty_cache()  # the child needs 150 GB of the device: give back what earlier tests left in torch's cache
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    run = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--config", "5", "--steps", "1", "--warmup", "3",
                          "--no-cpu-baseline", "--no-e2e", "--no-next", "--verify"], capture_output=True, text=True, timeout=1500)
    assert run.returncode == 0, run.stderr[-2000:]
    line = json.loads(run.stdout.strip().splitlines()[-1])
    v = line["verify"]
    assert line["config"]["workload"] == "cfg5_imrt_streamed" and v["records"] == 1_000_000_000
    assert v["ok"] and len(v["builds"]) == 10 and all(b["ok"] for b in v["builds"]), v


def test_config5_variant_5b_restream_selects_what_the_index_route_selects():
    """no index; every beam re-streams the chunks from host memory and is built on the fly with
    (type, energy) keys.  Against the oracle element by element, and against the index route (5a): the index route's
    survivors are exactly the re-stream's survivors that lie in the position bins the beam's ROI selects (the ROI is a
    margin: a few scattered particles outside it would still have passed the jaws), with the same weights;
    only the order inside a (type, energy) batch differs (load order here, PSL order there)."""
    w = W.config(5, 400_000)
    r = w.records()
    g = w.grid
    grid = dict(g, n_xbins=1, n_ybins=1, x_min=-20.0, y_min=-20.0, dx=40.0, dy=40.0)
    w_otf = W.Workload("cfg5b", w.n_records, w.gen, 0, grid, geometry=w.geometry)
    idx = run_library(w, r, None, chunk=w.chunk_records, mem="pinned")
    otf = None
    orc = O.Oracle(grid, w.geometry)
    cut = 0
    for beam in w.beams[:4]:
        idx.build_batches(beam)
        a = library_result(idx)
        otf = run_library(w_otf, r, dict(beam, roi=None), chunk=w.chunk_records, mem="pinned", ctx=otf)
        b = library_result(otf)
        assert_matches_oracle(b, orc.build(r, dict(beam, roi=None)))
        rx0, rx1, ry0, ry1 = idx.roi_bins(beam)
        ix = np.floor(b["x"] * np.float32(1.0 / g["dx"])).astype(np.int64) - int(round(g["x_min"] / g["dx"]))
        iy = np.floor(b["y"] * np.float32(1.0 / g["dy"])).astype(np.int64) - int(round(g["y_min"] / g["dy"]))
        sel = (rx0 <= ix) & (ix <= rx1) & (ry0 <= iy) & (iy <= ry1)
        cut += int((~sel).sum())
        assert 0 < a["n_survivors"] == int(sel.sum()) and (~sel).sum() < 0.002 * len(sel)
        ia, ib = np.argsort(a["src_index"]), np.argsort(b["src_index"][sel])
        assert np.array_equal(a["src_index"][ia], b["src_index"][sel][ib])
        for f in ("E", "x", "y", "u", "v", "w", "wt"):
            assert np.array_equal(a[f][ia].view(np.uint32), b[f][sel][ib].view(np.uint32)), f
        otf.reset()
    assert cut > 0  # the case exists at this size: the two routes are NOT the same set, by the method's design
    idx.destroy()
    otf.destroy()


def test_bench_variant_5b_runs_at_reduced_size():
    import json
    import os
    import subprocess
    import sys

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    run = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--config", "5", "--variant", "5b", "--records",
                          "20000000", "--steps", "1"], capture_output=True, text=True, timeout=900)
    assert run.returncode == 0, run.stderr[-2000:]
    line = json.loads(run.stdout.strip().splitlines()[-1])
    assert line["config"]["variant"] == "5b" and line["config"]["beams"] == 9 and line["gpu_launches"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 9 * 20_000_000 * 28 and 0.3 < line["e2e"]["h2d_frac"] <= 1.05
    assert len(line["workload_stats"]["survivors_per_beam"]) == 9 and min(line["workload_stats"]["survivors_per_beam"]) > 0


# ---------------------------------------------------------------------------------------------
# x/y-asymmetric configurations: n_xbins != n_ybins, dx != dy, x_min != y_min, z_jaw_x != z_jaw_y != z_map,
# map_nx != map_ny, map_dx != map_dy, map_x0 != map_y0 (every other case in this file is symmetric in x and y, so a
# swapped pair in the kernels or in make_beam would pass it); mirrors tests/test_oracle_pins.py's asymmetric pins
# ---------------------------------------------------------------------------------------------
ASYM_GEOMETRY = dict(z_src=-100.0, z_plane=0.0, z_jaw_x=40.0, z_jaw_y=60.0, z_map=80.0, z_iso=100.0)


def asym_beam(roi=None, seed=3):
    return W.make_beam(jaws=(-9.0, 11.0, -3.0, 2.0), fluence=W.fluence_uniform(seed, nx=96, ny=40), map_x0=-12.0,
                       map_y0=-10.0, map_dx=0.25, map_dy=0.5, roi=roi, mu_weight=0.5)


@pytest.mark.parametrize("keys", ["few", "many"])
def test_asymmetric_grid_planes_and_map_onthefly(keys):
    """ONTHEFLY with position bins: 160 keys (4096-record tiles, compacted survivors for the rejecting beam) and
    1920 keys (1024-record tiles); method 1 (no beam), a rejecting beam, a beam that only weights"""
    shape = dict(n_types=2, n_ebins=2, n_xbins=8, n_ybins=5, x_min=-12.0, y_min=-3.0, dx=3.0, dy=1.0) if keys == "few" else \
        dict(n_types=2, n_ebins=4, n_xbins=48, n_ybins=5, x_min=-12.0, y_min=-3.0, dx=0.5, dy=1.0)
    g = W._grid(**shape)
    w = W.Workload("asym_otf", 300_000, W.GenParams(17, half_x=13.0, half_y=3.0), W.MODE_ONTHEFLY, g, geometry=ASYM_GEOMETRY)
    r = dirty(w.records(), 31)
    nomap = W.make_beam(jaws=(-9.0, 11.0, -3.0, 2.0), mu_weight=0.25)
    weight_only = dict(asym_beam(), jaws=None)
    for beam in (None, asym_beam(), nomap, weight_only):
        lib = check(w, r, beam, chunk=70_000, flags=P().OUT_PROJ, proj=True)
        assert lib["n_survivors"] > 1000
    # the x and y extents differ: a record at (10, 0) is inside, one at (0, 10) is outside
    probe = np.zeros(8, dtype=W.RECORD_DTYPE)
    probe[:] = (0, 1.0, 0.0, 0.0, 0.0, 0.0, 1.0)
    probe["x"][:4], probe["y"][4:] = 10.0, 10.0
    lib = check(w, probe, None)
    assert lib["n_survivors"] == 4 and lib["stats"]["n_outside_grid"] == 4


def test_asymmetric_grid_planes_and_map_index():
    """INDEX: 48 x 20 position bins of 0.5 x 0.25 cm from (-12, -2.5), the bare index, then beams whose ROI row and
    column ranges differ, with PSL_OUT_PROJ"""
    g = W._grid(n_ebins=8, n_xbins=48, n_ybins=20, x_min=-12.0, y_min=-2.5, dx=0.5, dy=0.25)
    w = W.Workload("asym_idx", 400_000, W.GenParams(18, half_x=13.0, half_y=3.0), W.MODE_INDEX, g, geometry=ASYM_GEOMETRY)
    r = dirty(w.records(), 32)
    orc = O.Oracle(g, ASYM_GEOMETRY)
    ctx = run_library(w, r, None, chunk=150_000, flags=P().OUT_PROJ)
    assert_matches_oracle(library_result(ctx), orc.build(r, None), index_only=True)
    for roi in ((-6.2, 7.9, -1.3, 1.1), (-12.0, 12.0, 0.0, 0.25), (3.0, 3.5, -2.5, 2.5), None):
        beam = asym_beam(roi)
        ctx.build_batches(beam)
        lib = library_result(ctx)
        assert_matches_oracle(lib, orc.build(r, beam), proj=True)
        if roi is not None:
            assert ctx.roi_bins(beam) == orc.roi_bins(beam)
        assert lib["n_survivors"] > 50
    assert ctx.roi_bins(asym_beam((-6.2, 7.9, -1.3, 1.1))) == (11, 39, 4, 14)
    ctx.destroy()


def test_index_mode_with_an_energy_edge_table():
    """INDEX + PSL_EBIN_EDGES (k_count_raw<IDX, POS, EDGES>, pass A with the edge search): config 1's 32 log-spaced
    bins over a non-square position grid"""
    g = W._grid(ebin_mode=W.EBIN_EDGES, n_ebins=32, e_min=0.01, e_max=6.0, e_edges=W.log_edges(0.01, 6.0, 32),
                n_xbins=40, n_ybins=16, x_min=-20.0, y_min=-16.0, dx=1.0, dy=2.0)
    w = W.Workload("idx_edges", 600_000, W.GenParams(19), W.MODE_INDEX, g)
    r = dirty(w.records(), 33)
    orc = O.Oracle(g, w.geometry)
    ctx = run_library(w, r, None, chunk=200_000)
    assert_matches_oracle(library_result(ctx), orc.build(r, None), index_only=True)
    beam = W.make_beam(jaws=(-9.0, 5.0, -4.0, 12.0), fluence=W.fluence_uniform(4), roi=(-5.5, 3.5, -3.0, 7.0))
    ctx.build_batches(beam)
    assert_matches_oracle(library_result(ctx), orc.build(r, beam))
    ctx.destroy()
    # no position bins at all: INDEX over (type, energy) only, edge table
    g1 = W._grid(ebin_mode=W.EBIN_EDGES, n_ebins=32, e_min=0.01, e_max=6.0, e_edges=W.log_edges(0.01, 6.0, 32))
    w1 = W.Workload("idx_edges_nopos", 100_000, W.GenParams(20), W.MODE_INDEX, g1)
    r1 = w1.records()
    ctx = run_library(w1, r1, None)
    assert_matches_oracle(library_result(ctx), O.Oracle(g1, w1.geometry).build(r1, None), index_only=True)
    ctx.destroy()


def test_index_mid_size_chunks_use_two_table_columns_per_tile():
    """1e7 records in 100 000-record chunks: 98 tiles per chunk, each cut into 98 segments x 2 histogram CTAs = 196
    table columns, i.e. twice the tile count (the capacity of the column table must allow for it)"""
    w = W.config(4, 10_000_000)
    p = P()
    import torch

    n, chunk = w.n_records, 100_000
    host = torch.empty(n * 28, dtype=torch.uint8, pin_memory=True)
    W.generate_into(w.gen, 0, n, host.data_ptr(), threads=8)
    dev = host.cuda()
    ctx = p.PslContext(w.grid, w.geometry, w.mode, max_records=n)
    for f in range(0, n, chunk):
        ctx.load_chunk(dev[f * 28:(f + chunk) * 28], p.MEM_DEVICE)
    ctx.build_batches(w.beams[0])
    r = host.numpy().view(W.RECORD_DTYPE)
    assert_matches_oracle(library_result(ctx), O.Oracle(w.grid, w.geometry).build(r, w.beams[0]))
    ctx.destroy()


def test_beam_then_bare_index_without_a_sync_in_between():
    """psl_build_batches(beam) leaves an asynchronous copy of its batch offsets in flight; the bare index exposed right
    after it must report the index's own batches"""
    w = W.config(4, 300_000)
    r = w.records()
    ctx = run_library(w, r, None)
    orc = O.Oracle(w.grid, w.geometry).build(r, None)
    for _ in range(20):
        ctx.build_batches(w.beams[0])
        ctx.build_batches(None)
        b = ctx.get_batch(0, 5)
        k0 = 5 * 6400
        assert b["first"] == orc["offsets"][k0] and b["count"] == orc["offsets"][k0 + 6400] - orc["offsets"][k0]
    ctx.destroy()


def test_roi_far_outside_the_grid_is_empty_and_fast():
    import time

    w = W.config(4, 10_000)
    ctx = run_library(w, w.records(), None)
    t0 = time.perf_counter()
    for roi in ((1e12, 2e12, -1.0, 1.0), (-2e12, -1e12, -1.0, 1.0), (-1.0, 1.0, 1e30, 2e30), (-1e30, 1e30, -1e30, 1e30)):
        beam = W.make_beam(jaws=(-5, 5, -5, 5), roi=roi)
        ctx.build_batches(beam)
        assert_matches_oracle(library_result(ctx), O.Oracle(w.grid, w.geometry).build(w.records(), beam))
    assert time.perf_counter() - t0 < 5.0
    ctx.destroy()


# ---------------------------------------------------------------------------------------------
# skewed key distributions: the ranking inside a tile is built for ~1000 buckets hit at random; these inputs put whole
# tiles into one bucket, alternate between two, or arrive already sorted / reverse sorted
# ---------------------------------------------------------------------------------------------
def _skewed(w, kind, n=300_001, seed=11):
    r = W.generate(W.GenParams(seed), 0, n)
    rng = np.random.default_rng(seed)
    if kind == "one_key":
        r["type"][:] = 0
        r["E"][:] = np.float32(1.2345)
        r["x"][:] = np.float32(0.26)
        r["y"][:] = np.float32(-0.74)
    elif kind == "two_keys_alternating":
        r["type"][:] = np.arange(n) % 2
        r["E"][:] = np.where(np.arange(n) % 2 == 0, np.float32(0.3), np.float32(5.9))
        r["x"][:] = np.where(np.arange(n) % 2 == 0, np.float32(-19.9), np.float32(19.9))
        r["y"][:] = np.where(np.arange(n) % 2 == 0, np.float32(-19.9), np.float32(19.9))
    elif kind == "hot_bin":
        hot = rng.random(n) < 0.9
        r["type"][hot] = 0
        r["E"][hot] = np.float32(0.51)
        r["x"][hot] = rng.uniform(1.0, 1.49, int(hot.sum())).astype(np.float32)
        r["y"][hot] = rng.uniform(2.0, 2.49, int(hot.sum())).astype(np.float32)
    elif kind in ("sorted", "reverse_sorted"):
        cls, keys = O.Oracle(w.grid, w.geometry).classify(r, None)
        order = np.argsort(np.where(cls == O.SURVIVOR, keys, -1), kind="stable")
        r = r[order[::-1] if kind == "reverse_sorted" else order].copy()
    return r


@pytest.mark.parametrize("kind", ["one_key", "two_keys_alternating", "hot_bin", "sorted", "reverse_sorted"])
def test_skewed_key_distributions_index(kind):
    w = W.config(4, 300_001)
    r = _skewed(w, kind)
    ctx = run_library(w, r, None, chunk=100_000)
    orc = O.Oracle(w.grid, w.geometry)
    assert_matches_oracle(library_result(ctx), orc.build(r, None), index_only=True)
    ctx.build_batches(w.beams[0])
    assert_matches_oracle(library_result(ctx), orc.build(r, w.beams[0]))
    ctx.destroy()


@pytest.mark.parametrize("kind", ["one_key", "two_keys_alternating", "hot_bin", "sorted", "reverse_sorted"])
@pytest.mark.parametrize("cfg", [2, 3])
def test_skewed_key_distributions_onthefly(kind, cfg):
    w = W.config(cfg, 300_001)
    r = _skewed(w, kind)
    check(w, r, w.beams[0], chunk=100_000)
    wide = W.Workload("otf_pos", w.n_records, w.gen, w.mode,  # 1536 keys: the 1024-record-tile scatter
                      W._grid(n_types=3, n_ebins=8, n_xbins=8, n_ybins=8, x_min=-20.0, y_min=-20.0, dx=5.0, dy=5.0),
                      geometry=w.geometry)
    check(wide, r, w.beams[0], chunk=100_000)
