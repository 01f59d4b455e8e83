"""-m gpu: SURVEY 8(f) on the device against the oracle -- budgets, launch lists (bit-exact: the generator is the
same integers on both sides), transport-ready particles after jaws / weights / rotations / surface projection, APR at
index-build time, capacity-N shipments."""
import numpy as np
import pytest

import workloads as W
from helpers import assert_matches_oracle, dirty, library_result, run_library
from oracle import psl_oracle as O

pytestmark = pytest.mark.gpu

ASYM_GEOMETRY = dict(z_src=-100.0, z_plane=0.0, z_jaw_x=40.0, z_jaw_y=60.0, z_map=80.0, z_iso=100.0)
PHANTOM = ((-12.0, -9.0, -14.0), (12.0, 11.0, 10.0))


def P():
    import paper_1302_1861_b200 as P_

    return P_


def _np(t, dtype=None):
    if t is None:  # an empty launch has no arrays
        return np.empty(0, dtype or np.uint8)
    a = t.detach().cpu().numpy()
    return a if dtype is None else a.view(dtype)


def plan_case(n=400_000, flags=0):
    g = W._grid(n_ebins=6, n_xbins=24, n_ybins=10, x_min=-12.0, y_min=-2.5, dx=1.0, dy=0.5)
    w = W.Workload("plan", n, W.GenParams(31, half_x=12.5, half_y=2.8), W.MODE_INDEX, g, geometry=ASYM_GEOMETRY, flags=flags)
    beams = [
        W.make_beam(jaws=(-9.0, 11.0, -3.0, 2.0), fluence=W.fluence_uniform(3, nx=96, ny=40), map_x0=-12.0, map_y0=-10.0,
                    map_dx=0.25, map_dy=0.5, roi=(-6.2, 7.9, -1.3, 1.1), mu_weight=0.25, gantry_deg=30.0, coll_deg=10.0),
        W.make_beam(jaws=(-4.0, 16.0, -2.0, 4.5), roi=(-3.0, 9.5, -1.0, 2.4), mu_weight=0.5, gantry_deg=250.0, couch_deg=15.0),
        W.make_beam(roi=(-12.0, -7.0, -2.5, 0.0), mu_weight=0.25, gantry_deg=180.0, coll_deg=-45.0, couch_deg=-20.0),
    ]
    return w, beams


def compare_launch(lib, slot, beam, orc_out):
    assert lib["n_list"] == len(slot)
    assert np.array_equal(_np(lib["slot"], np.uint32), slot) and np.array_equal(_np(lib["beam"]), beam)
    st = orc_out["stats"]
    assert (lib["n_launch"], lib["n_jaw_rejected"], lib["n_zero_weight"], lib["n_missed"]) == \
        (st["n_launched"], st["n_jaw_rejected"], st["n_zero_weight"], st["n_missed"])
    assert np.array_equal(_np(lib["src_index"], np.uint32), orc_out["src_index"])
    assert np.array_equal(_np(lib["beam_of"]), orc_out["beam"])
    for f in ("E", "X", "Y", "Z", "U", "V", "W", "wt"):
        a, b = _np(lib[f]), orc_out[f]
        assert np.allclose(a, b, rtol=1e-6, atol=1e-6), f
        assert np.array_equal(a.view(np.uint32), b.view(np.uint32)), f + " (bit-equality diagnostic)"


@pytest.mark.parametrize("flags", [0, 2])
def test_budgets_launch_lists_and_emitted_particles(flags):
    w, beams = plan_case(flags=flags)
    r = dirty(w.records(), 41)
    orc = O.Oracle(w.grid, w.geometry, flags=flags)
    idx = orc.build(r, None)
    ctx = P().PslContext(w.grid, w.geometry, w.mode, max_records=len(r), flags=flags, max_launch_records=3_000_000)
    run_library(w, r, None, chunk=150_000, ctx=ctx)
    assert_matches_oracle(library_result(ctx), idx, index_only=True)
    n_sim = 5 * orc.plan_total(beams, idx["counts"]) // 2 + 17
    for seed, group in ((7, 4), (8, 1)):
        total, lens = ctx.plan_set(beams, n_sim, seed=seed, rr_group=group, phantom=PHANTOM)
        assert total == orc.plan_total(beams, idx["counts"])
        budget, mask = orc.plan_budgets(beams, idx["counts"], n_sim)
        lb, lm = ctx.plan_tables()
        assert np.array_equal(_np(lb, np.uint32), budget) and np.array_equal(_np(lm, np.uint32), mask)
        plan = orc.plan(n_sim, seed=seed, rr_group=group, phantom=PHANTOM)
        for t, ie in ((0, 0), (0, 3), (1, 2), (2, 5)):
            slot, beam = orc.sample_batch(beams, idx["counts"], idx["offsets"], plan, t, ie, cap=3_000_000)
            assert lens[t * 6 + ie] == len(slot)
            lib = ctx.sample_batch(t, ie)
            compare_launch(lib, slot, beam, orc.emit(beams, plan, idx, slot, beam))
        assert sum(lens) == sum(int(budget[k]) * bin(int(mask[k])).count("1") for k in range(orc.n_keys) if idx["counts"][k])
    ctx.destroy()


def test_plan_edge_cases_and_errors():
    p = P()
    w, beams = plan_case(60_000)
    r = w.records()
    orc = O.Oracle(w.grid, w.geometry)
    idx = orc.build(r, None)
    ctx = p.PslContext(w.grid, w.geometry, w.mode, max_records=len(r), max_launch_records=5000)
    with pytest.raises(p.PslError) as e:
        ctx.plan_set(beams, 1000)
    assert e.value.status_name == "PSL_ERR_STATE"  # no index yet
    run_library(w, r, None, ctx=ctx)
    with pytest.raises(p.PslError) as e:
        ctx.sample_batch(0, 0)
    assert e.value.status_name == "PSL_ERR_STATE"  # no plan yet
    # nothing selected: empty lists; a tiny plan: most budgets round down to zero
    far = [W.make_beam(roi=(50.0, 60.0, 50.0, 60.0))]
    total, lens = ctx.plan_set(far, 1000, phantom=PHANTOM)
    assert total == 0 and sum(lens) == 0 and ctx.sample_batch(0, 0)["n_list"] == 0
    total, lens = ctx.plan_set(beams, 300, seed=5, rr_group=3, phantom=PHANTOM)
    plan = orc.plan(300, seed=5, rr_group=3, phantom=PHANTOM)
    slot, beam = orc.sample_batch(beams, idx["counts"], idx["offsets"], plan, 0, 1, cap=5000)
    compare_launch(ctx.sample_batch(0, 1), slot, beam, orc.emit(beams, plan, idx, slot, beam))
    # a plan whose lists do not fit
    total, lens = ctx.plan_set(beams, 10 * total, phantom=PHANTOM)
    assert max(lens) > 5000
    with pytest.raises(p.PslError) as e:
        ctx.sample_batch(0, int(np.argmax(lens[:6])))
    assert e.value.status_name == "PSL_ERR_CAPACITY"
    with pytest.raises(p.PslError) as e:
        ctx.plan_set(beams, 100, rr_group=0)
    assert e.value.status_name == "PSL_ERR_ARG"
    ctx.destroy()


def test_launch_lists_at_config4_scale():
    """2e6 records on the 80 x 80 grid of config 4, three overlapping fields, a whole-recycling plan: the photon
    division with the most particles (4e4 entries, dozens of rounds)"""
    w = W.config(4, 2_000_000)
    r = w.records()
    beams = [dict(w.beams[0], gantry_deg=0.0), W.make_beam(jaws=(-8.0, 2.0, -3.0, 7.0), roi=(-5.0, 2.0, -2.5, 4.5), mu_weight=0.3, gantry_deg=120.0),
             W.make_beam(jaws=(-2.0, 9.0, -9.0, 1.0), fluence=W.fluence_uniform(8), roi=(-2.0, 5.5, -5.5, 1.5), mu_weight=0.2, gantry_deg=240.0, coll_deg=30.0)]
    orc = O.Oracle(w.grid, w.geometry)
    idx = orc.build(r, None)
    ctx = P().PslContext(w.grid, w.geometry, w.mode, max_records=len(r), max_launch_records=400_000)
    run_library(w, r, None, chunk=500_000, ctx=ctx)
    total = orc.plan_total(beams, idx["counts"])
    n_sim = 2 * total
    got_total, lens = ctx.plan_set(beams, n_sim, seed=99, rr_group=4)
    assert got_total == total and sum(lens) == n_sim
    plan = orc.plan(n_sim, seed=99, rr_group=4)
    b = int(np.argmax(lens))
    for t, ie in ((b // 64, b % 64), (1, 20)):
        slot, beam = orc.sample_batch(beams, idx["counts"], idx["offsets"], plan, t, ie, cap=400_000)
        compare_launch(ctx.sample_batch(t, ie), slot, beam, orc.emit(beams, plan, idx, slot, beam))
    assert lens[b] > 30_000
    ctx.destroy()


def test_apr_at_index_build_time():
    p = P()
    w = W.config(4, 600_000)
    r = dirty(w.records(), 5)
    orc = O.Oracle(w.grid, w.geometry)
    turned = orc.apr(2024, r)
    for chunk, mem in ((200_000, "device"), (68 * 1000, "pinned")):
        ctx = p.PslContext(w.grid, w.geometry, w.mode, max_records=len(r), flags=p.APR, apr_seed=2024)
        run_library(w, r, None, chunk=chunk, mem=mem, ctx=ctx)
        assert_matches_oracle(library_result(ctx), orc.build(turned, None), index_only=True)
        ctx.build_batches(w.beams[0])
        assert_matches_oracle(library_result(ctx), orc.build(turned, w.beams[0]))
        ctx.destroy()
    # the redistribution moves particles between PSLs: not the index of the unturned records
    assert not np.array_equal(orc.build(turned, None)["counts"], orc.build(r, None)["counts"])
    with pytest.raises(p.PslError):
        p.PslContext(W.config(2, 1000).grid, w.geometry, p.MODE_ONTHEFLY, max_records=1000, flags=p.APR)


@pytest.mark.parametrize("cfg", [2, 3])
def test_capacity_n_shipments(cfg):
    p = P()
    w = W.config(cfg, 300_000)
    r = dirty(w.records(), 6)
    orc = O.Oracle(w.grid, w.geometry)
    res = orc.build(r, w.beams[0], want_classes=True)
    ctx = p.PslContext(w.grid, w.geometry, w.mode, max_records=len(r), max_launch_records=320_000)
    run_library(w, r, w.beams[0], chunk=100_000, ctx=ctx)
    for capacity in (1, 7, 64, 4096, 10 ** 6):
        ek, ef, ec = orc.flush_schedule(res, capacity)
        lib = ctx.flush_schedule(capacity)
        assert lib["n_events"] == len(ek)
        assert np.array_equal(_np(lib["key"], np.uint32), ek)
        assert np.array_equal(_np(lib["first"], np.uint32), ef) and np.array_equal(_np(lib["count"], np.uint32), ec)
    small = p.PslContext(w.grid, w.geometry, w.mode, max_records=len(r), max_launch_records=100)
    run_library(w, r, w.beams[0], ctx=small)
    with pytest.raises(p.PslError) as e:
        small.flush_schedule(1)
    assert e.value.status_name == "PSL_ERR_CAPACITY"
    small.destroy()
    ctx.destroy()
