"""Pins for the oracle's section-8(f) functions (sampling layer, field rotations + surface projection, APR,
capacity-N emission) against what the paper and the mathematics fix: the paper's budget equations worked by hand and
in exact rational arithmetic, a published known-answer vector for the generator, conservation laws of the round-robin
(every particle of a PSL read the same number of times when the plan asks for whole recyclings), textbook rotations,
brute-force ray / box intersection, invariants of a rotation about the beam axis, and a literal simulation of bins of
capacity N.  PAPER.md:47, :67-71, :82-105."""
import os
from fractions import Fraction

import numpy as np
import pytest

import workloads as W
from oracle import psl_oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
M64 = 2 ** 64 - 1
GAMMA = 0x9E3779B97F4A7C15


def recs(rows):
    a = np.zeros(len(rows), dtype=W.RECORD_DTYPE)
    for i, r in enumerate(rows):
        a[i] = tuple(r)
    return a


def small_psl(n=60_000, seed=5, **grid):
    g = W._grid(**dict(dict(n_types=2, n_ebins=4, n_xbins=10, n_ybins=6, x_min=-5.0, y_min=-3.0, dx=1.0, dy=1.0), **grid))
    w = W.Workload("next", n, W.GenParams(seed, half_x=5.5, half_y=3.5), W.MODE_INDEX, g)
    return w, w.records()


# ---------------------------------------------------------------------------------------------
# the generator (reading S2)
# ---------------------------------------------------------------------------------------------
def test_mix64_reproduces_the_published_splitmix64_vector():
    want = [int(l) for l in open(os.path.join(GOLDEN, "splitmix64.txt")) if l.strip() and l[0] != "#"]
    o = O.Oracle(W._grid(), W.GEOMETRY)
    state, got = 1234567, []
    for _ in want:
        state = (state + GAMMA) & M64
        got.append(o.mix64(state))
    assert got == want


def test_rng32_is_two_nested_rounds_and_uniform():
    o = O.Oracle(W._grid(), W.GEOMETRY)
    for seed, a, b in ((1, 0, 0), (77, 5, 9), (2 ** 63 + 11, 1228799, 4_000_000_000), (0, 2 ** 40, 3)):
        h = o.mix64((seed + GAMMA * (a + 1)) & M64)
        assert o.rng32(seed, a, b) == o.mix64((h + GAMMA * (b + 1)) & M64) >> 32
    r = np.array([o.rng32(42, k, m) for k in range(200) for m in range(100)], dtype=np.uint64)
    cells = np.bincount((r * 64 >> 32).astype(np.int64), minlength=64)
    chi2 = ((cells - len(r) / 64) ** 2 / (len(r) / 64)).sum()
    assert chi2 < 120  # 63 degrees of freedom: mean 63, 120 is beyond 4 sigma
    assert len(set(r.tolist())) > 0.999 * len(r)
    # neighbouring counters are unrelated: about half of the 32 bits differ
    flips = np.array([bin(o.rng32(42, 7, m) ^ o.rng32(42, 7, m + 1)).count("1") for m in range(2000)])
    assert abs(flips.mean() - 16) < 0.5


# ---------------------------------------------------------------------------------------------
# budgets
# ---------------------------------------------------------------------------------------------
def test_budgets_hand_worked_one_and_two_fields():
    # 2 type divisions, 1 energy bin, 2 x 1 position bins; photons: 30 and 10 per PSL, electrons: 6 and 2
    g = W._grid(n_types=2, n_ebins=1, n_xbins=2, n_ybins=1, x_min=-1.0, y_min=0.0, dx=1.0, dy=1.0)
    o = O.Oracle(g, W.GEOMETRY)
    counts = np.array([30, 10, 6, 2], np.uint32)
    whole = W.make_beam(roi=(-1.0, 1.0, 0.0, 1.0))
    assert o.plan_total([whole], counts) == 48
    b, m = o.plan_budgets([whole], counts, 480)
    # P_ij = N_sim P_j / N_total = 480 * 30 / 48 = 300, 480 * 10 / 48 = 100;  E_ij = P_ij E_j / P_j = 300 * 6 / 30 = 60, 100 * 2 / 10 = 20
    assert list(b) == [300, 100, 60, 20] and list(m) == [1, 1, 1, 1]
    left = W.make_beam(roi=(-1.0, 0.0, 0.0, 1.0))  # selects column 0 only
    # N_total = (30 + 6) + (30 + 10 + 6 + 2) = 84 (summed over fields, then over each field's PSLs)
    assert o.plan_total([left, whole], counts) == 84
    b, m = o.plan_budgets([left, whole], counts, 840)
    assert list(b) == [300, 100, 60, 20] and list(m) == [3, 2, 3, 2]
    per_field = [sum(int(b[k]) for k in range(4) if m[k] & (1 << i)) for i in range(2)]
    assert per_field == [360, 480] and sum(per_field) == 840  # every simulated particle is accounted for
    none = W.make_beam(roi=(5.0, 6.0, 0.0, 1.0))
    b, m = o.plan_budgets([none], counts, 100)
    assert list(b) == [0, 0, 0, 0] and list(m) == [0, 0, 0, 0]


def test_budgets_equal_the_papers_equations_in_rational_arithmetic():
    w, r = small_psl()
    o = O.Oracle(w.grid, w.geometry)
    counts = o.build(r, None)["counts"]
    beams = [W.make_beam(roi=(-2.5, 1.2, -1.0, 2.2)), W.make_beam(roi=(-0.5, 4.9, -3.0, 0.1)), W.make_beam()]
    n_sim = 1_234_567
    total = o.plan_total(beams, counts)
    budget, mask = o.plan_budgets(beams, counts, n_sim)
    sels = [o.roi_bins(b) if b["roi"] is not None else (0, 9, 0, 5) for b in beams]
    npos, want_total = 60, 0
    for i, s in enumerate(sels):
        for k in range(o.n_keys):
            ix, iy = (k % npos) % 10, (k % npos) // 10
            inside = s[0] <= ix <= s[1] and s[2] <= iy <= s[3]
            assert bool(mask[k] & (1 << i)) == inside
            want_total += int(counts[k]) if inside else 0
    assert total == want_total
    n_e = 4
    for j in range(n_e * npos):  # j = (energy, position): a photon PSL and an electron PSL
        P_j, E_j = int(counts[j]), int(counts[n_e * npos + j])
        if mask[j] == 0:
            assert budget[j] == 0 and budget[n_e * npos + j] == 0
            continue
        P_ij = Fraction(n_sim * P_j, total)
        assert budget[j] == P_ij.numerator // P_ij.denominator
        if P_j > 0:
            E_ij = P_ij * Fraction(E_j, P_j)
            assert budget[n_e * npos + j] == E_ij.numerator // E_ij.denominator
    simulated = sum(int(budget[k]) * bin(int(mask[k])).count("1") for k in range(o.n_keys))
    pairs = sum(bin(int(mask[k])).count("1") for k in range(o.n_keys))
    assert n_sim - pairs < simulated <= n_sim  # rounding down loses less than one particle per (field, PSL)


# ---------------------------------------------------------------------------------------------
# the launch list of one energy division
# ---------------------------------------------------------------------------------------------
def _round_robin(shares, group):
    """the reading loop, literally: PSL ids in the order their particles are read"""
    left, order = list(shares), []
    while any(left):
        for k, n in enumerate(left):
            take = min(group, n)
            order += [k] * take
            left[k] -= take
    return order


def test_launch_list_is_the_round_robin_over_the_selected_psls():
    w, r = small_psl(20_000)
    o = O.Oracle(w.grid, w.geometry)
    idx = o.build(r, None)
    counts, offsets = idx["counts"], idx["offsets"]
    beams = [W.make_beam(roi=(-2.5, 1.2, -1.0, 2.2)), W.make_beam(roi=(-0.5, 4.9, -3.0, 0.1))]
    n_sim = 3 * o.plan_total(beams, counts) // 2
    budget, mask = o.plan_budgets(beams, counts, n_sim)
    for (t, ie, group) in ((0, 1, 4), (1, 0, 1), (0, 3, 7)):
        plan = o.plan(n_sim, seed=9, rr_group=group)
        k0 = (t * 4 + ie) * 60
        shares = [int(budget[k0 + p]) * bin(int(mask[k0 + p])).count("1") for p in range(60)]
        slot, beam = o.sample_batch(beams, counts, offsets, plan, t, ie, cap=sum(shares) + 10)
        assert len(slot) == sum(shares) > 0
        psl = np.searchsorted(offsets, slot, side="right") - 1 - k0  # which PSL each slot belongs to
        assert list(psl) == _round_robin(shares, group)
        for p in range(60):  # inside a PSL: consecutive particles, wrapping around at the end of the file
            mine = slot[psl == p].astype(np.int64) - int(offsets[k0 + p])
            if len(mine) > 1:
                assert ((np.diff(mine) - 1) % int(counts[k0 + p]) == 0).all()
            assert ((mine >= 0) & (mine < max(int(counts[k0 + p]), 1))).all()
            assert all(int(mask[k0 + p]) & (1 << int(b)) for b in beam[psl == p])  # only fields that selected the PSL


def test_whole_recyclings_read_every_particle_equally_often():
    w, r = small_psl(30_000)
    o = O.Oracle(w.grid, w.geometry)
    idx = o.build(r, None)
    beams = [W.make_beam(roi=(-2.5, 1.2, -1.0, 2.2)), W.make_beam(roi=(-0.5, 4.9, -3.0, 0.1))]
    total = o.plan_total(beams, idx["counts"])
    plan = o.plan(3 * total, seed=4, rr_group=5)  # N_sim = 3 N_total: budget = 3 x the PSL's particles
    budget, mask = o.plan_budgets(beams, idx["counts"], 3 * total)
    assert np.array_equal(budget[mask != 0], 3 * idx["counts"][mask != 0])
    reads = np.zeros(idx["n_survivors"], np.int64)
    n_list = 0
    for t in range(2):
        for ie in range(4):
            slot, _ = o.sample_batch(beams, idx["counts"], idx["offsets"], plan, t, ie, cap=4 * total)
            np.add.at(reads, slot, 1)
            n_list += len(slot)
    assert n_list == 3 * total  # sum over fields and PSLs of the budgets = N_total^simulated
    keys_of_slot = np.repeat(np.arange(o.n_keys), idx["counts"])
    fields = np.array([bin(int(m)).count("1") for m in mask])
    assert np.array_equal(reads, 3 * fields[keys_of_slot])  # whatever the random starts: the wrap-around closes the circle


def test_random_start_and_field_assignment_are_uniform_and_seeded():
    w, r = small_psl(60_000, n_ebins=1, n_types=2)
    o = O.Oracle(w.grid, w.geometry)
    idx = o.build(r, None)
    counts, offsets = idx["counts"], idx["offsets"]
    beams = [W.make_beam(), W.make_beam(), W.make_beam(roi=(-5.0, 0.0, -3.0, 3.0))]
    total = o.plan_total(beams, counts)
    starts, assigned = [], np.zeros((2, 3), np.int64)
    for seed in range(1, 41):
        plan = o.plan(total // 4, seed=seed, rr_group=2)
        slot, beam = o.sample_batch(beams, counts, offsets, plan, 0, 0, cap=total)
        psl = np.searchsorted(offsets, slot, side="right") - 1
        first = {}
        for s_, p in zip(slot, psl):
            first.setdefault(int(p), int(s_))
        starts += [(s_ - int(offsets[p])) / int(counts[p]) for p, s_ in first.items() if counts[p] >= 50]
        left = (psl % 60) % 10 < 5  # PSLs the third field selects as well
        assigned[1] += np.bincount(beam[left], minlength=3)
        assigned[0] += np.bincount(beam[~left], minlength=3)
    cells = np.bincount((np.array(starts) * 16).astype(int), minlength=16)
    chi2 = ((cells - len(starts) / 16) ** 2 / (len(starts) / 16)).sum()
    assert len(starts) > 1500 and chi2 < 50  # 15 degrees of freedom
    assert assigned[0][2] == 0  # a field never receives a particle of a PSL it did not select
    for row, m in ((assigned[0], 2), (assigned[1], 3)):
        n = row.sum()
        for c in row[:m]:
            assert abs(c - n / m) < 4.5 * np.sqrt(n * (1 / m) * (1 - 1 / m))
    a, _ = o.sample_batch(beams, counts, offsets, o.plan(total // 4, seed=1, rr_group=2), 0, 0, cap=total)
    b, _ = o.sample_batch(beams, counts, offsets, o.plan(total // 4, seed=2, rr_group=2), 0, 0, cap=total)
    c, _ = o.sample_batch(beams, counts, offsets, o.plan(total // 4, seed=1, rr_group=2), 0, 0, cap=total)
    assert np.array_equal(a, c) and not np.array_equal(a, b)  # jobs on other GPUs start elsewhere


# ---------------------------------------------------------------------------------------------
# field rotations and projection to the phantom surface (reading S5, S6)
# ---------------------------------------------------------------------------------------------
def _R(axis, deg):
    a = np.deg2rad(deg)
    c, s = np.cos(a), np.sin(a)
    return np.array([[c, -s, 0], [s, c, 0], [0, 0, 1]]) if axis == "z" else np.array([[c, 0, s], [0, 1, 0], [-s, 0, c]])


def test_rotation_matrix_textbook_cases():
    o = O.Oracle(W._grid(), W.GEOMETRY)
    ident = o.beam_matrix(W.make_beam())
    assert np.array_equal(ident, np.eye(3, dtype=np.float32))
    g90 = o.beam_matrix(W.make_beam(gantry_deg=90.0))
    assert np.allclose(g90 @ [0, 0, 1], [1, 0, 0], atol=1e-7)    # the source (on +Zb) swings to +X
    assert np.allclose(g90 @ [0, 0, -1], [-1, 0, 0], atol=1e-7)  # and the beam points along -X
    assert np.allclose(g90 @ [0, 1, 0], [0, 1, 0], atol=1e-7)    # the gantry axis stays
    assert np.allclose(o.beam_matrix(W.make_beam(gantry_deg=180.0)) @ [0, 0, 1], [0, 0, -1], atol=1e-7)
    assert np.allclose(o.beam_matrix(W.make_beam(coll_deg=90.0)) @ [1, 0, 0], [0, 1, 0], atol=1e-7)
    assert np.allclose(o.beam_matrix(W.make_beam(couch_deg=90.0)) @ [1, 0, 0], [0, -1, 0], atol=1e-7)  # table turns, room seen from it turns back
    rng = np.random.default_rng(3)
    for g, c, t in rng.uniform(-180, 360, (40, 3)):
        M = o.beam_matrix(W.make_beam(gantry_deg=g, coll_deg=c, couch_deg=t)).astype(np.float64)
        assert np.allclose(M, _R("z", -t) @ _R("y", g) @ _R("z", c), atol=1.5e-7)  # order: collimator, gantry, couch
        assert np.allclose(M @ M.T, np.eye(3), atol=5e-7) and abs(np.linalg.det(M) - 1) < 1e-6
        v = rng.normal(size=3)
        got = o.rotate(M.astype(np.float32), v.astype(np.float32))
        assert np.allclose(got, M @ v.astype(np.float32), rtol=0, atol=1e-6 * np.abs(v).max())
        assert abs(np.linalg.norm(got) - np.linalg.norm(v.astype(np.float32))) < 1e-6 * np.linalg.norm(v)


def test_surface_projection_closed_forms_and_brute_force():
    o = O.Oracle(W._grid(), W.GEOMETRY)
    lo, hi = (-15.0, -10.0, -20.0), (15.0, 10.0, 5.0)
    hit, S = o.surface((1.0, 2.0, 50.0), (0.0, 0.0, -1.0), lo, hi)
    assert hit and list(S) == [1.0, 2.0, 5.0]                      # straight down onto the top face
    hit, S = o.surface((1.0, 2.0, 0.0), (0.0, 0.0, -1.0), lo, hi)
    assert hit and list(S) == [1.0, 2.0, 0.0]                      # already inside: stays
    assert not o.surface((16.0, 0.0, 50.0), (0.0, 0.0, -1.0), lo, hi)[0]   # passes beside the box
    assert not o.surface((0.0, 0.0, 50.0), (0.0, 0.0, 1.0), lo, hi)[0]     # flies away from it
    hit, S = o.surface((-45.0, 0.0, -5.0), (1.0, 0.0, 0.0), lo, hi)
    assert hit and list(S) == [-15.0, 0.0, -5.0]                   # a lateral field enters through the side
    d = np.array([0.6, 0.0, -0.8], np.float32)
    hit, S = o.surface((-30.0, 0.0, 45.0), d, lo, hi)              # top face at t = 50: x = 0
    assert hit and np.allclose(S, [0.0, 0.0, 5.0], atol=1e-5)
    rng = np.random.default_rng(8)
    n_hit = 0
    for trial in range(400):
        P = rng.uniform(-60, 60, 3).astype(np.float32)
        D = rng.normal(size=3) if trial % 2 else rng.uniform(lo, hi) - P  # every other ray is aimed at the box
        D = (D / np.linalg.norm(D)).astype(np.float32)
        hit, S = o.surface(P, D, lo, hi)
        ts = np.linspace(0.0, 250.0, 25001)
        pts = P[None, :].astype(np.float64) + ts[:, None] * D[None, :].astype(np.float64)
        inside = ((pts >= np.array(lo) - 1e-9) & (pts <= np.array(hi) + 1e-9)).all(axis=1)
        if inside.any():
            first = pts[np.argmax(inside)]
            if hit:
                n_hit += 1
                assert np.allclose(S, first, atol=0.02)  # the step of the brute-force march
                on_face = np.isclose(S, lo, atol=1e-4) | np.isclose(S, hi, atol=1e-4)
                was_inside = ((P >= np.array(lo)) & (P <= np.array(hi))).all()
                assert on_face.any() or was_inside
            else:
                assert inside.sum() <= 2  # a graze the march sees and the slab test may not
        else:
            assert not hit or np.abs(np.clip(S, lo, hi) - S).max() < 1e-4  # at most a graze between two march steps
    assert n_hit > 150


def test_emit_applies_each_particles_own_field():
    w, r = small_psl(40_000)
    geo = dict(z_src=-100.0, z_plane=0.0, z_jaw_x=40.0, z_jaw_y=60.0, z_map=80.0, z_iso=100.0)
    o = O.Oracle(w.grid, geo)
    idx = o.build(r, None)
    f0 = W.make_beam(jaws=(-6.0, 2.0, -3.0, 5.0), fluence=W.fluence_uniform(1, nx=40, ny=24), map_x0=-10.0, map_y0=-6.0,
                     map_dx=0.5, map_dy=0.5, roi=(-4.0, 2.0, -2.5, 3.0), mu_weight=0.25, gantry_deg=30.0, coll_deg=10.0)
    f1 = W.make_beam(jaws=(-2.0, 8.0, -5.0, 1.0), roi=(-2.0, 5.0, -3.0, 1.5), mu_weight=0.75, gantry_deg=250.0, couch_deg=15.0)
    beams = [f0, f1]
    plan = o.plan(2 * o.plan_total(beams, idx["counts"]), seed=3, rr_group=3, phantom=((-12.0, -12.0, -12.0), (12.0, 12.0, 12.0)))
    slot, beam = o.sample_batch(beams, idx["counts"], idx["offsets"], plan, 0, 1, cap=10 ** 6)
    out = o.emit(beams, plan, idx, slot, beam)
    st = out["stats"]
    assert st["n_list"] == len(slot) and st["n_jaw_rejected"] + st["n_zero_weight"] + st["n_missed"] + st["n_launched"] == len(slot)
    assert 0 < st["n_launched"] < len(slot) and st["n_jaw_rejected"] > 0
    # every launched particle passes ITS field's jaws in the hot path's own (separately pinned) classification, carries
    # that field's weight, and the launched ones are the list's entries in list order
    src_list = idx["src_index"][slot]
    per_beam = [o.build(r, dict(b, roi=None), want_classes=True) for b in beams]
    keep = np.array([per_beam[b]["classes"][s_] == O.SURVIVOR for s_, b in zip(src_list, beam)])
    assert keep.sum() == st["n_launched"] + st["n_missed"]
    hit_mask = np.zeros(len(slot), bool)
    j = 0
    for e in np.nonzero(keep)[0]:
        if j < out["n_launched"] and out["src_index"][j] == src_list[e] and out["beam"][j] == beam[e]:
            hit_mask[e] = True
            j += 1
    assert j == out["n_launched"]
    for b in range(2):
        wt_of = dict(zip(per_beam[b]["src_index"].tolist(), per_beam[b]["wt"].tolist()))
        sel = out["beam"] == b
        assert sel.any()
        assert np.array_equal(out["wt"][sel], np.array([wt_of[s_] for s_ in out["src_index"][sel]], np.float32))
    # geometry: the entry point lies on the phantom surface, the direction is the rotated one, energy is a bit copy
    S = np.stack([out["X"], out["Y"], out["Z"]], 1)
    assert (np.isclose(np.abs(S), 12.0, atol=1e-4).any(axis=1)).all() and (np.abs(S) <= 12.0 + 1e-4).all()
    D = np.stack([out["U"], out["V"], out["W"]], 1).astype(np.float64)
    assert np.allclose(np.linalg.norm(D, axis=1), 1.0, atol=2e-6)
    for b in range(2):
        sel = np.nonzero(out["beam"] == b)[0][:200]
        M = o.beam_matrix(beams[b]).astype(np.float64)
        rr = r[out["src_index"][sel]]
        wz = np.sqrt(1 - rr["u"].astype(np.float64) ** 2 - rr["v"].astype(np.float64) ** 2)
        d_b = np.stack([rr["u"], rr["v"], -wz], 1)
        assert np.allclose(D[sel], d_b @ M.T, atol=2e-6)
        p_b = np.stack([rr["x"], rr["y"], np.full(len(sel), 100.0)], 1) @ M.T
        t_ = ((S[sel] - p_b) * D[sel]).sum(1)
        assert (t_ > 0).all() and np.allclose(p_b + t_[:, None] * D[sel], S[sel], atol=2e-4)  # on the particle's own ray
        assert np.array_equal(out["E"][sel].view(np.uint32), rr["E"].view(np.uint32))
    # the beam axis of a field at gantry 30 comes from the source at (100 sin 30, 0, 100 cos 30)
    axis = o.rotate(o.beam_matrix(f0), (0.0, 0.0, 1.0))
    assert np.allclose(axis, [0.5, 0.0, np.sqrt(0.75)], atol=1e-6)


# ---------------------------------------------------------------------------------------------
# azimuthal particle redistribution (reading S7)
# ---------------------------------------------------------------------------------------------
def test_apr_cos_sin_against_the_library_and_exact_quarter_turns():
    o = O.Oracle(W._grid(), W.GEOMETRY)
    assert o.apr_cos_sin(0) == (1.0, 0.0)
    for k, want in ((1, (0.0, 1.0)), (2, (-1.0, 0.0)), (3, (0.0, -1.0))):
        c, s = o.apr_cos_sin(k << 30)
        assert (c, s) == want  # -0.0 == 0.0
    rng = np.random.default_rng(6)
    rs = np.concatenate([rng.integers(0, 2 ** 32, 20000, dtype=np.uint64), [2 ** 29 - 1, 2 ** 29, 2 ** 29 + 1, 2 ** 32 - 1, 3 * 2 ** 29]])
    cs = np.array([o.apr_cos_sin(int(r)) for r in rs], np.float64)
    phi = 2 * np.pi * rs.astype(np.float64) / 2 ** 32
    assert np.abs(cs[:, 0] - np.cos(phi)).max() < 1.5e-7 and np.abs(cs[:, 1] - np.sin(phi)).max() < 1.5e-7
    assert np.abs(cs[:, 0] ** 2 + cs[:, 1] ** 2 - 1).max() < 3e-7


def test_apr_turns_position_and_direction_together_and_uniformly():
    w = W.config(4, 100_000)
    r = w.records()
    o = O.Oracle(w.grid, w.geometry)
    a = o.apr(11, r)
    for f in ("type", "E", "wt"):
        assert np.array_equal(a[f], r[f])
    x, y, u, v = (r[f].astype(np.float64) for f in ("x", "y", "u", "v"))
    X, Y, U, V = (a[f].astype(np.float64) for f in ("x", "y", "u", "v"))
    assert np.allclose(X * X + Y * Y, x * x + y * y, rtol=1e-6, atol=1e-9)      # radius kept
    assert np.allclose(U * U + V * V, u * u + v * v, rtol=1e-6, atol=1e-12)     # polar angle of the direction kept
    assert np.allclose(X * U + Y * V, x * u + y * v, rtol=0, atol=3e-6)          # radial component of the direction kept
    assert np.allclose(X * V - Y * U, x * v - y * u, rtol=0, atol=3e-6)          # and its tangential one
    turn = np.arctan2(x * Y - y * X, x * X + y * Y)                               # the angle each record turned by
    far = x * x + y * y > 1.0
    cells = np.bincount(((turn[far] + np.pi) / (2 * np.pi) * 64).astype(int).clip(0, 63), minlength=64)
    chi2 = ((cells - far.sum() / 64) ** 2 / (far.sum() / 64)).sum()
    assert chi2 < 120                                                             # uniform in azimuth
    want = 2 * np.pi * np.array([o.rng32(11, i, 0) for i in range(300)]) / 2 ** 32
    d = (turn[:300] - want + np.pi) % (2 * np.pi) - np.pi
    assert np.abs(d[far[:300]]).max() < 1e-5                                      # record i turns by 2 pi rng(seed, i) / 2^32
    # counter = load-order index: any sub-range can be redistributed on its own
    assert np.array_equal(o.apr(11, r[5000:9000], first_index=5000).tobytes(), a[5000:9000].tobytes())
    assert not np.array_equal(o.apr(12, r[:100])["x"], a[:100]["x"])
    # the radial histogram of the phase-space is unchanged, the azimuthal one becomes flat
    h0, _ = np.histogram(np.hypot(x, y), bins=20, range=(0, 28))
    h1, _ = np.histogram(np.hypot(X, Y), bins=20, range=(0, 28))
    assert np.abs(h0 - h1).max() <= 2


# ---------------------------------------------------------------------------------------------
# bins of capacity N (reading S9)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("capacity", [1, 7, 64, 10 ** 6])
def test_flush_schedule_is_the_literal_bin_filling_process(capacity):
    w = W.config(3, 30_000)
    r = w.records()
    o = O.Oracle(w.grid, w.geometry)
    res = o.build(r, w.beams[0], want_classes=True)
    ek, ef, ec = o.flush_schedule(res, capacity)
    # literal simulation with Python lists: a bin per key, shipped when it holds `capacity` particles
    bins, shipped = {}, []
    for i in np.nonzero(res["classes"] == O.SURVIVOR)[0]:
        b = bins.setdefault(int(res["keys"][i]), [])
        b.append(int(i))
        if len(b) == capacity:
            shipped.append((int(res["keys"][i]), list(b)))
            b.clear()
    for k in sorted(bins):
        if bins[k]:
            shipped.append((k, list(bins[k])))
    assert len(ek) == len(shipped)
    for (k, members), key, first, count in zip(shipped, ek, ef, ec):
        assert k == key and count == len(members)
        assert list(res["src_index"][first:first + count]) == members  # the shipped particles, in the build's output
    assert int(ec.sum()) == res["n_survivors"]
    full = ec == capacity
    trigger = res["src_index"][ef[full] + ec[full] - 1]
    assert (np.diff(trigger.astype(np.int64)) > 0).all()  # bins fill up in the order their last particle arrives
    if capacity == 10 ** 6:
        assert list(ek) == [k for k in range(o.n_keys) if res["counts"][k] > 0]  # only the final partial bins
