"""Pins for the CPU oracle (oracle/psl_oracle.c) against what the paper and the mathematics fix.

None of these retype the oracle's own formula in its own precision: they use closed forms at
exact bin edges, double-precision interval arithmetic, numpy's library stable sort, O(N^2) brute
force, rational-arithmetic area overlap, the paper's worked key-space example (tests/golden/),
and special cases that collapse to identities.  Each is chosen so that a plausible slip (dropped
term, wrong sign / index, transposed operand, closed vs half-open edge) fails at least one.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

import workloads as W
from oracle import psl_oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def grid_te(**kw):
    return W._grid(**kw)


def grid_psl(**kw):
    return W._grid(n_xbins=80, n_ybins=80, dx=0.5, dy=0.5, **kw)


def recs(rows):
    a = np.zeros(len(rows), dtype=W.RECORD_DTYPE)
    for i, r in enumerate(rows):
        a[i] = tuple(r)
    return a


def below(x):
    return np.nextafter(np.float32(x), np.float32(-np.inf))


# ---------------------------------------------------------------------------------------------
# record layout / decode
# ---------------------------------------------------------------------------------------------
def test_record_layout_is_28_packed_bytes():
    assert W.RECORD_DTYPE.itemsize == 28 and O.RECORD_DTYPE == W.RECORD_DTYPE
    r = recs([(2, 1.5, -3.25, 4.5, 0.125, -0.25, 0.75)])
    raw = r.tobytes()
    assert len(raw) == 28
    assert np.frombuffer(raw[:4], "<i4")[0] == 2
    assert list(np.frombuffer(raw[4:], "<f4")) == [1.5, -3.25, 4.5, 0.125, -0.25, 0.75]


def test_decode_round_trip_is_bit_copy_and_src_index_is_bijection():
    w = W.config(2, 20000)
    r = w.records()
    o = O.Oracle(w.grid, w.geometry).build(r, None)
    assert o["n_survivors"] == len(r)
    src = o["src_index"]
    assert np.array_equal(np.sort(src), np.arange(len(r), dtype=np.uint32))
    for f in ("E", "x", "y", "u", "v"):
        assert np.array_equal(o[f].view(np.uint32), r[f][src].view(np.uint32)), f
    assert np.array_equal(o["wt"].view(np.uint32), r["wt"][src].view(np.uint32))


# ---------------------------------------------------------------------------------------------
# direction cosine w
# ---------------------------------------------------------------------------------------------
def test_w_closed_forms():
    o = O.Oracle(grid_te(), W.GEOMETRY)
    assert o.w(0.0, 0.0) == 1.0
    assert o.w(0.6, 0.0) == pytest.approx(0.8, rel=2e-7)
    rng = np.random.default_rng(1)
    uv = rng.uniform(-0.7, 0.7, size=(2000, 2)).astype(np.float32)
    for u, v in uv:
        w = o.w(float(u), float(v))
        assert abs(float(u) ** 2 + float(v) ** 2 + w * w - 1.0) < 2.0 ** -22
        # against double precision, within one fp32 rounding of each of the five operations
        assert w == pytest.approx(np.sqrt(1.0 - (float(u) ** 2 + float(v) ** 2)), rel=1e-6)


def test_sideways_or_backward_direction_is_invalid():
    o = O.Oracle(grid_te(), W.GEOMETRY)
    r = recs([(0, 1.0, 0, 0, 0.6, 0.8, 1.0), (0, 1.0, 0, 0, 1.0, 0.0, 1.0), (0, 1.0, 0, 0, 0.9, 0.9, 1.0),
              (0, 1.0, 0, 0, 0.6, 0.79, 1.0)])
    cls, _ = o.classify(r, None)
    assert list(cls) == [O.INVALID, O.INVALID, O.INVALID, O.SURVIVOR]


def test_invalid_records():
    o = O.Oracle(grid_te(), W.GEOMETRY)
    nan, inf = np.nan, np.inf
    rows = [(-1, 1, 0, 0, 0, 0, 1), (3, 1, 0, 0, 0, 0, 1), (0, nan, 0, 0, 0, 0, 1), (0, inf, 0, 0, 0, 0, 1),
            (0, -1, 0, 0, 0, 0, 1), (0, 0, 0, 0, 0, 0, 1), (0, 1, nan, 0, 0, 0, 1), (0, 1, 0, inf, 0, 0, 1),
            (0, 1, 0, 0, nan, 0, 1), (0, 1, 0, 0, 0, -inf, 1), (0, 1, 0, 0, 0, 0, nan), (0, 1, 0, 0, 0, 0, inf)]
    cls, keys = o.classify(recs(rows), None)
    assert (cls == O.INVALID).all() and (keys == 0xFFFFFFFF).all()
    ok = recs([(0, 1, 0, 0, 0, 0, 1), (1, 1, 0, 0, 0, 0, 0.0), (2, 1e-30, 1e3, -1e3, 0, 0, -2.0)])
    cls, _ = o.classify(ok, None)
    assert (cls == O.SURVIVOR).all()


# ---------------------------------------------------------------------------------------------
# energy bins
# ---------------------------------------------------------------------------------------------
def test_linear_energy_bin_closed_form_at_every_edge():
    o = O.Oracle(grid_te(), W.GEOMETRY)
    assert o.bin_width() == 0.09375  # 6/64, exact in fp32
    k = np.arange(1, 64)
    edges = (k * 0.09375).astype(np.float32)
    assert np.array_equal(edges.astype(np.float64), k * 0.09375)  # the edges themselves are exact floats
    assert np.array_equal(o.energy_bins(edges), k)
    assert np.array_equal(o.energy_bins(below(edges)), k - 1)
    assert np.array_equal(o.energy_bins(np.nextafter(edges, np.float32(np.inf))), k)


def test_linear_energy_bin_equals_double_precision_interval_binning():
    o = O.Oracle(grid_te(), W.GEOMETRY)
    rng = np.random.default_rng(7)
    E = np.concatenate([rng.uniform(1e-6, 6.0, 500_000), rng.exponential(0.5, 500_000)]).astype(np.float32)
    E = E[E > 0]
    want = np.clip(np.floor(E.astype(np.float64) / 0.09375), 0, 63).astype(np.int32)
    got = o.energy_bins(E)
    assert np.array_equal(got, want)
    srt = np.sort(E)
    assert (np.diff(o.energy_bins(srt)) >= 0).all()  # monotone


def test_energy_bin_clamps_and_offset_origin():
    o = O.Oracle(grid_te(), W.GEOMETRY)
    assert list(o.energy_bins(np.array([6.0, 6.5, 1e30, 1e-38], np.float32))) == [63, 63, 63, 0]
    o2 = O.Oracle(grid_te(n_ebins=10, e_min=1.0, e_max=6.0), W.GEOMETRY)  # width 0.5, exact
    E = np.array([0.5, 1.0, 1.49, 1.5, 5.99, 6.0], np.float32)
    assert list(o2.energy_bins(E)) == [0, 0, 0, 1, 9, 9]


def test_edge_table_energy_bin_brackets():
    edges = W.log_edges(0.01, 6.0, 32)
    o = O.Oracle(grid_te(ebin_mode=1, n_ebins=32, e_min=0.01, e_max=6.0, e_edges=edges), W.GEOMETRY)
    rng = np.random.default_rng(3)
    E = np.exp(rng.uniform(np.log(0.01), np.log(6.0), 200_000)).astype(np.float32)
    ie = o.energy_bins(E)
    inside = (E >= edges[0]) & (E < edges[-1])
    assert (edges[ie[inside]] <= E[inside]).all() and (E[inside] < edges[ie[inside] + 1]).all()
    # library routine: searchsorted on the same table
    want = np.clip(np.searchsorted(edges, E, side="right") - 1, 0, 31)
    assert np.array_equal(ie, want)
    k = np.arange(1, 32)
    assert np.array_equal(o.energy_bins(edges[k]), k)
    assert np.array_equal(o.energy_bins(below(edges[k])), k - 1)
    assert list(o.energy_bins(np.array([0.001, 6.0, 100.0], np.float32))) == [0, 31, 31]
    # log spacing: constant ratio between consecutive edges (double formula, fp32 rounding)
    ratio = edges[1:].astype(np.float64) / edges[:-1]
    assert np.allclose(ratio, (6.0 / 0.01) ** (1 / 32), rtol=1e-6)


# ---------------------------------------------------------------------------------------------
# position bins and map pixels
# ---------------------------------------------------------------------------------------------
def test_position_bin_is_the_true_interval_at_every_edge():
    o = O.Oracle(grid_psl(), W.GEOMETRY)
    k = np.arange(0, 80)
    x = (-20.0 + 0.5 * k).astype(np.float32)
    assert np.array_equal(o.axis_bins(x, -20.0, 0.5, 80), k)
    b = o.axis_bins(below(x), -20.0, 0.5, 80)
    assert np.array_equal(b, k - 1)  # k=0 -> -1 = outside
    assert list(o.axis_bins(np.array([20.0, 19.999998, -20.000002, 1e30, -1e30], np.float32), -20.0, 0.5, 80)) == \
        [-1, 79, -1, -1, -1]
    # 0.25-cm map pixels, 160 of them
    k = np.arange(0, 160)
    x = (-20.0 + 0.25 * k).astype(np.float32)
    assert np.array_equal(o.axis_bins(x, -20.0, 0.25, 160), k)
    assert np.array_equal(o.axis_bins(below(x), -20.0, 0.25, 160), k - 1)
    # the paper's 1-cm bins over 20x20
    k = np.arange(0, 20)
    x = (-10.0 + k).astype(np.float32)
    assert np.array_equal(o.axis_bins(x, -10.0, 1.0, 20), k)
    assert np.array_equal(o.axis_bins(below(x), -10.0, 1.0, 20), k - 1)


def test_position_bin_equals_double_precision_interval_binning():
    o = O.Oracle(grid_psl(), W.GEOMETRY)
    rng = np.random.default_rng(11)
    x = rng.uniform(-21, 21, 1_000_000).astype(np.float32)
    want = np.floor((x.astype(np.float64) + 20.0) / 0.5).astype(np.int64)
    want[(want < 0) | (want >= 80)] = -1
    assert np.array_equal(o.axis_bins(x, -20.0, 0.5, 80), want.astype(np.int32))


# ---------------------------------------------------------------------------------------------
# key space (PAPER.md:77 worked example) and hand-worked keys
# ---------------------------------------------------------------------------------------------
def test_key_space_matches_paper_worked_example_and_configs():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "paper_keyspace.txt")) if l.strip() and l[0] != "#"]
    seen = set()
    for name, nt, ne, nx, ny, npos, nk in rows:
        nt, ne, nx, ny, npos, nk = map(int, (nt, ne, nx, ny, npos, nk))
        g = W._grid(n_types=nt, n_ebins=ne, n_xbins=nx, n_ybins=ny, x_min=-nx / 2 * 1.0, y_min=-ny / 2 * 1.0, dx=1.0,
                    dy=1.0)
        o = O.Oracle(g, W.GEOMETRY)
        assert nx * ny == npos and o.n_keys == nk, name
        seen.add(name)
        if name.startswith("cfg"):
            assert W.config(int(name[3])).n_keys == nk
    assert {"paper_worked_example", "cfg1", "cfg2", "cfg3", "cfg4", "cfg5"} <= seen


def test_paper_example_keys_enumerate_every_psl_exactly_once():
    # 20x20 cm^2, 1 cm bins, 10 energy bins on [0, 6], 2 type divisions: one particle at the centre of
    # every (type, energy, y, x) cell must get a distinct key, in type-major/energy/row/column order.
    g = W._grid(n_types=2, n_ebins=10, n_xbins=20, n_ybins=20, x_min=-10.0, y_min=-10.0, dx=1.0, dy=1.0)
    o = O.Oracle(g, W.GEOMETRY)
    rows = []
    for t in range(2):
        for ie in range(10):
            for iy in range(20):
                for ix in range(20):
                    rows.append((t, (ie + 0.5) * 0.6, -10 + ix + 0.5, -10 + iy + 0.5, 0, 0, 1))
    cls, keys = o.classify(recs(rows), None)
    assert (cls == O.SURVIVOR).all()
    assert np.array_equal(keys, np.arange(8000, dtype=np.uint32))


def test_electron_positron_merge_with_two_type_divisions():
    g2 = W._grid(n_types=2)
    r = recs([(1, 2.0, 0, 0, 0, 0, 1), (2, 2.0, 0, 0, 0, 0, 1), (0, 2.0, 0, 0, 0, 0, 1)])
    _, k2 = O.Oracle(g2, W.GEOMETRY).classify(r, None)
    _, k3 = O.Oracle(W._grid(), W.GEOMETRY).classify(r, None)
    assert k2[0] == k2[1] == 64 + 21 and k2[2] == 21
    assert list(k3) == [64 + 21, 128 + 21, 21]


def test_hand_worked_cases():
    grids = {"te": grid_te(), "psl": grid_psl()}
    n = 0
    for line in open(os.path.join(GOLDEN, "hand_cases.txt")):
        if not line.strip() or line[0] == "#":
            continue
        g, t, E, x, y, u, v, wt, cls, key = line.split()
        o = O.Oracle(grids[g], W.GEOMETRY)
        c, k = o.classify(recs([(int(t), float(E), float(x), float(y), float(u), float(v), float(wt))]), None)
        assert (int(c[0]), int(k[0])) == (int(cls), int(key)), line
        n += 1
    assert n >= 11


# ---------------------------------------------------------------------------------------------
# histogram, scan, stable order
# ---------------------------------------------------------------------------------------------
def _dirty_records(w, n, seed):
    """generator output with a sprinkling of invalid / out-of-grid records"""
    r = w.records(0, n).copy()
    rng = np.random.default_rng(seed)
    idx = rng.choice(n, size=max(4, n // 50), replace=False)
    q = len(idx) // 4
    r["type"][idx[:q]] = 7
    r["E"][idx[q:2 * q]] = np.nan
    r["x"][idx[2 * q:3 * q]] = 25.0
    r["u"][idx[3 * q:]] = 1.0
    r["wt"] = rng.uniform(0.5, 1.5, n).astype(np.float32)
    return r


@pytest.mark.parametrize("cfg", [1, 3, 4])
def test_counts_offsets_partition_and_weight_conservation(cfg):
    w = W.config(cfg, 60_000)
    r = _dirty_records(w, w.n_records, cfg)
    o = O.Oracle(w.grid, w.geometry)
    res = o.build(r, w.beams[0], want_classes=True)
    st = res["stats"]
    assert st["n_in"] == len(r)
    assert st["n_invalid"] + st["n_outside_grid"] + st["n_roi_skipped"] + st["n_jaw_rejected"] + \
        st["n_zero_weight"] + st["n_survivors"] == st["n_in"]
    assert st["n_invalid"] > 0
    assert int(res["counts"].sum()) == st["n_survivors"] == res["n_survivors"]
    assert res["offsets"][0] == 0 and res["offsets"][-1] == st["n_survivors"]
    assert np.array_equal(np.diff(res["offsets"].astype(np.int64)), res["counts"])
    cls = res["classes"]
    valid = cls != O.INVALID
    assert st["sum_wt_in"] == pytest.approx(r["wt"][valid].astype(np.float64).sum(), rel=1e-12)
    ingrid = valid & (cls != O.OUTSIDE_GRID)
    assert st["sum_wt_indexed"] == pytest.approx(r["wt"][ingrid].astype(np.float64).sum(), rel=1e-12)
    assert st["sum_wt_out"] == pytest.approx(res["wt"].astype(np.float64).sum(), rel=1e-12)
    # each particle lands in exactly the bin its fields define
    keys_out = np.repeat(np.arange(o.n_keys, dtype=np.uint32), res["counts"])
    assert np.array_equal(keys_out, res["keys"][res["src_index"]])


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_order_equals_library_stable_sort(cfg):
    w = W.config(cfg, 50_000)
    r = _dirty_records(w, w.n_records, 100 + cfg)
    res = O.Oracle(w.grid, w.geometry).build(r, w.beams[0], want_classes=True)
    surv = np.nonzero(res["classes"] == O.SURVIVOR)[0]
    order = surv[np.argsort(res["keys"][surv], kind="stable")]
    assert np.array_equal(res["src_index"], order.astype(np.uint32))
    k = res["keys"][res["src_index"]]
    assert (np.diff(k.astype(np.int64)) >= 0).all()
    same = np.diff(k.astype(np.int64)) == 0
    assert (np.diff(res["src_index"].astype(np.int64))[same] > 0).all()


def test_slots_by_brute_force_on_tiny_input():
    w = W.config(4, 400)
    r = _dirty_records(w, 400, 5)
    o = O.Oracle(w.grid, w.geometry)
    beam = W.make_beam(jaws=(-30, 30, -30, 30), roi=(-20, 20, -20, 20))
    res = o.build(r, beam, want_classes=True)
    cls, keys = res["classes"], res["keys"]
    S = [i for i in range(400) if cls[i] == O.SURVIVOR]
    slot = {}
    for i in S:
        lower_keys = sum(1 for j in S if keys[j] < keys[i])
        earlier_same = sum(1 for j in S if j < i and keys[j] == keys[i])
        slot[i] = lower_keys + earlier_same
    assert sorted(slot.values()) == list(range(len(S)))
    for i, s in slot.items():
        assert res["src_index"][s] == i
        assert res["E"][s] == r["E"][i] and res["x"][s] == r["x"][i]


# ---------------------------------------------------------------------------------------------
# ROI -> bins (Fig. 1 caption PAPER.md:196)
# ---------------------------------------------------------------------------------------------
def test_roi_config4_selects_24x24_of_6400_bins():
    o = O.Oracle(grid_psl(), W.GEOMETRY)
    sel = o.roi_bins(W.make_beam(roi=(-6, 6, -6, 6)))
    assert sel == (28, 51, 28, 51)
    assert (sel[1] - sel[0] + 1) * (sel[3] - sel[2] + 1) == 576


def test_roi_selection_by_rational_area_overlap():
    g = W._grid(n_xbins=8, n_ybins=6, x_min=-2.0, y_min=-1.5, dx=0.5, dy=0.5)
    o = O.Oracle(g, W.GEOMETRY)
    rng = np.random.default_rng(2)
    cases = [(-0.75, 0.6, -0.2, 0.3), (-2.0, 2.0, -1.5, 1.5), (0.5, 1.0, 0.0, 0.5), (0.5, 0.5, 0.0, 1.0),
             (-9, -8, 0, 1), (1.9, 7, 1.4, 9), (-1.0, -0.5, -1.0, -0.5)]
    cases += [tuple(np.sort(rng.uniform(-2.5, 2.5, 2))) + tuple(np.sort(rng.uniform(-2, 2, 2))) for _ in range(40)]
    for roi in cases:
        roi = tuple(float(np.float32(v)) for v in roi)
        sel = o.roi_bins(W.make_beam(roi=roi))
        chosen = set()
        for iy in range(6):
            for ix in range(8):
                l, r_ = Fraction(-2) + Fraction(ix, 2), Fraction(-2) + Fraction(ix + 1, 2)
                b, t = Fraction(-3, 2) + Fraction(iy, 2), Fraction(-3, 2) + Fraction(iy + 1, 2)
                ox = min(r_, Fraction(roi[1])) - max(l, Fraction(roi[0]))
                oy = min(t, Fraction(roi[3])) - max(b, Fraction(roi[2]))
                if ox > 0 and oy > 0:
                    chosen.add((ix, iy))
        rect = {(ix, iy) for ix in range(sel[0], sel[1] + 1) for iy in range(sel[2], sel[3] + 1)}
        assert rect == chosen, roi


def test_whole_plane_roi_equals_no_roi_and_empty_roi_keeps_nothing():
    w = W.config(4, 30_000)
    r = w.records()
    o = O.Oracle(w.grid, w.geometry)
    jaws = (-5, 5, -5, 5)
    a = o.build(r, W.make_beam(jaws=jaws, roi=(-20, 20, -20, 20)))
    b = o.build(r, W.make_beam(jaws=jaws))
    assert np.array_equal(a["src_index"], b["src_index"]) and np.array_equal(a["offsets"], b["offsets"])
    e = o.build(r, W.make_beam(jaws=jaws, roi=(3.0, 3.0, -20, 20)))
    assert e["n_survivors"] == 0 and e["stats"]["n_roi_skipped"] == len(r)
    # excluded PSLs "may still include some particles that would pass" the jaws
    c = o.build(r, W.make_beam(jaws=(-15, 15, -15, 15), roi=(-1, 1, -1, 1)))
    d = o.build(r, W.make_beam(jaws=(-15, 15, -15, 15)))
    assert 0 < c["n_survivors"] < d["n_survivors"]
    assert set(c["src_index"]) <= set(d["src_index"])


def test_roi_from_jaws_closed_form():
    geo = dict(z_src=0.0, z_plane=50.0, z_jaw_x=75.0, z_jaw_y=80.0, z_map=100.0, z_iso=100.0)
    o = O.Oracle(grid_psl(), geo)
    rc, roi = o.roi_from_jaws(W.make_beam(jaws=(-5, 5, -4, 4)), 0.0)
    # x: edge at the jaw plane 5*75/100 = 3.75; lever (100-50)/(100-75) = 2 -> 7.5
    # y: edge 4*80/100 = 3.2; lever 50/20 = 2.5 -> 8
    assert rc == 0 and roi == pytest.approx((-7.5, 7.5, -8.0, 8.0), rel=1e-6)
    rc, roi = o.roi_from_jaws(W.make_beam(jaws=(2, 6, -4, 4)), 1.0)
    # centre 4; jaw-plane edges 1.5, 4.5 -> 4 + (1.5-4)*2 = -1 ; 4 + 0.5*2 = 5 ; margin 1
    assert roi[:2] == pytest.approx((-2.0, 6.0), rel=1e-6)
    rc, _ = O.Oracle(grid_psl(), W.GEOMETRY).roi_from_jaws(W.make_beam(jaws=(-5, 5, -5, 5)), 0.0)
    assert rc != 0  # jaws in the isocentre plane: the construction is undefined


# ---------------------------------------------------------------------------------------------
# index route == direct route (sort once per phase-space, select per beam)
# ---------------------------------------------------------------------------------------------
def test_beam_result_from_sorted_index_equals_direct_filter_then_sort():
    w = W.config(4, 80_000)
    r = _dirty_records(w, w.n_records, 9)
    o = O.Oracle(w.grid, w.geometry)
    beam = w.beams[0]
    direct = o.build(r, beam, want_classes=True)
    index = o.build(r, None, want_classes=True)
    # route 2: take the index order (all valid in-grid records by key), keep those the beam keeps
    keep = direct["classes"][index["src_index"]] == O.SURVIVOR
    assert np.array_equal(index["src_index"][keep], direct["src_index"])
    # and the index order is numpy's stable sort of the keys
    ok = np.nonzero(index["classes"] == O.SURVIVOR)[0]
    assert np.array_equal(index["src_index"], ok[np.argsort(index["keys"][ok], kind="stable")].astype(np.uint32))


# ---------------------------------------------------------------------------------------------
# jaws
# ---------------------------------------------------------------------------------------------
def test_pencil_rays_project_to_themselves_and_half_open_aperture():
    o = O.Oracle(grid_te(), W.GEOMETRY)
    X1, X2 = o.jaw_edge(-2.0, 100.0), o.jaw_edge(2.0, 100.0)
    assert (X1, X2) == (-2.0, 2.0)  # jaw plane = isocentre plane: scale 200/200
    xs = np.array([X1, below(X1), below(X2), X2, 0.0], np.float32)
    r = recs([(0, 1.0, float(x), 0.0, 0.0, 0.0, 1.0) for x in xs])
    xj, yj = o.jaw_points(r)
    assert np.array_equal(xj.view(np.uint32), xs.view(np.uint32)) and (yj == 0).all()
    cls, _ = o.classify(r, W.make_beam(jaws=(-2, 2, -2, 2)))
    assert list(cls) == [O.SURVIVOR, O.JAW_REJECTED, O.SURVIVOR, O.JAW_REJECTED, O.SURVIVOR]
    ry = recs([(0, 1.0, 0.0, float(x), 0.0, 0.0, 1.0) for x in xs])
    cls, _ = o.classify(ry, W.make_beam(jaws=(-2, 2, -2, 2)))
    assert list(cls) == [O.SURVIVOR, O.JAW_REJECTED, O.SURVIVOR, O.JAW_REJECTED, O.SURVIVOR]


def test_jaw_edge_scaling_from_source():
    geo = dict(W.GEOMETRY, z_jaw_x=-50.0, z_jaw_y=0.0)
    o = O.Oracle(grid_te(), geo)
    assert o.jaw_edge(8.0, -50.0) == 2.0   # 8 * 50/200
    assert o.jaw_edge(8.0, 0.0) == 4.0     # 8 * 100/200


def test_point_source_rays_scale_linearly_and_fraction_matches_area():
    w = W.config(3, 200_000)
    gp = W.GenParams(seed=99, sigma_deg=0.0)
    r = W.generate(gp, 0, 200_000)
    o = O.Oracle(w.grid, w.geometry)
    xj, yj = o.jaw_points(r)
    # ideal rays from (0,0,-100): at z=+100 the transverse position doubles
    big = np.abs(r["x"]) > 0.5
    assert np.allclose(xj[big], 2.0 * r["x"][big].astype(np.float64), rtol=2e-6)
    big = np.abs(r["y"]) > 0.5
    assert np.allclose(yj[big], 2.0 * r["y"][big].astype(np.float64), rtol=2e-6)
    res = o.build(r, W.make_beam(jaws=(-15, 15, -15, 15)))
    p = (15.0 / 40.0) ** 2  # field maps to +-7.5 cm on the 40x40 plane
    n = len(r)
    assert abs(res["n_survivors"] - n * p) < 4 * np.sqrt(n * p * (1 - p))
    wide = o.build(r, W.make_beam(jaws=(-100, 100, -100, 100)))
    assert wide["n_survivors"] == n and wide["stats"]["n_jaw_rejected"] == 0


def test_asymmetric_jaws_catch_a_swapped_axis_or_sign():
    w = W.config(3, 100_000)
    r = w.records()
    o = O.Oracle(w.grid, w.geometry)
    res = o.build(r, W.make_beam(jaws=(2.0, 14.0, -12.0, -4.0)))
    xj, yj = o.jaw_points(r)
    s = res["src_index"]
    assert res["n_survivors"] > 100
    assert (xj[s] >= 2.0).all() and (xj[s] < 14.0).all() and (yj[s] >= -12.0).all() and (yj[s] < -4.0).all()
    # double-precision projection agrees away from the edges
    tx = r["u"].astype(np.float64) / np.sqrt(1 - r["u"].astype(np.float64) ** 2 - r["v"].astype(np.float64) ** 2)
    assert np.allclose(xj, r["x"] + tx * 100.0, rtol=1e-5, atol=1e-5)
    inside = (xj > 2.001) & (xj < 13.999) & (yj > -11.999) & (yj < -4.001)
    assert set(np.nonzero(inside)[0]) <= set(s)


def test_zero_projection_distance_is_the_identity():
    geo = dict(z_src=-100.0, z_plane=0.0, z_jaw_x=0.0, z_jaw_y=0.0, z_map=0.0, z_iso=0.0)
    w = W.config(1, 20_000)
    r = w.records()
    o = O.Oracle(w.grid, geo)
    xj, yj = o.jaw_points(r)
    assert np.array_equal(xj.view(np.uint32), r["x"].view(np.uint32))
    assert np.array_equal(yj.view(np.uint32), r["y"].view(np.uint32))
    res = o.build(r, W.make_beam(jaws=(-2, 2, -2, 2)), want_classes=True)
    want = (r["x"] >= -2) & (r["x"] < 2) & (r["y"] >= -2) & (r["y"] < 2)
    assert np.array_equal(res["classes"] == O.SURVIVOR, want)


# ---------------------------------------------------------------------------------------------
# fluence map and weights
# ---------------------------------------------------------------------------------------------
def test_constant_map_scales_weight_exactly_and_mu_multiplies_last():
    w = W.config(3, 40_000)
    r = w.records().copy()
    r["wt"] = np.random.default_rng(4).uniform(0.1, 2.0, len(r)).astype(np.float32)
    o = O.Oracle(w.grid, w.geometry)
    c = np.float32(0.3)
    m = np.full((160, 160), c, np.float32)
    res = o.build(r, W.make_beam(jaws=(-15, 15, -15, 15), fluence=m, mu_weight=0.7))
    src = res["src_index"]
    want = (r["wt"][src] * c) * np.float32(0.7)
    assert np.array_equal(res["wt"].view(np.uint32), want.view(np.uint32))
    nomap = o.build(r, W.make_beam(jaws=(-15, 15, -15, 15), mu_weight=0.7))
    assert np.array_equal(nomap["wt"].view(np.uint32), (r["wt"][nomap["src_index"]] * np.float32(0.7)).view(np.uint32))


def test_index_map_recovers_the_pixel_hit_at_the_map_plane():
    w = W.config(3, 100_000)
    r = w.records()
    o = O.Oracle(w.grid, w.geometry)
    m = np.arange(160 * 160, dtype=np.float32).reshape(160, 160)  # exact below 2^24
    res = o.build(r, W.make_beam(jaws=(-19, 19, -19, 19), fluence=m))
    xm, ym = res["xm"].astype(np.float64), res["ym"].astype(np.float64)
    px, py = np.floor((xm + 20) / 0.25), np.floor((ym + 20) / 0.25)
    clear = (np.abs((xm + 20) / 0.25 - np.round((xm + 20) / 0.25)) > 1e-3) & \
            (np.abs((ym + 20) / 0.25 - np.round((ym + 20) / 0.25)) > 1e-3)
    assert clear.mean() > 0.98
    assert np.array_equal(res["wt"][clear], (py * 160 + px)[clear].astype(np.float32))
    # xm, ym are the jaw points here (same plane), and agree with double precision
    xj, yj = o.jaw_points(r)
    assert np.array_equal(res["xm"], xj[res["src_index"]]) and np.array_equal(res["ym"], yj[res["src_index"]])
    # row/column transposition would break this asymmetric probe
    probe = dict(W.make_beam(fluence=m))
    assert o.fluence_at(probe, -19.9, 0.1) == 80 * 160 + 0
    assert o.fluence_at(probe, 0.1, -19.9) == 0 * 160 + 80
    assert o.fluence_at(probe, 20.0, 0.0) == 0.0 and o.fluence_at(probe, 0.0, -20.1) == 0.0


def test_weights_are_map_values_and_zero_weight_flag():
    w = W.config(3, 60_000)
    r = w.records()
    m = W.fluence_uniform(5)
    m[:, :80] = 0.0  # left half blocked
    beam = W.make_beam(jaws=(-15, 15, -15, 15), fluence=m)
    keep = O.Oracle(w.grid, w.geometry).build(r, beam)
    assert np.isin(keep["wt"], m).all()  # wt = 1 in the generator, mu = 1
    assert (keep["wt"] == 0).any()       # zero-weight particles are kept: jaws are the only reject
    drop = O.Oracle(w.grid, w.geometry, flags=O.FLAG_DROP_ZERO_WEIGHT).build(r, beam)
    nz = keep["wt"] != 0
    assert drop["stats"]["n_zero_weight"] == int((~nz).sum()) > 0
    assert np.array_equal(drop["src_index"], keep["src_index"][nz])
    assert (drop["xm"] >= 0).all()


def test_method1_no_beam_keeps_weights_untouched():
    w = W.config(2, 30_000)
    r = w.records().copy()
    r["wt"] = np.linspace(0.5, 1.5, len(r)).astype(np.float32)
    res = O.Oracle(w.grid, w.geometry).build(r, None)
    assert res["n_survivors"] == len(r)
    assert np.array_equal(res["wt"], r["wt"][res["src_index"]])
    assert res["stats"]["sum_wt_in"] == pytest.approx(res["stats"]["sum_wt_out"], rel=1e-12)


def test_generator_shape_matches_recipe():
    r = W.config(1).records()
    frac = np.bincount(r["type"], minlength=3) / len(r)
    assert abs(frac[0] - 0.98) < 0.003 and abs(frac[1] - 0.018) < 0.002 and abs(frac[2] - 0.002) < 0.001
    ph = r["E"][r["type"] == 0]
    assert ph.min() >= 0.01 and ph.max() <= 6.0
    hist, _ = np.histogram(ph, bins=24, range=(0, 6))
    assert np.argmax(hist) in (1, 2)  # mode near 0.5 MeV
    assert abs(ph.mean() - 1.0) < 0.02  # Gamma(2, 0.5) mean = 1 (truncation removes < 0.1 %)
    assert (r["wt"] == 1.0).all() and np.abs(r["x"]).max() < 20 and np.abs(r["y"]).max() < 20


# ---------------------------------------------------------------------------------------------
# x/y-asymmetric parameters: non-square grid, distinct jaw / map planes, non-square map.  Every pin above uses
# n_xbins == n_ybins, dx == dy, a square map and z_jaw_x == z_jaw_y == z_map; the ones below are chosen so that
# an x<->y slip in the key, the jaw planes, the map plane or the map's row stride fails at least one of them
# (tests/test_oracle_mutations.py applies exactly those slips to a copy of the oracle and checks that they do).
# SURVEY 8(c) steps 3, 4, 6, 7.
# ---------------------------------------------------------------------------------------------
ASYM_GRID = dict(n_types=2, n_ebins=3, n_xbins=12, n_ybins=5, x_min=-3.0, y_min=-0.5, dx=0.5, dy=0.25)
ASYM_GEOMETRY = dict(z_src=-100.0, z_plane=0.0, z_jaw_x=40.0, z_jaw_y=60.0, z_map=80.0, z_iso=100.0)


def test_non_square_grid_keys_enumerate_every_cell_exactly_once():
    # 12 x 5 position bins of 0.5 x 0.25 cm from (-3, -0.5), 3 energy bins on [0, 6], 2 type divisions: one
    # particle at the centre of every (t, ie, iy, ix) cell, written in key order => keys = 0 .. K-1
    g = W._grid(**ASYM_GRID)
    o = O.Oracle(g, W.GEOMETRY)
    assert o.n_keys == 2 * 3 * 12 * 5
    rows = []
    for t in range(2):
        for ie in range(3):
            for iy in range(5):
                for ix in range(12):
                    rows.append((t, (ie + 0.5) * 2.0, -3.0 + (ix + 0.5) * 0.5, -0.5 + (iy + 0.5) * 0.25, 0, 0, 1))
    r = recs(rows)
    cls, keys = o.classify(r, None)
    assert (cls == O.SURVIVOR).all()
    assert np.array_equal(keys, np.arange(o.n_keys, dtype=np.uint32))
    # the same through the whole build, fed in reverse: one record per key, slots = keys
    res = o.build(r[::-1].copy(), None)
    assert (res["counts"] == 1).all() and np.array_equal(res["offsets"], np.arange(o.n_keys + 1, dtype=np.uint32))
    assert np.array_equal(res["src_index"], np.arange(o.n_keys, dtype=np.uint32)[::-1])
    # grid edges per axis: x in [-3, 3), y in [-0.5, 0.75)
    edge = recs([(0, 1.0, 2.99, 0.74, 0, 0, 1), (0, 1.0, 3.0, 0.0, 0, 0, 1), (0, 1.0, 0.0, 0.75, 0, 0, 1),
                 (0, 1.0, -3.0, -0.5, 0, 0, 1), (0, 1.0, below(-3.0), 0.0, 0, 0, 1), (0, 1.0, 0.0, below(-0.5), 0, 0, 1),
                 (0, 1.0, 0.8, 0.0, 0, 0, 1)])  # the last one: inside in x only if x uses n_xbins * dx, row 2, column 7
    cls, keys = o.classify(edge, None)
    assert list(cls) == [O.SURVIVOR, O.OUTSIDE_GRID, O.OUTSIDE_GRID, O.SURVIVOR, O.OUTSIDE_GRID, O.OUTSIDE_GRID, O.SURVIVOR]
    assert keys[0] == 4 * 12 + 11 and keys[3] == 0 and keys[6] == 2 * 12 + 7


def test_non_square_grid_roi_rows_and_columns():
    g = W._grid(**ASYM_GRID)
    o = O.Oracle(g, W.GEOMETRY)
    # x: [-1.2, 0.6) touches columns 3 (-1.5..-1.0) .. 7 (0.5..1.0); y: [0.0, 0.3) rows 2 (0..0.25), 3 (0.25..0.5)
    assert o.roi_bins(W.make_beam(roi=(-1.2, 0.6, 0.0, 0.3))) == (3, 7, 2, 3)
    rows = [(0, 1.0, -3.0 + (ix + 0.5) * 0.5, -0.5 + (iy + 0.5) * 0.25, 0, 0, 1) for iy in range(5) for ix in range(12)]
    cls, keys = o.classify(recs(rows), W.make_beam(roi=(-1.2, 0.6, 0.0, 0.3)))
    want = np.array([O.SURVIVOR if (3 <= ix <= 7 and 2 <= iy <= 3) else O.ROI_SKIPPED for iy in range(5) for ix in range(12)])
    assert np.array_equal(cls, want)


def _ideal_rays(n, seed, half_x, half_y):
    """point-source rays (no angular jitter) through a half_x x half_y rectangle of the scoring plane"""
    return W.generate(W.GenParams(seed=seed, sigma_deg=0.0, half_x=half_x, half_y=half_y), 0, n)


def test_distinct_planes_each_axis_projects_to_its_own_plane():
    # z_src = -100, z_plane = 0, z_jaw_x = 40, z_jaw_y = 60, z_map = 80, z_iso = 100: an ideal ray through (x, y)
    # is at x * (z - z_src) / (z_plane - z_src) on the plane z
    o = O.Oracle(grid_te(), ASYM_GEOMETRY)
    r = _ideal_rays(50_000, 41, 12.0, 9.0)
    x, y = r["x"].astype(np.float64), r["y"].astype(np.float64)
    xj, yj = o.jaw_points(r)
    far = (np.abs(x) > 0.5) & (np.abs(y) > 0.5)
    assert np.allclose(xj[far], 1.4 * x[far], rtol=2e-6, atol=0)
    assert np.allclose(yj[far], 1.6 * y[far], rtol=2e-6, atol=0)
    assert not np.allclose(xj[far], 1.6 * x[far], rtol=1e-3) and not np.allclose(yj[far], 1.4 * y[far], rtol=1e-3)
    res = o.build(r, W.make_beam(mu_weight=1.0))  # no jaws: everything survives, xm/ym for every record
    s = res["src_index"]
    f = far[s]
    assert np.allclose(res["xm"][f], 1.8 * x[s][f], rtol=2e-6, atol=0)
    assert np.allclose(res["ym"][f], 1.8 * y[s][f], rtol=2e-6, atol=0)
    # jaw edges, given at the isocentre, scale to each axis' own plane: x by 140/200, y by 160/200
    assert o.jaw_edge(10.0, 40.0) == pytest.approx(7.0, rel=1e-7) and o.jaw_edge(10.0, 60.0) == pytest.approx(8.0, rel=1e-7)


def test_distinct_planes_jaw_box_accepts_only_with_the_right_plane_per_axis():
    o = O.Oracle(grid_te(), ASYM_GEOMETRY)
    beam = W.make_beam(jaws=(-10.0, 10.0, -10.0, 10.0))
    # pencil rays (u = v = 0) stay at (x, y): the aperture at the jaw planes is [-7, 7) x [-8, 8)
    pts = [(6.9, 7.9), (7.1, 0.0), (0.0, 8.1), (-7.0, -8.0), (below(-7.0), 0.0), (0.0, below(-8.0)), (7.5, 7.5), (6.9, -7.5)]
    cls, _ = o.classify(recs([(0, 1.0, px, py, 0.0, 0.0, 1.0) for px, py in pts]), beam)
    J, S = O.JAW_REJECTED, O.SURVIVOR
    assert list(cls) == [S, J, J, S, J, J, J, S]
    # ideal point-source rays: the field edge seen from the source is |x|, |y| < 5 at the scoring plane whatever the
    # jaw planes are -- but only if each axis is projected to the plane its edges were scaled to
    r = _ideal_rays(100_000, 42, 6.0, 6.0)
    res = o.build(r, beam, want_classes=True)
    x, y = r["x"].astype(np.float64), r["y"].astype(np.float64)
    clear = (np.abs(np.abs(x) - 5.0) > 1e-4) & (np.abs(np.abs(y) - 5.0) > 1e-4)
    want = (np.abs(x) < 5.0) & (np.abs(y) < 5.0)
    assert clear.mean() > 0.999
    assert np.array_equal((res["classes"] == S)[clear], want[clear])
    # hand-placed: x = 4.7 passes (1.4 * 4.7 = 6.58 < 7) and would fail on the y plane (1.6 * 4.7 = 7.52);
    #              y = 5.4 fails (1.6 * 5.4 = 8.64 >= 8) and would pass on the x plane (1.4 * 5.4 = 7.56 < 8)
    def ray(px, py):
        d = np.array([px, py, 100.0])
        d /= np.linalg.norm(d)
        return (0, 1.0, px, py, d[0], d[1], 1.0)

    cls, _ = o.classify(recs([ray(4.7, 0.0), ray(0.0, 5.4), ray(4.7, 4.7), ray(0.0, -4.9)]), beam)
    assert list(cls) == [S, J, S, S]


def test_non_square_map_index_map_recovers_the_pixel():
    # 96 columns of 0.25 cm from x = -12, 160 rows of 0.5 cm from y = -40, at z_map = 80 where an ideal ray through
    # (x, y) sits at (1.8 x, 1.8 y); F[py, px] = py * 96 + px (exact in fp32)
    o = O.Oracle(grid_te(), ASYM_GEOMETRY)
    nx, ny = 96, 160
    m = np.arange(nx * ny, dtype=np.float32).reshape(ny, nx)
    beam = W.make_beam(fluence=m, map_x0=-12.0, map_y0=-40.0, map_dx=0.25, map_dy=0.5)
    r = _ideal_rays(100_000, 43, 8.0, 24.0)  # +-14.4 x +-43.2 at the map plane: some rays miss the map
    res = o.build(r, beam)
    assert res["n_survivors"] == len(r)  # no jaws: nothing is rejected, zero-weight records are kept
    s = res["src_index"]
    xm, ym = 1.8 * r["x"][s].astype(np.float64), 1.8 * r["y"][s].astype(np.float64)
    fx, fy = (xm + 12.0) / 0.25, (ym + 40.0) / 0.5
    clear = (np.abs(fx - np.round(fx)) > 1e-3) & (np.abs(fy - np.round(fy)) > 1e-3)
    px, py = np.floor(fx), np.floor(fy)
    inside = (px >= 0) & (px < nx) & (py >= 0) & (py < ny)
    want = np.where(inside, py * nx + px, 0.0).astype(np.float32)
    assert clear.mean() > 0.98 and 0.5 < inside.mean() < 0.95
    assert np.array_equal(res["wt"][clear], want[clear])
    # direct probes of the lookup: row stride is map_nx, x picks the column, y the row
    assert o.fluence_at(beam, -11.9, -39.9) == 0.0
    assert o.fluence_at(beam, -11.9 + 0.25 * 5, -39.9) == 5.0
    assert o.fluence_at(beam, -11.9, -39.9 + 0.5 * 3) == 3.0 * 96
    assert o.fluence_at(beam, 11.9, 39.9) == 159.0 * 96 + 95
    assert o.fluence_at(beam, 12.1, 0.0) == 0.0 and o.fluence_at(beam, 0.0, 40.1) == 0.0  # off the map
    assert o.fluence_at(beam, 0.0, 30.0) == 140.0 * 96 + 48  # y beyond +-12 is still on this 80-cm-tall map


def test_asymmetric_everything_index_route_equals_direct_route():
    # non-square grid + distinct planes + non-square map + ROI through the whole build, both routes
    g = W._grid(**dict(ASYM_GRID, n_types=3, n_ebins=8, n_xbins=48, n_ybins=20, x_min=-12.0, y_min=-2.5))
    o = O.Oracle(g, ASYM_GEOMETRY)
    r = _dirty_records(W.Workload("asym", 40_000, W.GenParams(7, half_x=13.0, half_y=3.0), W.MODE_INDEX, g), 40_000, 5)
    m = W.fluence_uniform(3, nx=96, ny=40)
    beam = W.make_beam(jaws=(-9.0, 11.0, -3.0, 2.0), fluence=m, map_x0=-12.0, map_y0=-10.0, map_dx=0.25, map_dy=0.5,
                       roi=(-6.2, 7.9, -1.3, 1.1), mu_weight=0.5)
    direct = o.build(r, beam, want_classes=True)
    index = o.build(r, None)
    keep = direct["classes"][index["src_index"]] == O.SURVIVOR
    assert np.array_equal(index["src_index"][keep], direct["src_index"])
    assert 100 < direct["n_survivors"] < direct["stats"]["n_in"] - direct["stats"]["n_roi_skipped"]
    sel = o.roi_bins(beam)
    assert sel == (11, 39, 4, 14)  # x: (-6.2+12)/0.5 = 11.6 -> 11, (7.9+12)/0.5 = 39.8 -> 39; y: 1.2/0.25 -> 4, 3.6/0.25 -> 14
