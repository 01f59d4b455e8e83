"""Mutation check of the oracle's pins: plausible slips are applied, one at a time, to a COPY of oracle/psl_oracle.c;
each mutated oracle must fail at least one pin of tests/test_oracle_pins.py.  This is what makes "pinned" mean
something: a pin set that a wrong oracle passes pins nothing.  The list starts with the four x<->y slips that
passed every pin of round 1 (square grids, square maps, one plane for everything)."""
import os
import subprocess
import sys
import tempfile

import pytest

from oracle import psl_oracle as O

import test_oracle_pins as pins
import test_oracle_pins_next as pins_next

SRC = os.path.join(os.path.dirname(O.__file__), "psl_oracle.c")

# (name, text in psl_oracle.c, replacement)
MUTATIONS = [
    ("key row stride n_ybins", "npos + (uint32_t)(iy * c->n_xbins + ix);\n}", "npos + (uint32_t)(iy * c->n_ybins + ix);\n}"),
    ("jaw planes swapped between the axes",
     "float dzx = c->z_jaw_x - c->z_plane;\n    float dzy = c->z_jaw_y - c->z_plane;\n    float sx = tx * dzx;\n    float sy = ty * dzy;\n    float xj = r->x + sx;",
     "float dzx = c->z_jaw_y - c->z_plane;\n    float dzy = c->z_jaw_x - c->z_plane;\n    float sx = tx * dzx;\n    float sy = ty * dzy;\n    float xj = r->x + sx;"),
    ("map projection to the jaw plane", "float dz = c->z_map - c->z_plane;", "float dz = c->z_jaw_x - c->z_plane;"),
    ("map row stride map_ny", "(size_t)py * (size_t)b->map_nx + (size_t)px", "(size_t)py * (size_t)b->map_ny + (size_t)px"),
    ("position bin: dy used for x", "if (!orc_axis_bin(x, c->x_min, c->dx, c->n_xbins, ix)) return 0;",
     "if (!orc_axis_bin(x, c->x_min, c->dy, c->n_xbins, ix)) return 0;"),
    ("position bin: n_xbins used for y", "if (!orc_axis_bin(y, c->y_min, c->dy, c->n_ybins, iy)) return 0;",
     "if (!orc_axis_bin(y, c->y_min, c->dy, c->n_xbins, iy)) return 0;"),
    ("map pixel: map_dx used for y", "if (!orc_axis_bin(ym, b->map_y0, b->map_dy, b->map_ny, &py)) return 0.0f;",
     "if (!orc_axis_bin(ym, b->map_y0, b->map_dx, b->map_ny, &py)) return 0.0f;"),
    ("map pixel: map_x0 used for y", "if (!orc_axis_bin(ym, b->map_y0, b->map_dy, b->map_ny, &py)) return 0.0f;",
     "if (!orc_axis_bin(ym, b->map_x0, b->map_dy, b->map_ny, &py)) return 0.0f;"),
    ("jaw y edges scaled to the x jaw plane", "float Y1 = orc_jaw_edge(b->jaw_y1, c->z_jaw_y, c->z_src, c->z_iso);",
     "float Y1 = orc_jaw_edge(b->jaw_y1, c->z_jaw_x, c->z_src, c->z_iso);"),
    ("ROI rows selected with the x extent", "orc_axis_select(c->y_min, c->dy, c->n_ybins, b->roi_y1, b->roi_y2, &out[2], &out[3]);",
     "orc_axis_select(c->y_min, c->dy, c->n_ybins, b->roi_x1, b->roi_x2, &out[2], &out[3]);"),
    ("ROI test transposed", "if (b->has_roi && !(sel[0] <= ix && ix <= sel[1] && sel[2] <= iy && iy <= sel[3]))",
     "if (b->has_roi && !(sel[0] <= iy && iy <= sel[1] && sel[2] <= ix && ix <= sel[3]))"),
    ("closed upper jaw edge", "X1 <= xj && xj < X2", "X1 <= xj && xj <= X2"),
    ("w from 1 + s", "float q = 1.0f - s;", "float q = 1.0f + s;"),
    ("mu applied twice", "return a * b->mu_weight;", "return a * b->mu_weight * b->mu_weight;"),
    ("energy bin by multiplication with the reciprocal", "float g = d / dE;", "float g = d * (1.0f / dE);"),
    ("type-minor key", "((uint32_t)(t * c->n_ebins + ie)) * npos", "((uint32_t)(ie * c->n_types + t)) * npos"),
    ("unstable order inside a key", "uint32_t slot = cursor[my_keys[i]]++;",
     "uint32_t slot = offsets[my_keys[i] + 1] - 1 - (cursor[my_keys[i]]++ - offsets[my_keys[i]]);"),
    # section 8(f)
    ("budget from the PSL's own field count instead of N_total", "budget[k] = (uint32_t)(p / total);",
     "budget[k] = (uint32_t)(p / (total / n_beams));"),
    ("N_total counts a PSL once however many fields select it", "if (orc_beam_mask(c, beams, n_beams, ix, iy) & (1u << i))",
     "if (i == 0 && orc_beam_mask(c, beams, n_beams, ix, iy))"),
    ("no wrap-around at the end of a PSL", "uint32_t slot = offsets[k] + (uint32_t)((start + m) % counts[k]);",
     "uint32_t slot = offsets[k] + (uint32_t)((start + m) < counts[k] ? (start + m) : counts[k] - 1);"),
    ("one particle per PSL per round whatever rr_group says", "for (uint32_t j = 0; j < G && cursor[pos] < share; ++j) {",
     "for (uint32_t j = 0; j < 1 && cursor[pos] < share; ++j) {"),
    ("field picked among all fields, not among those that selected the PSL",
     "beam_out[n_out] = (uint8_t)orc_nth_set_bit(mask[k], which);", "beam_out[n_out] = (uint8_t)which;"),
    ("start offset not random", "uint32_t start = orc_below(orc_rng32(plan->seed, k, 0), counts[k]);", "uint32_t start = 0;"),
    ("gantry turns the other way", "double Rg[9] = { cg, 0, sg, 0, 1, 0, -sg, 0, cg };", "double Rg[9] = { cg, 0, -sg, 0, 1, 0, sg, 0, cg };"),
    ("collimator applied after the gantry", "for (int k = 0; k < 3; ++k) A[3 * i + j] += Rg[3 * i + k] * Rc[3 * k + j];",
     "for (int k = 0; k < 3; ++k) A[3 * i + j] += Rc[3 * i + k] * Rg[3 * k + j];"),
    ("direction keeps +w", "db[3] = { r.u, r.v, -w }", "db[3] = { r.u, r.v, w }"),
    ("surface: far face instead of near face", "if (tn > tnear) tnear = tn;", "if (tf > tnear) tnear = tf;"),
    ("emit weights with field 0's map", "float wt = orc_final_weight(c, b, &r, &xm, &ym);", "float wt = orc_final_weight(c, &beams[0], &r, &xm, &ym);"),
    ("APR turns the direction the other way", "out->u = uc - vs;\n    out->v = us + vc;", "out->u = uc + vs;\n    out->v = vc - us;"),
    ("APR: sine series loses its cubic term", "t = t + s1; t = t * a2;", "t = t * a2;"),
    ("APR: remainder measured from the quarter turn below", "uint32_t k = (uint32_t)(((uint64_t)r + 0x20000000ull) >> 30);",
     "uint32_t k = (uint32_t)(((uint64_t)r + 0x10000000ull) >> 30);"),
    ("partial bins shipped first", "if (++fill[k] == capacity) {", "if (++fill[k] == capacity + 1) {"),
    ("mix64 second multiplier", "0x94D049BB133111EBull", "0x94D049BB133111E9ull"),
]

PINS = [getattr(m, n) for m in (pins_next, pins) for n in dir(m) if n.startswith("test_") and n != "test_generator_shape_matches_recipe"]


def _run_pins(stop_at_first=False):
    """names of the pins that fail with the currently loaded oracle"""
    failed = []
    for fn in PINS:
        marks = [m for m in getattr(fn, "pytestmark", []) if m.name == "parametrize"]
        cases = [()] if not marks else [(v,) if not isinstance(v, tuple) else v for v in marks[0].args[1]]
        for case in cases:
            try:
                fn(*case)
            except (AssertionError, IndexError, ValueError, KeyError, ZeroDivisionError):
                failed.append(fn.__name__)
                break
        if failed and stop_at_first:
            break
    return failed


@pytest.mark.parametrize("name,old,new", MUTATIONS, ids=[m[0] for m in MUTATIONS])
def test_every_mutation_fails_a_pin(name, old, new):
    text = open(SRC).read()
    assert text.count(old) == 1, "the mutation's anchor text must occur exactly once in psl_oracle.c"
    here = os.path.dirname(os.path.abspath(__file__))
    with tempfile.TemporaryDirectory() as tmp:
        c, so = os.path.join(tmp, "mutant.c"), os.path.join(tmp, "libmutant.so")
        open(c, "w").write(text.replace(old, new))
        subprocess.run(["gcc", *O.CFLAGS, "-shared", "-fPIC", "-o", so, c, "-lm"], check=True)
        # in a process of its own: a wrong oracle may well write out of bounds, and a crash is a failed pin too
        prog = ("import sys; sys.path[:0] = [%r, %r]\n"
                "from oracle import psl_oracle as O\nO.use_library(%r)\n"
                "import test_oracle_mutations as T\n"
                "print('FAILED-PINS', T._run_pins(stop_at_first=True))\n" % (os.path.dirname(here), here, so))
        run = subprocess.run([sys.executable, "-c", prog], capture_output=True, text=True, timeout=600)
    crashed = run.returncode != 0
    failed = "FAILED-PINS [" in run.stdout and "FAILED-PINS []" not in run.stdout
    assert crashed or failed, f"mutation '{name}' passes every pin"


def test_the_real_oracle_passes_every_pin_through_the_same_runner():
    O.use_library(None)
    assert _run_pins() == []
