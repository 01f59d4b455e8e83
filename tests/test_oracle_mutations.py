"""Mutation check of the oracle's pins: plausible slips are applied, one at a time, to a COPY of oracle/psl_oracle.c;
each mutated oracle must fail at least one pin of tests/test_oracle_pins.py.  This is what makes "pinned" mean
something: a pin set that a wrong oracle passes pins nothing.  The list starts with the four x<->y slips that
passed every pin of round 1 (square grids, square maps, one plane for everything)."""
import os
import subprocess
import tempfile

import pytest

from oracle import psl_oracle as O

import test_oracle_pins as pins

SRC = os.path.join(os.path.dirname(O.__file__), "psl_oracle.c")

# (name, text in psl_oracle.c, replacement)
MUTATIONS = [
    ("key row stride n_ybins", "(uint32_t)(iy * c->n_xbins + ix)", "(uint32_t)(iy * c->n_ybins + ix)"),
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
    ("ROI test transposed", "sel[0] <= ix && ix <= sel[1] && sel[2] <= iy && iy <= sel[3]",
     "sel[0] <= iy && iy <= sel[1] && sel[2] <= ix && ix <= sel[3]"),
    ("closed upper jaw edge", "X1 <= xj && xj < X2", "X1 <= xj && xj <= X2"),
    ("w from 1 + s", "float q = 1.0f - s;", "float q = 1.0f + s;"),
    ("mu applied twice", "return a * b->mu_weight;", "return a * b->mu_weight * b->mu_weight;"),
    ("energy bin by multiplication with the reciprocal", "float g = d / dE;", "float g = d * (1.0f / dE);"),
    ("type-minor key", "((uint32_t)(t * c->n_ebins + ie)) * npos", "((uint32_t)(ie * c->n_types + t)) * npos"),
    ("unstable order inside a key", "uint32_t slot = cursor[my_keys[i]]++;",
     "uint32_t slot = offsets[my_keys[i] + 1] - 1 - (cursor[my_keys[i]]++ - offsets[my_keys[i]]);"),
]

PINS = [getattr(pins, n) for n in dir(pins) if n.startswith("test_") and n != "test_generator_shape_matches_recipe"]


def _run_pins():
    """names of the pins that fail with the currently loaded oracle"""
    failed = []
    for fn in PINS:
        marks = [m for m in getattr(fn, "pytestmark", []) if m.name == "parametrize"]
        cases = [()] if not marks else [(v,) if not isinstance(v, tuple) else v for v in marks[0].args[1]]
        for case in cases:
            try:
                fn(*case)
            except (AssertionError, IndexError, ValueError):
                failed.append(fn.__name__)
                break
    return failed


@pytest.mark.parametrize("name,old,new", MUTATIONS, ids=[m[0] for m in MUTATIONS])
def test_every_mutation_fails_a_pin(name, old, new):
    text = open(SRC).read()
    assert text.count(old) == 1, "the mutation's anchor text must occur exactly once in psl_oracle.c"
    with tempfile.TemporaryDirectory() as tmp:
        c, so = os.path.join(tmp, "mutant.c"), os.path.join(tmp, "libmutant.so")
        open(c, "w").write(text.replace(old, new))
        subprocess.run(["gcc", *O.CFLAGS, "-shared", "-fPIC", "-o", so, c, "-lm"], check=True)
        O.use_library(so)
        try:
            failed = _run_pins()
        finally:
            O.use_library(None)
    assert failed, f"mutation '{name}' passes every pin"


def test_the_real_oracle_passes_every_pin_through_the_same_runner():
    O.use_library(None)
    assert _run_pins() == []
