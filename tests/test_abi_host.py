"""-m "not gpu": the C-ABI library loads, exports every symbol include/psl.h declares, its host-only entry
points work, and everything that needs a device fails loudly (no CPU fallback).  No compute calls."""
import ctypes as C

import numpy as np
import pytest

import paper_1302_1861_b200 as P
import workloads as W
from paper_1302_1861_b200 import binding as B


def test_library_loads_and_exports_every_declared_symbol():
    lib = P.load_library()
    names = P.exported_symbols()
    assert {"psl_create", "psl_load_chunk", "psl_build_batches", "psl_get_batch"} <= set(names)  # north_star's four
    assert len(names) == 21
    for n in names:
        assert hasattr(lib, n), n


def test_struct_layouts_match_the_header():
    import os
    import subprocess
    import tempfile

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    prog = ('#include <stdio.h>\n#include <stddef.h>\n#include "psl.h"\nint main(){printf("%zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu %zu\\n",'
            'sizeof(psl_config),sizeof(psl_beam),sizeof(psl_stats),sizeof(psl_batch),sizeof(psl_record),'
            'offsetof(psl_config,workspace),offsetof(psl_beam,mu_weight),sizeof(psl_plan),sizeof(psl_launch),sizeof(psl_flush),'
            'offsetof(psl_plan,phantom_lo),sizeof(psl_count_totals));return 0;}')
    with tempfile.TemporaryDirectory() as d:
        open(os.path.join(d, "s.c"), "w").write(prog)
        subprocess.run(["gcc", "-I", os.path.join(root, "include"), os.path.join(d, "s.c"), "-o", os.path.join(d, "s")],
                       check=True)
        sizes = [int(v) for v in subprocess.run([os.path.join(d, "s")], capture_output=True, text=True).stdout.split()]
    assert sizes == [C.sizeof(B.Config), C.sizeof(B.Beam), C.sizeof(B.Stats), C.sizeof(B.Batch), 28,
                     B.Config.workspace.offset, B.Beam.mu_weight.offset, C.sizeof(B.Plan), C.sizeof(B.Launch), C.sizeof(B.Flush),
                     B.Plan.phantom_lo.offset, C.sizeof(B.CountTotals)]
    w = W.config(2)
    cfg, _ = B.make_config(w.grid, w.geometry, w.mode, 1000)
    cfg.struct_size = 8  # a stale header must be rejected
    assert P.load_library().psl_workspace_bytes(C.byref(cfg)) == 0


def test_workspace_bytes_scales_and_rejects_bad_configs():
    w2, w4 = W.config(2), W.config(4)
    a = P.workspace_bytes(w2.grid, w2.geometry, w2.mode, 10_000_000, max_host_records=0)
    b = P.workspace_bytes(w2.grid, w2.geometry, w2.mode, 20_000_000, max_host_records=0)
    assert 0 < a < b < 2.3 * a
    assert a >= 10_000_000 * 32  # at least the SoA output
    c = P.workspace_bytes(w4.grid, w4.geometry, w4.mode, 1_000_000)
    assert c >= 1_000_000 * (28 + 32 + 28)
    bad = dict(w2.grid, n_types=4)
    assert P.workspace_bytes(bad, w2.geometry, w2.mode, 1000) == 0
    assert P.workspace_bytes(dict(w4.grid, x_min=-20.1), w4.geometry, w4.mode, 1000) == 0  # origin off the bin lattice
    assert P.workspace_bytes(w4.grid, w4.geometry, P.MODE_ONTHEFLY, 1000) == 0  # 1.2 M keys need the index
    assert P.workspace_bytes(w2.grid, dict(w2.geometry, z_src=5.0), w2.mode, 1000) == 0  # source below the plane
    assert P.workspace_bytes(w2.grid, w2.geometry, w2.mode, 0) == 0
    assert P.workspace_bytes(w2.grid, w2.geometry, w2.mode, 2 ** 32) == 0
    edges = W.log_edges(0.01, 6, 32)
    edges[5] = edges[4]
    assert P.workspace_bytes(dict(W.config(1).grid, e_edges=edges), w2.geometry, 0, 1000) == 0


def test_roi_from_jaws_host_call_closed_form_and_geometry_error():
    geo = dict(z_src=0.0, z_plane=50.0, z_jaw_x=75.0, z_jaw_y=80.0, z_map=100.0, z_iso=100.0)
    rc, roi = P.psl_roi_from_jaws(geo, (-5, 5, -4, 4), 0.0)
    assert rc == 0 and roi == pytest.approx((-7.5, 7.5, -8.0, 8.0), rel=1e-6)
    rc, roi = P.psl_roi_from_jaws(geo, (2, 6, -4, 4), 1.0)
    assert rc == 0 and roi[:2] == pytest.approx((-2.0, 6.0), rel=1e-6)
    rc, _ = P.psl_roi_from_jaws(W.GEOMETRY, (-5, 5, -5, 5), 0.0)  # jaws in the isocentre plane
    assert rc == 4  # PSL_ERR_GEOMETRY


def test_create_fails_loudly_without_a_device_or_with_a_bad_workspace():
    import torch

    lib = P.load_library()
    w = W.config(2)
    cfg, _ = B.make_config(w.grid, w.geometry, w.mode, 4096)
    h = C.c_void_p()
    cfg.workspace, cfg.workspace_bytes = None, 1 << 40
    assert lib.psl_create(C.byref(cfg), C.byref(h)) == 1 and not h  # PSL_ERR_ARG: no workspace
    cfg.workspace, cfg.workspace_bytes = 0x10000, 16
    assert lib.psl_create(C.byref(cfg), C.byref(h)) == 3 and not h  # PSL_ERR_CAPACITY
    assert b"workspace too small" in lib.psl_last_error(None)
    if not torch.cuda.is_available():
        cfg.workspace_bytes = 1 << 40
        assert lib.psl_create(C.byref(cfg), C.byref(h)) == 5 and not h  # PSL_ERR_CUDA: no silent CPU path
        with pytest.raises(P.PslError):
            P.PslContext(w.grid, w.geometry, w.mode, 4096)


def test_product_path_never_touches_the_oracle():
    import os
    import re

    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    pkg = os.path.join(root, "paper_1302_1861_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle|psl_oracle|orc_", text, flags=re.M), f
    for f in ("psl_oracle.c", "psl_oracle.py"):
        text = open(os.path.join(root, "oracle", f)).read()
        assert "paper_1302_1861_b200 import" not in text and "import paper_1302_1861_b200" not in text
        assert "psl.h" not in text and "psl_device" not in text
