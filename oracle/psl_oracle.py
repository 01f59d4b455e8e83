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
    ]


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
            b.get("mu_weight", 1.0),
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
