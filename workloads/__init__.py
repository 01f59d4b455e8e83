"""Seeded synthetic inputs for the phase-space source hot path (INPUTS ONLY).

This module serves both the CPU oracle (``oracle/``) and the CUDA library
(``paper_1302_1861_b200/``).  It holds none of the method's arithmetic: it only
draws records, fluence maps and run parameters shaped like BASELINE.json's five
configs (which in turn stand in for the paper's 6 MV Varian 21EX phase-space,
PAPER.md:127-131, section 2.6 -- data that is not in this container).

Everything returned is plain numpy / plain Python: a ``Workload`` carries a
``grid`` dict, a ``geometry`` dict and a list of ``beam`` dicts; the oracle
wrapper and the library binding each marshal those into their own C structs.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field
from typing import Dict, List, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "phsp_gen.c")
_LIB = os.path.join(_HERE, "libphsp_gen.so")

#: 28-byte packed record: BASELINE.json config 1 ("int32 type ... fp32 energy, x, y, u, v, weight")
RECORD_DTYPE = np.dtype(
    [("type", "<i4"), ("E", "<f4"), ("x", "<f4"), ("y", "<f4"), ("u", "<f4"), ("v", "<f4"), ("wt", "<f4")]
)
assert RECORD_DTYPE.itemsize == 28

SEED_BASE = 0x1302186100

MODE_ONTHEFLY = 0  # paper methods 1 and 2
MODE_INDEX = 1     # paper method 3, the PSL method

EBIN_LINEAR = 0
EBIN_EDGES = 1


class _Params(ctypes.Structure):
    _fields_ = [
        ("seed", ctypes.c_uint64),
        ("half_x", ctypes.c_double),
        ("half_y", ctypes.c_double),
        ("src_dist", ctypes.c_double),
        ("sigma_rad", ctypes.c_double),
        ("frac_photon", ctypes.c_double),
        ("frac_electron", ctypes.c_double),
        ("e_lo", ctypes.c_double),
        ("e_hi", ctypes.c_double),
        ("e_scale", ctypes.c_double),
    ]


def build(force: bool = False) -> str:
    """Compile the generator (gcc, OpenMP) next to its source; returns the .so path."""
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if force or stale:
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.wl_generate.argtypes = [ctypes.POINTER(_Params), ctypes.c_uint64, ctypes.c_uint64, ctypes.c_void_p]
        lib.wl_generate.restype = None
        lib.wl_record_bytes.restype = ctypes.c_uint32
        assert lib.wl_record_bytes() == 28
        _lib = lib
    return _lib


@dataclass
class GenParams:
    seed: int
    half_x: float = 20.0
    half_y: float = 20.0
    src_dist: float = 100.0
    sigma_deg: float = 0.5
    frac_photon: float = 0.98
    frac_electron: float = 0.018
    e_lo: float = 0.01
    e_hi: float = 6.0
    e_scale: float = 0.5

    def _c(self) -> _Params:
        return _Params(
            self.seed, self.half_x, self.half_y, self.src_dist, np.deg2rad(self.sigma_deg),
            self.frac_photon, self.frac_electron, self.e_lo, self.e_hi, self.e_scale,
        )


def generate(gp: GenParams, first: int, n: int, out: Optional[np.ndarray] = None) -> np.ndarray:
    """Records ``first .. first+n`` of the stream ``gp`` as a RECORD_DTYPE array."""
    if out is None:
        out = np.empty(n, dtype=RECORD_DTYPE)
    assert out.dtype == RECORD_DTYPE and out.flags.c_contiguous and out.shape[0] >= n
    c = gp._c()
    _load().wl_generate(ctypes.byref(c), first, n, out.ctypes.data)
    return out[:n]


def generate_into(gp: GenParams, first: int, n: int, address: int, threads: int = 0) -> None:
    """Same stream written straight to ``address`` (e.g. a pinned torch buffer), 28*n bytes.  The generator is
    counter-based, so ``threads`` > 1 fills disjoint sub-ranges concurrently (ctypes releases the GIL)."""
    c = gp._c()
    lib = _load()
    if threads <= 1 or n < 1_000_000:
        lib.wl_generate(ctypes.byref(c), first, n, ctypes.c_void_p(address))
        return
    from concurrent.futures import ThreadPoolExecutor

    piece = (n + threads - 1) // threads
    piece += (-piece) % 4
    jobs = [(f, min(piece, n - f)) for f in range(0, n, piece)]
    with ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(lambda j: lib.wl_generate(ctypes.byref(c), first + j[0], j[1],
                                              ctypes.c_void_p(address + RECORD_DTYPE.itemsize * j[0])), jobs))


# ----------------------------------------------------------------------------------------
# run parameters
# ----------------------------------------------------------------------------------------

#: reading G10: source 100 cm above the scoring plane, isocentre 100 cm below it.
GEOMETRY = dict(z_src=-100.0, z_plane=0.0, z_jaw_x=100.0, z_jaw_y=100.0, z_map=100.0, z_iso=100.0)


def log_edges(e_min: float, e_max: float, n: int) -> np.ndarray:
    """n+1 log-spaced bin edges, evaluated once in double and rounded to fp32 (config data)."""
    k = np.arange(n + 1, dtype=np.float64)
    e = e_min * (e_max / e_min) ** (k / n)
    e[0], e[-1] = e_min, e_max
    return e.astype(np.float32)


def fluence_uniform(seed: int, nx: int = 160, ny: int = 160) -> np.ndarray:
    """'Fluence map of 160x160 fp32 pixels ... values uniform in [0,1] from the seed' (config 3)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return rng.random((ny, nx), dtype=np.float32)


def fluence_segments(seed: int, nx: int = 160, ny: int = 160) -> np.ndarray:
    """IMRT-like map (config 5): sum of 5-15 seeded rectangular segments, weights U[0.2,1],
    normalised by the sum of the weights.  Rectangles live in the central 24x24 cm of the map."""
    rng = np.random.Generator(np.random.PCG64(seed))
    nseg = int(rng.integers(5, 16))
    m = np.zeros((ny, nx), dtype=np.float64)
    wsum = 0.0
    for _ in range(nseg):
        w = float(rng.uniform(0.2, 1.0))
        cx, cy = rng.integers(nx // 2 - 32, nx // 2 + 32, size=2)
        hx, hy = rng.integers(4, 17, size=2)  # half sizes 1..4 cm at 0.25 cm pixels
        x0, x1 = max(0, cx - hx), min(nx, cx + hx)
        y0, y1 = max(0, cy - hy), min(ny, cy + hy)
        m[y0:y1, x0:x1] += w
        wsum += w
    return (m / wsum).astype(np.float32)


def make_beam(jaws=None, fluence=None, map_x0=-20.0, map_y0=-20.0, map_d=0.25, roi=None, mu_weight=1.0,
              gantry_deg=0.0, coll_deg=0.0, couch_deg=0.0, map_dx=None, map_dy=None) -> Dict:
    """A per-field description: jaws = (x1, x2, y1, y2) at isocentre or None; fluence = 2-D fp32
    array [ny, nx] or None (pixel size map_d, or map_dx x map_dy when they differ); roi = (x1, x2, y1, y2)
    at the scoring plane or None; the three angles in degrees."""
    return dict(jaws=jaws, fluence=fluence, map_x0=map_x0, map_y0=map_y0,
                map_dx=map_d if map_dx is None else map_dx, map_dy=map_d if map_dy is None else map_dy,
                roi=roi, mu_weight=mu_weight, gantry_deg=gantry_deg, coll_deg=coll_deg, couch_deg=couch_deg)


@dataclass
class Workload:
    name: str
    n_records: int
    gen: GenParams
    mode: int
    grid: Dict                      # n_types, ebin_mode, n_ebins, e_min, e_max, e_edges, n_xbins, n_ybins, x_min, y_min, dx, dy
    geometry: Dict = field(default_factory=lambda: dict(GEOMETRY))
    beams: List[Optional[Dict]] = field(default_factory=lambda: [None])
    chunk_records: int = 0          # 0 = one chunk
    flags: int = 0

    @property
    def n_keys(self) -> int:
        g = self.grid
        return g["n_types"] * g["n_ebins"] * g["n_xbins"] * g["n_ybins"]

    def records(self, first: int = 0, n: Optional[int] = None) -> np.ndarray:
        return generate(self.gen, first, self.n_records - first if n is None else n)

    def chunks(self):
        """(first, n) pairs covering the stream in chunk_records pieces."""
        c = self.chunk_records or self.n_records
        first = 0
        while first < self.n_records:
            n = min(c, self.n_records - first)
            yield first, n
            first += n


def _grid(n_types=3, ebin_mode=EBIN_LINEAR, n_ebins=64, e_min=0.0, e_max=6.0, e_edges=None,
          n_xbins=1, n_ybins=1, x_min=-20.0, y_min=-20.0, dx=40.0, dy=40.0) -> Dict:
    return dict(n_types=n_types, ebin_mode=ebin_mode, n_ebins=n_ebins, e_min=e_min, e_max=e_max,
                e_edges=e_edges, n_xbins=n_xbins, n_ybins=n_ybins, x_min=x_min, y_min=y_min, dx=dx, dy=dy)


def imrt_beams(seed: int, n_beams: int = 9, margin: float = 1.0, geometry: Dict = GEOMETRY) -> List[Dict]:
    """Config 5: nine beams at 40-degree gantry spacing, each with its own segment map, jaws fit to
    the bounding box of the non-zero pixels, ROI = source back-projection of the jaw box to the
    scoring plane plus `margin` cm."""
    g = geometry
    back = (g["z_plane"] - g["z_src"]) / (g["z_iso"] - g["z_src"])
    beams = []
    for b in range(n_beams):
        m = fluence_segments(seed * 1000 + b)
        ys, xs = np.nonzero(m)
        jx1, jx2 = -20.0 + 0.25 * xs.min(), -20.0 + 0.25 * (xs.max() + 1)
        jy1, jy2 = -20.0 + 0.25 * ys.min(), -20.0 + 0.25 * (ys.max() + 1)
        roi = (jx1 * back - margin, jx2 * back + margin, jy1 * back - margin, jy2 * back + margin)
        beams.append(make_beam(jaws=(jx1, jx2, jy1, jy2), fluence=m, roi=roi, mu_weight=1.0 / n_beams,
                               gantry_deg=40.0 * b))
    return beams


def config(i: int, n_records: Optional[int] = None) -> Workload:
    """BASELINE.json config ``i`` (1..5).  ``n_records`` overrides the size (parity tests use the
    same shapes at sizes the oracle finishes in seconds)."""
    seed = SEED_BASE + i
    if i == 1:
        return Workload(
            name="cfg1_tiny_open_4x4", n_records=n_records or 100_000, gen=GenParams(seed), mode=MODE_ONTHEFLY,
            grid=_grid(ebin_mode=EBIN_EDGES, n_ebins=32, e_min=0.01, e_max=6.0, e_edges=log_edges(0.01, 6.0, 32)),
            beams=[make_beam(jaws=(-2.0, 2.0, -2.0, 2.0))],
        )
    if i == 2:
        return Workload(
            name="cfg2_patient_dependent_10x10", n_records=n_records or 10_000_000,
            gen=GenParams(seed, half_x=6.0, half_y=6.0), mode=MODE_ONTHEFLY, grid=_grid(),
            beams=[None], chunk_records=1_000_000 if n_records is None else max(4, (n_records // 10) // 4 * 4),
        )
    if i == 3:
        return Workload(
            name="cfg3_jaws_fluence_30x30", n_records=n_records or 50_000_000, gen=GenParams(seed),
            mode=MODE_ONTHEFLY, grid=_grid(),
            beams=[make_beam(jaws=(-15.0, 15.0, -15.0, 15.0), fluence=fluence_uniform(seed))],
        )
    psl_grid = _grid(n_xbins=80, n_ybins=80, dx=0.5, dy=0.5)
    if i == 4:
        return Workload(
            name="cfg4_psl_10x10", n_records=n_records or 200_000_000, gen=GenParams(seed), mode=MODE_INDEX,
            grid=psl_grid,
            beams=[make_beam(jaws=(-5.0, 5.0, -5.0, 5.0), fluence=fluence_uniform(seed), roi=(-6.0, 6.0, -6.0, 6.0))],
        )
    if i == 5:
        n = n_records or 1_000_000_000
        return Workload(
            name="cfg5_imrt_streamed", n_records=n, gen=GenParams(seed), mode=MODE_INDEX, grid=psl_grid,
            beams=imrt_beams(seed), chunk_records=9_586_980 if n_records is None else max(4, (n // 7) // 4 * 4),
        )
    raise ValueError("config index must be 1..5")
