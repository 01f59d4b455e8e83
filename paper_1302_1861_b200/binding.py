"""ctypes binding of include/psl.h -- argument marshalling only.

``PslContext`` has one method per C-ABI call with the same name minus the ``psl_`` prefix.  PyTorch is
used for what the C-ABI leaves to the caller: the device workspace, the fluence map on the device, the
CUDA stream, and zero-copy tensor views of the borrowed output pointers.  Every step of the hot path runs
in the kernels of libpsl_b200.so; if the library is missing this module raises -- there is no fallback.
"""
from __future__ import annotations

import ctypes as C
import os
import re
from typing import Dict, Optional

import numpy as np

from . import _build

MODE_ONTHEFLY, MODE_INDEX = 0, 1
EBIN_LINEAR, EBIN_EDGES = 0, 1
MEM_PAGEABLE, MEM_PINNED, MEM_DEVICE = 0, 1, 2
OUT_PROJ, DROP_ZERO_WEIGHT, NO_COMPACT, APR = 1, 2, 4, 8
RECORD_BYTES = 28

_STATUS = {0: "PSL_OK", 1: "PSL_ERR_ARG", 2: "PSL_ERR_STATE", 3: "PSL_ERR_CAPACITY", 4: "PSL_ERR_GEOMETRY",
           5: "PSL_ERR_CUDA"}


class PslError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{_STATUS.get(status, status)}: {message}")
        self.status = status
        self.status_name = _STATUS.get(status, str(status))


class Geometry(C.Structure):
    _fields_ = [(n, C.c_float) for n in ("z_src", "z_plane", "z_jaw_x", "z_jaw_y", "z_map", "z_iso")]


class Config(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("mode", C.c_int32), ("n_types", C.c_int32), ("ebin_mode", C.c_int32),
        ("n_ebins", C.c_int32), ("e_min", C.c_float), ("e_max", C.c_float), ("e_edges", C.c_void_p),
        ("n_xbins", C.c_int32), ("n_ybins", C.c_int32),
        ("x_min", C.c_float), ("y_min", C.c_float), ("dx", C.c_float), ("dy", C.c_float),
        ("geom", Geometry),
        ("max_records", C.c_uint64), ("max_host_records", C.c_uint64), ("max_beam_records", C.c_uint64),
        ("max_chunks", C.c_uint32), ("flags", C.c_uint32),
        ("apr_seed", C.c_uint64), ("max_launch_records", C.c_uint64),
        ("device", C.c_int32), ("stream", C.c_void_p), ("workspace", C.c_void_p), ("workspace_bytes", C.c_uint64),
    ]


class Beam(C.Structure):
    _fields_ = [
        ("has_jaws", C.c_int32),
        ("jaw_x1", C.c_float), ("jaw_x2", C.c_float), ("jaw_y1", C.c_float), ("jaw_y2", C.c_float),
        ("fluence", C.c_void_p), ("map_nx", C.c_int32), ("map_ny", C.c_int32),
        ("map_x0", C.c_float), ("map_y0", C.c_float), ("map_dx", C.c_float), ("map_dy", C.c_float),
        ("has_roi", C.c_int32),
        ("roi_x1", C.c_float), ("roi_x2", C.c_float), ("roi_y1", C.c_float), ("roi_y2", C.c_float),
        ("mu_weight", C.c_float), ("gantry_deg", C.c_float), ("coll_deg", C.c_float), ("couch_deg", C.c_float),
    ]


class Stats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in
                ("n_in", "n_invalid", "n_outside_grid", "n_roi_skipped", "n_jaw_rejected", "n_zero_weight",
                 "n_survivors")] + [(n, C.c_double) for n in ("sum_wt_in", "sum_wt_indexed", "sum_wt_out")]

    def as_dict(self) -> Dict:
        return {n: getattr(self, n) for n, _ in self._fields_}


class Batch(C.Structure):
    _fields_ = [("first", C.c_uint32), ("count", C.c_uint32)] + \
               [(n, C.c_void_p) for n in ("E", "x", "y", "u", "v", "w", "wt", "xp", "yp", "src_index", "bin_offsets")] + \
               [("n_bins", C.c_uint32)]


class Plan(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_beams", C.c_uint32), ("beams", C.c_void_p), ("n_simulate", C.c_uint64),
                ("seed", C.c_uint64), ("rr_group", C.c_uint32), ("reserved", C.c_uint32),
                ("phantom_lo", C.c_float * 3), ("phantom_hi", C.c_float * 3)]


class Launch(C.Structure):
    _fields_ = [("n_list", C.c_uint32), ("n_launch", C.c_uint32), ("slot", C.c_void_p), ("beam", C.c_void_p)] + \
               [(n, C.c_void_p) for n in ("E", "X", "Y", "Z", "U", "V", "W", "wt", "src_index", "beam_of")] + \
               [(n, C.c_uint64) for n in ("n_jaw_rejected", "n_zero_weight", "n_missed")]


class Flush(C.Structure):
    _fields_ = [("n_events", C.c_uint32), ("key", C.c_void_p), ("first", C.c_void_p), ("count", C.c_void_p)]


class CountTotals(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("n_in", "n_invalid", "n_outside_grid", "n_binned")]


STATIC_MAX_KEYS, STATIC_SCRATCH_BYTES = 2048, 2641152

K_CLASSES = ("count", "scan", "scatter", "index_a", "index_b", "beam", "other", "count_keys", "sample")


class Profile(C.Structure):
    _fields_ = [("ms", C.c_double * len(K_CLASSES)), ("launches", C.c_uint64 * len(K_CLASSES))]


_lib = None


def library_path() -> str:
    return _build.LIB


def exported_symbols() -> list:
    """Every function include/psl.h declares (parsed from the header itself)."""
    hdr = os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", "include", "psl.h")
    text = open(hdr).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(psl_[a-z_]+)\s*\(", text)))


def load_library(build: bool = True):
    """dlopen libpsl_b200.so (building it first if the sources are newer).  Raises if it cannot."""
    global _lib
    if _lib is not None:
        return _lib
    if build:
        _build.build_library()
    if not os.path.exists(_build.LIB):
        raise PslError(5, f"{_build.LIB} is missing: run __graft_entry__.build() (nvcc, sm_100a); there is no CPU path")
    lib = C.CDLL(_build.LIB)
    P = C.POINTER
    lib.psl_workspace_bytes.restype = C.c_uint64
    lib.psl_workspace_bytes.argtypes = [P(Config)]
    lib.psl_create.restype = C.c_int
    lib.psl_create.argtypes = [P(Config), P(C.c_void_p)]
    lib.psl_load_chunk.restype = C.c_int
    lib.psl_load_chunk.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_int32]
    lib.psl_wait_loads.restype = C.c_int
    lib.psl_wait_loads.argtypes = [C.c_void_p]
    lib.psl_build_batches.restype = C.c_int
    lib.psl_build_batches.argtypes = [C.c_void_p, P(Beam), P(Stats)]
    lib.psl_get_stats.restype = C.c_int
    lib.psl_get_stats.argtypes = [C.c_void_p, P(Stats)]
    lib.psl_get_batch.restype = C.c_int
    lib.psl_get_batch.argtypes = [C.c_void_p, C.c_int32, C.c_int32, P(Batch)]
    lib.psl_get_tables.restype = C.c_int
    lib.psl_get_tables.argtypes = [C.c_void_p, P(C.c_void_p), P(C.c_void_p), P(C.c_uint32)]
    lib.psl_roi_from_jaws.restype = C.c_int
    lib.psl_roi_from_jaws.argtypes = [P(Geometry), P(Beam), C.c_float, P(C.c_float * 4)]
    lib.psl_roi_bins.restype = C.c_int
    lib.psl_roi_bins.argtypes = [C.c_void_p, P(Beam), P(C.c_int32 * 4)]
    lib.psl_plan_set.restype = C.c_int
    lib.psl_plan_set.argtypes = [C.c_void_p, P(Plan), P(C.c_uint64), P(P(C.c_uint64))]
    lib.psl_plan_tables.restype = C.c_int
    lib.psl_plan_tables.argtypes = [C.c_void_p, P(C.c_void_p), P(C.c_void_p)]
    lib.psl_sample_batch.restype = C.c_int
    lib.psl_sample_batch.argtypes = [C.c_void_p, C.c_int32, C.c_int32, P(Launch)]
    lib.psl_flush_schedule.restype = C.c_int
    lib.psl_flush_schedule.argtypes = [C.c_void_p, C.c_uint32, P(Flush)]
    lib.psl_reset.restype = C.c_int
    lib.psl_reset.argtypes = [C.c_void_p]
    lib.psl_destroy.restype = None
    lib.psl_destroy.argtypes = [C.c_void_p]
    lib.psl_last_error.restype = C.c_char_p
    lib.psl_last_error.argtypes = [C.c_void_p]
    lib.psl_kernel_launches.restype = C.c_uint64
    lib.psl_kernel_launches.argtypes = [C.c_void_p]
    lib.psl_profile_enable.restype = C.c_int
    lib.psl_profile_enable.argtypes = [C.c_void_p, C.c_int32]
    lib.psl_profile_read.restype = C.c_int
    lib.psl_profile_read.argtypes = [C.c_void_p, P(Profile)]
    lib.psl_count_static.restype = C.c_int
    lib.psl_count_static.argtypes = [P(Config), C.c_void_p, C.c_uint64, C.c_void_p, C.c_void_p]
    _lib = lib
    return lib


def _geometry(g: Dict) -> Geometry:
    return Geometry(g["z_src"], g["z_plane"], g["z_jaw_x"], g["z_jaw_y"], g["z_map"], g["z_iso"])


def make_config(grid: Dict, geometry: Dict, mode: int, max_records: int, max_host_records: Optional[int] = None,
                max_beam_records: int = 0, max_chunks: int = 0, flags: int = 0, device: int = 0,
                max_launch_records: int = 0, apr_seed: int = 0):
    """(Config, keepalive) for a workloads-style grid / geometry description."""
    edges = None
    if grid["ebin_mode"] == EBIN_EDGES:
        edges = np.ascontiguousarray(grid["e_edges"], dtype=np.float32)
    cfg = Config()
    cfg.struct_size = C.sizeof(Config)
    cfg.mode = mode
    cfg.n_types = grid["n_types"]
    cfg.ebin_mode = grid["ebin_mode"]
    cfg.n_ebins = grid["n_ebins"]
    cfg.e_min, cfg.e_max = grid["e_min"], grid["e_max"]
    cfg.e_edges = None if edges is None else edges.ctypes.data
    cfg.n_xbins, cfg.n_ybins = grid["n_xbins"], grid["n_ybins"]
    cfg.x_min, cfg.y_min, cfg.dx, cfg.dy = grid["x_min"], grid["y_min"], grid["dx"], grid["dy"]
    cfg.geom = _geometry(geometry)
    cfg.max_records = max_records
    cfg.max_host_records = max_records if max_host_records is None else max_host_records
    cfg.max_beam_records = max_beam_records
    cfg.max_chunks = max_chunks
    cfg.flags = flags
    cfg.apr_seed = apr_seed
    cfg.max_launch_records = max_launch_records
    cfg.device = device
    return cfg, edges


def workspace_bytes(grid: Dict, geometry: Dict, mode: int, max_records: int, **kw) -> int:
    """psl_workspace_bytes for a configuration (0 = the library rejects it).  Needs no GPU."""
    cfg, _keep = make_config(grid, geometry, mode, max_records, **kw)
    return int(load_library().psl_workspace_bytes(C.byref(cfg)))


def psl_roi_from_jaws(geometry: Dict, jaws, margin: float):
    """HOST-only C-ABI call; returns (status, (x1, x2, y1, y2))."""
    lib = load_library()
    g = _geometry(geometry)
    b = Beam()
    b.has_jaws = 1
    b.jaw_x1, b.jaw_x2, b.jaw_y1, b.jaw_y2 = jaws
    out = (C.c_float * 4)()
    rc = lib.psl_roi_from_jaws(C.byref(g), C.byref(b), margin, C.byref(out))
    return rc, tuple(float(v) for v in out)


def count_static(grid: Dict, geometry: Dict, records, counts, totals=None, stream=None):
    """psl_count_static: counts[K] of DEVICE-resident records with no allocation in the library.  ``records`` is a
    contiguous CUDA tensor of packed 28-byte records, ``counts`` a CUDA int32 tensor of K entries and ``totals`` an
    optional CUDA int64 tensor of 4 entries (n_in, n_invalid, n_outside_grid, n_binned), all on the same device; the
    work is enqueued on ``stream`` (default: torch's current stream of that device) and not waited for."""
    import torch

    lib = load_library()
    if not (isinstance(records, torch.Tensor) and records.is_cuda and records.is_contiguous()):
        raise TypeError("records must be a contiguous CUDA tensor")
    nbytes = records.numel() * records.element_size()
    assert nbytes % RECORD_BYTES == 0
    n_keys = grid["n_types"] * grid["n_ebins"] * grid["n_xbins"] * grid["n_ybins"]
    assert counts.is_cuda and counts.is_contiguous() and counts.dtype == torch.int32 and counts.numel() == n_keys
    assert counts.device == records.device
    if totals is not None:
        assert totals.is_cuda and totals.is_contiguous() and totals.dtype == torch.int64 and totals.numel() == 4
        assert totals.device == records.device
    cfg, _edges = make_config(grid, geometry, MODE_ONTHEFLY, 1, 0, device=records.device.index)
    st = stream if stream is not None else torch.cuda.current_stream(records.device)
    cfg.stream = st.cuda_stream
    rc = lib.psl_count_static(C.byref(cfg), records.data_ptr(), nbytes // RECORD_BYTES, counts.data_ptr(),
                              None if totals is None else totals.data_ptr())
    if rc != 0:
        raise PslError(rc, lib.psl_last_error(None).decode())


class PslContext:
    """One phase-space on one GPU.  Mirrors the C-ABI; owns the workspace tensor."""

    def __init__(self, grid: Dict, geometry: Dict, mode: int, max_records: int,
                 max_host_records: Optional[int] = None, max_beam_records: int = 0, max_chunks: int = 0,
                 flags: int = 0, device: int = 0, stream=None, max_launch_records: int = 0, apr_seed: int = 0):
        import torch

        self.torch = torch
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise PslError(5, "no CUDA device: libpsl_b200 has no CPU path")
        self.device = torch.device("cuda", device)
        self.cfg, self._edges = make_config(grid, geometry, mode, max_records, max_host_records, max_beam_records,
                                            max_chunks, flags, device, max_launch_records, apr_seed)
        need = int(self.lib.psl_workspace_bytes(C.byref(self.cfg)))
        if need == 0:
            raise PslError(1, self.lib.psl_last_error(None).decode())
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(need, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.cfg.stream = self.stream.cuda_stream
        self.cfg.workspace = self.workspace.data_ptr()
        self.cfg.workspace_bytes = need
        self._h = C.c_void_p()
        rc = self.lib.psl_create(C.byref(self.cfg), C.byref(self._h))
        if rc != 0:
            self._h = C.c_void_p()
            raise PslError(rc, self.lib.psl_last_error(None).decode())
        self._keep = []       # borrowed device chunks, host sources in flight
        self._beam_keep = {}  # id(source array) -> (source array, device fluence map)
        self.n_types, self.n_ebins = grid["n_types"], grid["n_ebins"]
        self.n_pos = grid["n_xbins"] * grid["n_ybins"]
        self.n_keys = self.n_types * self.n_ebins * self.n_pos

    # -- helpers -------------------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != 0:
            raise PslError(rc, self.lib.psl_last_error(self._h).decode())

    def _view(self, ptr: Optional[int], count: int, dtype):
        """zero-copy tensor over a borrowed workspace pointer"""
        if not ptr:
            return None
        size = 1 if dtype == self.torch.uint8 else 4
        off = ptr - self.workspace.data_ptr()
        assert 0 <= off and off + size * count <= self.workspace.numel()
        return self.workspace[off:off + size * count].view(dtype)

    def beam(self, b: Optional[Dict]) -> Optional[Beam]:
        """marshal a workloads-style beam dict; uploads the fluence map to the device"""
        if b is None:
            return None
        torch = self.torch
        out = Beam()
        j, r = b.get("jaws"), b.get("roi")
        out.has_jaws = 0 if j is None else 1
        if j is not None:
            out.jaw_x1, out.jaw_x2, out.jaw_y1, out.jaw_y2 = j
        fl = b.get("fluence")
        if fl is not None:
            # one device copy per source array, reused by later builds of the same beam (bounded: the oldest go first)
            hit = self._beam_keep.get(id(fl))
            if hit is not None and hit[0] is fl:
                dev_fl = hit[1]
            else:
                src = torch.from_numpy(np.ascontiguousarray(fl, dtype=np.float32)) if isinstance(fl, np.ndarray) else fl
                with torch.cuda.stream(self.stream):
                    dev_fl = src.to(self.device, dtype=torch.float32).contiguous()
                while len(self._beam_keep) >= 64:
                    self._beam_keep.pop(next(iter(self._beam_keep)))
                self._beam_keep[id(fl)] = (fl, dev_fl)
            out.fluence = dev_fl.data_ptr()
            out.map_ny, out.map_nx = dev_fl.shape
        out.map_x0, out.map_y0 = b.get("map_x0", 0.0), b.get("map_y0", 0.0)
        out.map_dx, out.map_dy = b.get("map_dx", 1.0), b.get("map_dy", 1.0)
        out.has_roi = 0 if r is None else 1
        if r is not None:
            out.roi_x1, out.roi_x2, out.roi_y1, out.roi_y2 = r
        out.mu_weight = b.get("mu_weight", 1.0)
        out.gantry_deg = b.get("gantry_deg", 0.0)
        out.coll_deg = b.get("coll_deg", 0.0)
        out.couch_deg = b.get("couch_deg", 0.0)
        return out

    # -- the C-ABI calls -----------------------------------------------------------------------------
    def load_chunk(self, records, mem_kind: Optional[int] = None):
        """records: numpy structured/uint8 array (pageable), torch CPU tensor (pinned if it is) or torch CUDA
        tensor (borrowed).  The object is kept alive until reset()."""
        torch = self.torch
        if isinstance(records, np.ndarray):
            assert records.flags.c_contiguous
            ptr, nbytes, kind = records.ctypes.data, records.nbytes, MEM_PAGEABLE
        elif isinstance(records, torch.Tensor):
            assert records.is_contiguous()
            ptr, nbytes = records.data_ptr(), records.numel() * records.element_size()
            kind = MEM_DEVICE if records.is_cuda else (MEM_PINNED if records.is_pinned() else MEM_PAGEABLE)
        else:
            raise TypeError("records must be a numpy array or a torch tensor")
        if mem_kind is not None:
            kind = mem_kind
        assert nbytes % RECORD_BYTES == 0
        self._keep.append(records)
        self._check(self.lib.psl_load_chunk(self._h, ptr, nbytes // RECORD_BYTES, kind))

    def wait_loads(self):
        self._check(self.lib.psl_wait_loads(self._h))

    def build_batches(self, beam=None, want_stats: bool = False) -> Optional[Dict]:
        b = beam if isinstance(beam, Beam) or beam is None else self.beam(beam)
        st = Stats() if want_stats else None
        self._check(self.lib.psl_build_batches(self._h, None if b is None else C.byref(b),
                                               None if st is None else C.byref(st)))
        return st.as_dict() if want_stats else None

    def get_stats(self) -> Dict:
        st = Stats()
        self._check(self.lib.psl_get_stats(self._h, C.byref(st)))
        return st.as_dict()

    def get_batch(self, t: int = -1, ie: int = -1) -> Dict:
        """dict of zero-copy tensors for batch (t, ie); (-1, -1) = the whole output"""
        torch = self.torch
        b = Batch()
        self._check(self.lib.psl_get_batch(self._h, t, ie, C.byref(b)))
        out = {"first": b.first, "count": b.count, "n_bins": b.n_bins}
        for name in ("E", "x", "y", "u", "v", "w", "wt", "xp", "yp"):
            out[name] = self._view(getattr(b, name), b.count, torch.float32)
        out["src_index"] = self._view(b.src_index, b.count, torch.int32)
        out["bin_offsets"] = self._view(b.bin_offsets, b.n_bins + 1, torch.int32)
        return out

    def get_tables(self):
        """(counts[K], offsets[K+1]) as zero-copy int32 tensors (values are uint32)"""
        c, o, k = C.c_void_p(), C.c_void_p(), C.c_uint32()
        self._check(self.lib.psl_get_tables(self._h, C.byref(c), C.byref(o), C.byref(k)))
        return self._view(c.value, k.value, self.torch.int32), self._view(o.value, k.value + 1, self.torch.int32)

    def roi_bins(self, beam) -> tuple:
        b = beam if isinstance(beam, Beam) else self.beam(beam)
        out = (C.c_int32 * 4)()
        self._check(self.lib.psl_roi_bins(self._h, C.byref(b), C.byref(out)))
        return tuple(int(v) for v in out)

    # -- plan -> launch lists -> transport-ready particles; capacity-N shipments -----------------
    def plan_set(self, beams, n_simulate: int, seed: int = 1, rr_group: int = 4,
                 phantom=((-15.0, -15.0, -15.0), (15.0, 15.0, 15.0))):
        """returns (N_total^psl, [launch-list length of every (type, energy) division])"""
        arr = (Beam * len(beams))(*[b if isinstance(b, Beam) else self.beam(b) for b in beams])
        p = Plan()
        p.struct_size = C.sizeof(Plan)
        p.n_beams = len(beams)
        p.beams = C.cast(arr, C.c_void_p)
        p.n_simulate, p.seed, p.rr_group = n_simulate, seed, rr_group
        p.phantom_lo[:] = phantom[0]
        p.phantom_hi[:] = phantom[1]
        total = C.c_uint64()
        lens = C.POINTER(C.c_uint64)()
        self._check(self.lib.psl_plan_set(self._h, C.byref(p), C.byref(total), C.byref(lens)))
        nb = self.n_types * self.n_ebins
        return int(total.value), [int(lens[i]) for i in range(nb)]

    def plan_tables(self):
        b, m = C.c_void_p(), C.c_void_p()
        self._check(self.lib.psl_plan_tables(self._h, C.byref(b), C.byref(m)))
        return self._view(b.value, self.n_keys, self.torch.int32), self._view(m.value, self.n_keys, self.torch.int32)

    def sample_batch(self, t: int, ie: int) -> Dict:
        torch = self.torch
        l = Launch()
        self._check(self.lib.psl_sample_batch(self._h, t, ie, C.byref(l)))
        out = {"n_list": l.n_list, "n_launch": l.n_launch, "n_jaw_rejected": l.n_jaw_rejected,
               "n_zero_weight": l.n_zero_weight, "n_missed": l.n_missed}
        out["slot"] = self._view(l.slot, l.n_list, torch.int32)
        out["beam"] = self._view(l.beam, l.n_list, torch.uint8)
        for name in ("E", "X", "Y", "Z", "U", "V", "W", "wt"):
            out[name] = self._view(getattr(l, name), l.n_launch, torch.float32)
        out["src_index"] = self._view(l.src_index, l.n_launch, torch.int32)
        out["beam_of"] = self._view(l.beam_of, l.n_launch, torch.uint8)
        return out

    def flush_schedule(self, capacity: int) -> Dict:
        f = Flush()
        self._check(self.lib.psl_flush_schedule(self._h, capacity, C.byref(f)))
        return {"n_events": f.n_events, "key": self._view(f.key, f.n_events, self.torch.int32),
                "first": self._view(f.first, f.n_events, self.torch.int32),
                "count": self._view(f.count, f.n_events, self.torch.int32)}

    def reset(self):
        self._check(self.lib.psl_reset(self._h))
        self._keep.clear()

    def kernel_launches(self) -> int:
        return int(self.lib.psl_kernel_launches(self._h))

    def profile_enable(self, on: bool = True):
        self._check(self.lib.psl_profile_enable(self._h, 1 if on else 0))

    def profile_read(self) -> Dict:
        """{class: (total ms, timed launches)} since the last read; synchronises"""
        p = Profile()
        self._check(self.lib.psl_profile_read(self._h, C.byref(p)))
        return {name: (p.ms[i], int(p.launches[i])) for i, name in enumerate(K_CLASSES)}

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h:
            self.lib.psl_destroy(self._h)
            self._h = C.c_void_p()
        self._keep = []
        self._beam_keep = {}

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()
