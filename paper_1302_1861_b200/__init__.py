"""B200-native phase-space source hot path (arXiv 1302.1861): thin Python binding over libpsl_b200.so.

The product is the CUDA library behind include/psl.h.  This package only marshals arguments
(``binding.PslContext`` mirrors the C-ABI call for call) and uses PyTorch for device memory and
streams.  There is no CPU fallback: importing works anywhere, but creating a context without the
built library or without a CUDA device raises.
"""
from .binding import (  # noqa: F401
    EBIN_EDGES, EBIN_LINEAR, MEM_DEVICE, MEM_PAGEABLE, MEM_PINNED, MODE_INDEX, MODE_ONTHEFLY, OUT_PROJ,
    DROP_ZERO_WEIGHT, NO_COMPACT, APR, PslContext, PslError, exported_symbols, library_path, load_library, psl_roi_from_jaws,
    workspace_bytes, count_static, STATIC_MAX_KEYS, STATIC_SCRATCH_BYTES,
)

__all__ = [
    "PslContext", "PslError", "load_library", "library_path", "exported_symbols", "workspace_bytes",
    "psl_roi_from_jaws", "MODE_ONTHEFLY", "MODE_INDEX", "EBIN_LINEAR", "EBIN_EDGES", "MEM_PAGEABLE", "MEM_PINNED",
    "MEM_DEVICE", "OUT_PROJ", "DROP_ZERO_WEIGHT", "NO_COMPACT", "APR", "count_static", "STATIC_MAX_KEYS",
    "STATIC_SCRATCH_BYTES",
]
