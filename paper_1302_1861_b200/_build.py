"""Build libpsl_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libpsl_b200.so")
SOURCES = ["psl_api.cu"]
HEADERS = ["psl_device.cuh", "psl_partition.cuh", "psl_bigtile.cuh", "psl_index.cuh", "psl_index_big.cuh", "psl_beam.cuh", "psl_compact.cuh", "psl_plan.cuh", "psl_static.cuh", os.path.join("..", "..", "include", "psl.h")]

#: -fmad=false: no FMA contraction anywhere in the TU (the arithmetic contract of include/psl.h);
#: division and square root stay IEEE (nvcc defaults -prec-div=true -prec-sqrt=true, no fast-math).
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-fmad=false",
    "-Xcompiler", "-fPIC,-Wall", "-shared",
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(os.path.normpath(d)) > t for d in deps)


def build_library(force: bool = False, verbose: bool = False) -> str:
    """Compile the CUDA library next to the package; returns its path."""
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc, *NVCC_FLAGS, "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
        if verbose:
            cmd += ["-Xptxas", "-v"]
        subprocess.run(cmd, check=True)
    return LIB
