"""Build libsl1m.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "csrc", "sl1m.cu")
SRC_QT = os.path.join(_HERE, "csrc", "sl1m_quadtree.cu")
SRC_PK = os.path.join(_HERE, "csrc", "sl1m_peaks.cu")
SRC_NA = os.path.join(_HERE, "csrc", "sl1m_noalloc.cu")     # sl1m_forward_noalloc: static device scratch, no cudaMalloc
DEPS = [SRC, SRC_QT, SRC_PK, SRC_NA, os.path.join(_HERE, "csrc", "sl1m_kernels.cuh"), os.path.join(_HERE, "csrc", "sl1m_epilogue.cuh"), os.path.join(_HERE, "csrc", "sl1m_persist.cuh"), os.path.join(_HERE, "csrc", "sl1m_internal.h"),
        os.path.join(os.path.dirname(_HERE), "include", "sl1m.h")]
LIB = os.path.join(_HERE, "libsl1m.so")
LIB_BOUNDS = os.path.join(_HERE, "libsl1m_bounds.so")      # debug build: canary bands + asserted prefetches (-DSL1M_BOUNDS)

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "shared"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def build_library(force: bool = False, verbose: bool = False, bounds: bool = False) -> str:
    lib = LIB_BOUNDS if bounds else LIB
    stale = not os.path.exists(lib) or any(os.path.getmtime(lib) < os.path.getmtime(d) for d in DEPS)
    if force or stale:
        tmp = lib + f".tmp{os.getpid()}"
        extra = os.environ.get("SL1M_NVCC_EXTRA", "").split() + (["-DSL1M_BOUNDS"] if bounds else [])   # SL1M_NVCC_EXTRA: tuning -D flags
        cmd = [_nvcc(), *NVCC_FLAGS, *extra, "-o", tmp, SRC, SRC_QT, SRC_PK, SRC_NA]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        subprocess.check_call(cmd)
        os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build_library(force=True, verbose=True))
