"""B200-native SL1M hot path (arXiv:1310.2078): direct measurement operator A, its adjoint A^H
and the positivity-constrained FISTA solver, as hand-written sm_100a CUDA kernels behind a C ABI
(`include/sl1m.h`, built into `libsl1m.so`).  This package is a thin ctypes binding with the
same names -- argument marshalling only; PyTorch provides device memory and streams.

There is no CPU fallback: using the binding without the built library or without a CUDA device
raises.
"""
from .binding import (  # noqa: F401
    GAUSS_PARAXIAL, GAUSS_WIDEFIELD, PHASE_FP64, DENSE_FORWARD, NO_PERSISTENT, Plan, Sl1mError, SolveInfo, build_library, library_path,
    load_library, exported_symbols, quadtree_refine, quadtree_solve, measure_peaks, forward_noalloc, NOALLOC_MAX_VIS, NOALLOC_MAX_PIX,
)
