"""ctypes binding of include/sl1m.h -- same names, argument marshalling only."""
from __future__ import annotations

import ctypes
import dataclasses
import os
import re
from typing import Optional

import numpy as np

from .build import LIB, build_library

GAUSS_PARAXIAL = 0   # eq (16)
GAUSS_WIDEFIELD = 1  # eq (17)
GAINS_ON_DEVICE = 1
PHASE_FP64 = 2
DENSE_FORWARD = 4
NO_PERSISTENT = 8

_HEADER = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "sl1m.h")


class Sl1mError(RuntimeError):
    def __init__(self, status: int, name: str, detail: str):
        super().__init__(f"{name} ({status}): {detail}")
        self.status, self.name, self.detail = status, name, detail


class _PlanInfo(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in (
        "n_pix_padded", "n_tiles", "gaussian", "gains", "fwd_rv", "fwd_vis_tiles", "fwd_pixel_splits",
        "fwd_tiles_per_split", "fwd_poly_per16", "adj_rp", "adj_pixel_groups", "adj_vis_splits",
        "adj_chunks_per_split", "adj_poly_per16", "mufu_per_term_mufu_path", "fwd_packed_pairs",
        "adj_packed_pairs", "phase_fp64")] + [("phase_span_rad", ctypes.c_float), ("zero_skip", ctypes.c_int32), ("persistent", ctypes.c_int32), ("adj_mufu_per_term", ctypes.c_int32)]


class _Peaks(ctypes.Structure):
    _fields_ = [("n_sm", ctypes.c_int32)] + [(n, ctypes.c_double) for n in (
        "sm_clock_mhz", "clock64_mhz", "mufu_per_s", "mufu_per_clk_sm", "mufu_cos_per_clk_sm", "ffma_per_s", "ffma_per_clk_sm",
        "ffma2_lanes_per_s", "ffma2_lanes_per_clk_sm", "coissue_mufu_per_clk_sm", "coissue_ffma2_lanes_per_clk_sm",
        "coissue_cycles_per_iter", "coissue_adj_mufu_per_clk_sm", "dfma_per_s", "dfma_per_clk_sm")]


class _QtLevel(ctypes.Structure):
    _fields_ = [("n_pix", ctypes.c_int64), ("L", ctypes.c_float), ("n_iter_done", ctypes.c_int32),
                ("l2_term", ctypes.c_double), ("l1_term", ctypes.c_double), ("nnz", ctypes.c_int64),
                ("seconds", ctypes.c_double)]


class _SolveInfo(ctypes.Structure):
    _fields_ = [("n_iter_done", ctypes.c_int32), ("L_used", ctypes.c_float),
                ("l2_term", ctypes.c_double), ("l1_term", ctypes.c_double), ("nnz", ctypes.c_int64)]


@dataclasses.dataclass
class SolveInfo:
    n_iter_done: int
    L_used: float
    l2_term: float
    l1_term: float
    nnz: int


def library_path() -> str:
    return LIB


def exported_symbols() -> list:
    """Every function name include/sl1m.h declares."""
    txt = open(_HEADER).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(sl1m_[a-z0-9_]+)\s*\(", txt)))


_lib = None


def load_library():
    """Load libsl1m.so, rebuilding it first when it is missing or older than any of its sources
    (build_library's mtime check; a no-op when up to date).  SL1M_LIBRARY names a prebuilt library
    to load as is.  Raises if the library cannot be had."""
    global _lib
    if _lib is not None:
        return _lib
    path = os.environ.get("SL1M_LIBRARY") or build_library(force=bool(os.environ.get("SL1M_REBUILD")))
    lib = ctypes.CDLL(path)
    vp, i64, i32, f32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_float
    lib.sl1m_plan_create.argtypes = [ctypes.POINTER(vp), i64, vp, vp, vp, i64, vp, vp, vp, i32, vp,
                                     ctypes.c_int, ctypes.c_uint32]
    lib.sl1m_forward.argtypes = [vp, vp, vp, vp]
    lib.sl1m_adjoint.argtypes = [vp, vp, vp, vp]
    lib.sl1m_forward_host.argtypes = [vp, vp, vp, vp]
    lib.sl1m_adjoint_host.argtypes = [vp, vp, vp, vp]
    lib.sl1m_max_eig.argtypes = [vp, ctypes.c_int, ctypes.POINTER(f32), vp]
    lib.sl1m_solve.argtypes = [vp, vp, f32, f32, ctypes.c_int, ctypes.c_int, vp, vp, vp,
                               ctypes.POINTER(_SolveInfo), vp]
    lib.sl1m_solve_host.argtypes = [vp, vp, f32, f32, ctypes.c_int, ctypes.c_int, vp, vp,
                                    ctypes.POINTER(_SolveInfo), vp]
    lib.sl1m_solve_tol.argtypes = [vp, vp, f32, f32, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_int,
                                   vp, vp, vp, ctypes.POINTER(_SolveInfo), vp]
    lib.sl1m_solve_stop.argtypes = [vp, vp, f32, f32, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                    ctypes.c_int, vp, vp, vp, ctypes.POINTER(_SolveInfo), vp]
    lib.sl1m_solve_stop_batch.argtypes = [vp, vp, vp, vp, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                          ctypes.c_int, vp, vp, vp, vp, vp]
    lib.sl1m_fista_begin.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.sl1m_fista_step.argtypes = [vp, ctypes.c_int, vp, vp]
    lib.sl1m_fista_image.argtypes = [vp, vp, ctypes.POINTER(ctypes.c_int32), vp]
    lib.sl1m_dirty_image.argtypes = [vp, vp, f32, vp, vp]
    lib.sl1m_plan_set_channels.argtypes = [vp, ctypes.c_int32, vp]
    lib.sl1m_plan_n_chan.argtypes = [vp]
    lib.sl1m_plan_n_chan.restype = ctypes.c_int32
    lib.sl1m_max_eig_batch.argtypes = [vp, ctypes.c_int, vp, vp]
    lib.sl1m_solve_batch.argtypes = [vp, vp, vp, vp, ctypes.c_int, ctypes.c_int, vp, vp, vp, vp, vp]
    f64 = ctypes.c_double
    lib.sl1m_quadtree_refine.argtypes = [i64, vp, vp, vp, vp, f64, f64, i64, vp, vp, vp, vp, vp,
                                         ctypes.POINTER(i64), ctypes.POINTER(i64)]
    lib.sl1m_quadtree_solve.argtypes = [i64, vp, vp, i64, vp, vp, vp, ctypes.c_int, f64, f64, f64, ctypes.c_int,
                                        f32, f32, ctypes.c_int, ctypes.c_int, f64, ctypes.c_int, i64, vp, vp, vp,
                                        vp, ctypes.POINTER(i64), ctypes.POINTER(_QtLevel),
                                        ctypes.POINTER(ctypes.c_int), vp]
    lib.sl1m_quadtree_solve_gains.argtypes = [i64, vp, vp, vp, vp, i32, vp, i64, vp, vp, vp, ctypes.c_int, f64, f64, f64,
                                              ctypes.c_int, f32, f32, ctypes.c_int, ctypes.c_int, f64, ctypes.c_int, i64,
                                              vp, vp, vp, vp, ctypes.POINTER(i64), ctypes.POINTER(_QtLevel),
                                              ctypes.POINTER(ctypes.c_int), vp]
    lib.sl1m_plan_describe.argtypes = [vp, ctypes.POINTER(_PlanInfo)]
    lib.sl1m_forward_active_pixels.argtypes = [vp, vp, vp]
    lib.sl1m_measure_peaks.argtypes = [ctypes.POINTER(_Peaks), vp]
    lib.sl1m_forward_noalloc.argtypes = [i64, vp, i64, vp, vp, vp, vp, vp]
    lib.sl1m_debug_check.argtypes = []
    lib.sl1m_debug_bounds_build.argtypes = []
    lib.sl1m_debug_poke_past_end.argtypes = [vp]
    lib.sl1m_launch_count.argtypes = [vp]
    lib.sl1m_launch_count.restype = i64
    lib.sl1m_plan_n_vis.argtypes = [vp]
    lib.sl1m_plan_n_vis.restype = i64
    lib.sl1m_plan_n_pix.argtypes = [vp]
    lib.sl1m_plan_n_pix.restype = i64
    lib.sl1m_destroy.argtypes = [vp]
    lib.sl1m_destroy.restype = None
    lib.sl1m_status_string.argtypes = [ctypes.c_int]
    lib.sl1m_status_string.restype = ctypes.c_char_p
    lib.sl1m_last_error.argtypes = []
    lib.sl1m_last_error.restype = ctypes.c_char_p
    _lib = lib
    return lib


_DEBUG_CHECK = bool(os.environ.get("SL1M_DEBUG_CHECK"))   # verify the canary bands of a -DSL1M_BOUNDS build after every call


def _check(st: int):
    lib = load_library()
    if st == 0 and _DEBUG_CHECK:
        st = lib.sl1m_debug_check()
    if st != 0:
        raise Sl1mError(st, lib.sl1m_status_string(st).decode(), lib.sl1m_last_error().decode())


def _np_ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _stream_ptr(stream) -> Optional[int]:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _dev_ptr(t, dtype, numel: int, name: str):
    import torch
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()
            and t.numel() == numel):
        raise ValueError(f"{name}: need a contiguous CUDA tensor of {dtype} with {numel} elements")
    return ctypes.c_void_p(t.data_ptr())


def measure_peaks(stream=None) -> dict:
    """sl1m_measure_peaks: MUFU / FFMA / FFMA2 issue rates of this GPU (roofline denominators)."""
    pk = _Peaks()
    _check(load_library().sl1m_measure_peaks(ctypes.byref(pk), _stream_ptr(stream)))
    return {n: (int(getattr(pk, n)) if n == "n_sm" else float(getattr(pk, n))) for n, _ in _Peaks._fields_}


NOALLOC_MAX_VIS = 524288      # SL1M_NOALLOC_MAX_VIS
NOALLOC_MAX_PIX = 16777216    # SL1M_NOALLOC_MAX_PIX


def forward_noalloc(uvw, l, m, x, out, stream=None):
    """sl1m_forward_noalloc: v = M x (eq 9, delta pixels, unit gains) without a plan and without the library asking the
    driver for memory -- for callers that cannot allocate at this point (busy real-time streams that a cudaMalloc would
    stall, device memory owned by another pool, fixed-footprint services).  Everything is a CUDA tensor the caller made
    beforehand: uvw [n_vis][3] float64, l / m [n_pix] float64, x [n_pix] float32, out [n_vis] complex64 (overwritten and
    returned; this function creates no tensor).  The partial sums live in one 4 MiB array inside the library, shared by
    every call on the device: at most NOALLOC_MAX_VIS visibilities per call, and do not let two calls overlap on the
    GPU.  Make the first call per device at start-up (it looks up the array's address); see include/sl1m.h."""
    import torch
    n_vis, n_pix = int(out.numel()), int(x.numel())
    _check(load_library().sl1m_forward_noalloc(
        n_vis, _dev_ptr(uvw, torch.float64, 3 * n_vis, "uvw"), n_pix, _dev_ptr(l, torch.float64, n_pix, "l"),
        _dev_ptr(m, torch.float64, n_pix, "m"), _dev_ptr(x, torch.float32, n_pix, "x"),
        _dev_ptr(out, torch.complex64, n_vis, "out"), _stream_ptr(stream)))
    return out


def quadtree_refine(l, m, side, I, frac: float, min_side: float):
    """sl1m_quadtree_refine (pure host code).  Returns (l, m, side, I0, parent, n_refined)."""
    l, m, side = (np.ascontiguousarray(a, dtype=np.float64) for a in (l, m, side))
    I = np.ascontiguousarray(I, dtype=np.float32)
    n = int(l.shape[0])
    cap = 4 * n
    lo, mo, so = np.empty(cap), np.empty(cap), np.empty(cap)
    xo, po = np.empty(cap, np.float32), np.empty(cap, np.int64)
    n_out, n_ref = ctypes.c_int64(0), ctypes.c_int64(0)
    _check(load_library().sl1m_quadtree_refine(n, _np_ptr(l), _np_ptr(m), _np_ptr(side), _np_ptr(I), float(frac),
                                               float(min_side), cap, _np_ptr(lo), _np_ptr(mo), _np_ptr(so),
                                               _np_ptr(xo), _np_ptr(po), ctypes.byref(n_out), ctypes.byref(n_ref)))
    k = n_out.value
    return lo[:k].copy(), mo[:k].copy(), so[:k].copy(), xo[:k].copy(), po[:k].copy(), int(n_ref.value)


def quadtree_solve(uvw, vis, l0, m0, side0, n_levels: int, frac: float, min_side: float, lam: float,
                   n_pow: int = 30, L_safety: float = 1.05, max_iter: int = 1000, tol: float = 1e-6,
                   check_every: int = 10, sigma_factor: float = 1.0, gauss_model: int = 1, capacity: int = None,
                   stream=None, ant_p=None, ant_q=None, gains0=None):
    """sl1m_quadtree_solve (sl1m_quadtree_solve_gains when gains0 [n_ant][n0] complex64 is given): coarse-to-fine /
    adaptive quadtree driver.  Host arrays in, host arrays out: dict(l, m, side, x, levels=[...])."""
    uvw = np.ascontiguousarray(uvw, dtype=np.float64)
    vis = np.ascontiguousarray(vis, dtype=np.complex64)
    l0, m0, side0 = (np.ascontiguousarray(a, dtype=np.float64) for a in (l0, m0, side0))
    n0 = int(l0.shape[0])
    cap = int(capacity) if capacity is not None else n0 * 4 ** max(int(n_levels) - 1, 0)
    lo, mo, so, xo = np.empty(cap), np.empty(cap), np.empty(cap), np.empty(cap, np.float32)
    levels = (_QtLevel * max(int(n_levels), 1))()
    n_out, n_done = ctypes.c_int64(0), ctypes.c_int(0)
    if gains0 is not None:
        g = np.ascontiguousarray(gains0, dtype=np.complex64)
        ap = np.ascontiguousarray(ant_p, dtype=np.int32)
        aq = np.ascontiguousarray(ant_q, dtype=np.int32)
        if g.ndim != 2 or g.shape[1] != n0 or ap.shape[0] != uvw.shape[0] or aq.shape[0] != uvw.shape[0]:
            raise ValueError("gains0 must be [n_ant][n0]; ant_p, ant_q [n_vis]")
        _check(load_library().sl1m_quadtree_solve_gains(
            int(uvw.shape[0]), _np_ptr(uvw), _np_ptr(vis), _np_ptr(ap), _np_ptr(aq), int(g.shape[0]), _np_ptr(g), n0,
            _np_ptr(l0), _np_ptr(m0), _np_ptr(side0), int(n_levels), float(frac), float(min_side), float(sigma_factor),
            int(gauss_model), float(lam), float(L_safety), int(n_pow), int(max_iter), float(tol), int(check_every), cap,
            _np_ptr(lo), _np_ptr(mo), _np_ptr(so), _np_ptr(xo), ctypes.byref(n_out), levels, ctypes.byref(n_done),
            _stream_ptr(stream)))
    else:
        _check(load_library().sl1m_quadtree_solve(
            int(uvw.shape[0]), _np_ptr(uvw), _np_ptr(vis), n0, _np_ptr(l0), _np_ptr(m0), _np_ptr(side0), int(n_levels),
            float(frac), float(min_side), float(sigma_factor), int(gauss_model), float(lam), float(L_safety), int(n_pow),
            int(max_iter), float(tol), int(check_every), cap, _np_ptr(lo), _np_ptr(mo), _np_ptr(so), _np_ptr(xo),
            ctypes.byref(n_out), levels, ctypes.byref(n_done), _stream_ptr(stream)))
    k = n_out.value
    lv = [dict(n_pix=int(q.n_pix), L=float(q.L), n_iter_done=int(q.n_iter_done), l2_term=float(q.l2_term),
               l1_term=float(q.l1_term), nnz=int(q.nnz), seconds=float(q.seconds)) for q in levels[:n_done.value]]
    return dict(l=lo[:k].copy(), m=mo[:k].copy(), side=so[:k].copy(), x=xo[:k].copy(), levels=lv)


class Plan:
    """sl1m_plan_create / sl1m_destroy.  Inputs are host arrays (numpy); see include/sl1m.h."""

    def __init__(self, uvw, l, m, sigma=None, ant_p=None, ant_q=None, gains=None,
                 gauss_model: int = GAUSS_WIDEFIELD, phase_fp64: bool = False, dense_forward: bool = False,
                 no_persistent: bool = False):
        import torch
        self._h = None
        lib = load_library()
        uvw = np.ascontiguousarray(uvw, dtype=np.float64).reshape(-1, 3)
        l = np.ascontiguousarray(l, dtype=np.float64).ravel()
        m = np.ascontiguousarray(m, dtype=np.float64).ravel()
        if m.shape != l.shape:
            raise ValueError("l and m differ in length")
        sg = None if sigma is None else np.ascontiguousarray(sigma, dtype=np.float64).ravel()
        if sg is not None and sg.shape != l.shape:
            raise ValueError("sigma and l differ in length")
        n_ant, g, flags = 0, None, (PHASE_FP64 if phase_fp64 else 0) | (DENSE_FORWARD if dense_forward else 0) | (NO_PERSISTENT if no_persistent else 0)
        ap = aq = None
        gptr = None
        if gains is not None:
            ap = np.ascontiguousarray(ant_p, dtype=np.int32).ravel()
            aq = np.ascontiguousarray(ant_q, dtype=np.int32).ravel()
            if ap.shape[0] != uvw.shape[0] or aq.shape[0] != uvw.shape[0]:
                raise ValueError("ant_p/ant_q and uvw differ in length")
            if isinstance(gains, torch.Tensor):
                if not (gains.is_cuda and gains.dtype == torch.complex64 and gains.is_contiguous()):
                    raise ValueError("device gains must be a contiguous CUDA complex64 tensor")
                g = gains
                n_ant = int(g.shape[0])
                gptr = ctypes.c_void_p(g.data_ptr())
                flags |= GAINS_ON_DEVICE
            else:
                g = np.ascontiguousarray(gains, dtype=np.complex64)
                n_ant = int(g.shape[0])
                gptr = _np_ptr(g)
            if g.ndim != 2 or g.shape[1] != l.shape[0]:
                raise ValueError("gains must be [n_ant][n_pix]")
        h = ctypes.c_void_p()
        _check(lib.sl1m_plan_create(ctypes.byref(h), uvw.shape[0], _np_ptr(uvw), _np_ptr(ap), _np_ptr(aq),
                                    l.shape[0], _np_ptr(l), _np_ptr(m), _np_ptr(sg), n_ant, gptr,
                                    int(gauss_model), flags))
        self._h = h
        self.n_vis, self.n_pix = int(uvw.shape[0]), int(l.shape[0])
        self.n_chan = 1

    def set_channels(self, scale):
        """sl1m_plan_set_channels: a batch of len(scale) channels, channel c on uvw * scale[c].
        forward/adjoint then take and return [n_chan][.] tensors; use max_eig_batch / solve_batch."""
        sc = np.ascontiguousarray(scale, dtype=np.float64).ravel()
        _check(load_library().sl1m_plan_set_channels(self._h, int(sc.shape[0]), _np_ptr(sc)))
        self.n_chan = int(load_library().sl1m_plan_n_chan(self._h))
        return self

    def _shape(self, n):
        return (n,) if self.n_chan == 1 else (self.n_chan, n)

    @classmethod
    def from_workload(cls, wl, gains_device=None, dense_forward: bool = False, no_persistent: bool = False,
                      phase_fp64: bool = False):
        g = wl.gains if gains_device is None else gains_device
        return cls(wl.uvw, wl.l, wl.m, wl.sigma, wl.ant_p, wl.ant_q, g, wl.gauss_model, dense_forward=dense_forward,
                   no_persistent=no_persistent, phase_fp64=phase_fp64)

    def close(self):
        if self._h is not None:
            load_library().sl1m_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- device-pointer calls (torch tensors) ----
    def forward(self, x, out=None, stream=None):
        """sl1m_forward: x float32 [n_pix] -> complex64 [n_vis]."""
        import torch
        if out is None:
            out = torch.empty(self._shape(self.n_vis), dtype=torch.complex64, device=x.device)
        _check(load_library().sl1m_forward(self._h, _dev_ptr(x, torch.float32, self.n_chan * self.n_pix, "x"),
                                           _dev_ptr(out, torch.complex64, self.n_chan * self.n_vis, "out"),
                                           _stream_ptr(stream)))
        return out

    def adjoint(self, r, out=None, stream=None):
        """sl1m_adjoint: r complex64 [n_vis] -> float32 [n_pix]."""
        import torch
        if out is None:
            out = torch.empty(self._shape(self.n_pix), dtype=torch.float32, device=r.device)
        _check(load_library().sl1m_adjoint(self._h, _dev_ptr(r, torch.complex64, self.n_chan * self.n_vis, "r"),
                                           _dev_ptr(out, torch.float32, self.n_chan * self.n_pix, "out"),
                                           _stream_ptr(stream)))
        return out

    def max_eig(self, n_pow: int = 30, stream=None) -> float:
        L = ctypes.c_float(0.0)
        _check(load_library().sl1m_max_eig(self._h, int(n_pow), ctypes.byref(L), _stream_ptr(stream)))
        return float(L.value)

    def max_eig_batch(self, n_pow: int = 30, stream=None) -> np.ndarray:
        """sl1m_max_eig_batch: one L per channel."""
        L = np.zeros(self.n_chan, np.float32)
        _check(load_library().sl1m_max_eig_batch(self._h, int(n_pow), _np_ptr(L), _stream_ptr(stream)))
        return L

    def solve_batch(self, vis, lam, L, n_iter: int, n_pow: int = 30, x0=None, out=None, trace=None,
                    want_info: bool = True, stream=None):
        """sl1m_solve_batch: vis [n_chan][n_vis] complex64, lam / L per channel (scalars are broadcast).
        Returns (x [n_chan][n_pix], [SolveInfo per channel] or None)."""
        import torch
        C = self.n_chan
        lam_a = np.ascontiguousarray(np.broadcast_to(np.asarray(lam, np.float32), (C,)))
        L_a = np.ascontiguousarray(np.broadcast_to(np.asarray(L, np.float32), (C,)))
        if out is None:
            out = torch.empty((C, self.n_pix), dtype=torch.float32, device=vis.device)
        infos = (_SolveInfo * C)()
        _check(load_library().sl1m_solve_batch(
            self._h, _dev_ptr(vis, torch.complex64, C * self.n_vis, "vis"), _np_ptr(lam_a), _np_ptr(L_a), int(n_pow),
            int(n_iter), _dev_ptr(x0, torch.float32, C * self.n_pix, "x0"),
            _dev_ptr(out, torch.float32, C * self.n_pix, "out"),
            _dev_ptr(trace, torch.float64, C * 3 * max(int(n_iter), 1), "trace") if trace is not None else None,
            ctypes.cast(infos, ctypes.c_void_p) if want_info else None, _stream_ptr(stream)))
        res = [SolveInfo(i.n_iter_done, i.L_used, i.l2_term, i.l1_term, i.nnz) for i in infos] if want_info else None
        return out, res

    def solve(self, vis, lam: float, L: float = 0.0, n_pow: int = 30, n_iter: int = 100, x0=None,
              out=None, trace=None, want_info: bool = True, stream=None):
        """sl1m_solve.  Returns (x, SolveInfo or None)."""
        import torch
        if out is None:
            out = torch.empty(self.n_pix, dtype=torch.float32, device=vis.device)
        info = _SolveInfo()
        _check(load_library().sl1m_solve(
            self._h, _dev_ptr(vis, torch.complex64, self.n_vis, "vis"), float(lam), float(L), int(n_pow),
            int(n_iter), _dev_ptr(x0, torch.float32, self.n_pix, "x0"),
            _dev_ptr(out, torch.float32, self.n_pix, "out"),
            _dev_ptr(trace, torch.float64, 3 * max(int(n_iter), 0), "trace") if trace is not None else None,
            ctypes.byref(info) if want_info else None, _stream_ptr(stream)))
        res = SolveInfo(info.n_iter_done, info.L_used, info.l2_term, info.l1_term, info.nnz) if want_info else None
        return out, res

    def solve_tol(self, vis, lam: float, L: float, max_iter: int, tol: float, check_every: int = 1,
                  n_pow: int = 30, x0=None, out=None, trace=None, stream=None):
        """sl1m_solve_tol: FISTA until the total error changes by <= tol (relative) or max_iter.
        Returns (x, SolveInfo); SolveInfo.n_iter_done is the iteration it stopped at."""
        import torch
        if out is None:
            out = torch.empty(self.n_pix, dtype=torch.float32, device=vis.device)
        info = _SolveInfo()
        _check(load_library().sl1m_solve_tol(
            self._h, _dev_ptr(vis, torch.complex64, self.n_vis, "vis"), float(lam), float(L), int(n_pow),
            int(max_iter), float(tol), int(check_every), _dev_ptr(x0, torch.float32, self.n_pix, "x0"),
            _dev_ptr(out, torch.float32, self.n_pix, "out"),
            _dev_ptr(trace, torch.float64, 3 * max(int(max_iter), 0), "trace") if trace is not None else None,
            ctypes.byref(info), _stream_ptr(stream)))
        return out, SolveInfo(info.n_iter_done, info.L_used, info.l2_term, info.l1_term, info.nnz)

    def solve_stop(self, vis, lam: float, L: float, max_iter: int, tol: float = -1.0, nnz_tol: float = -1.0,
                   check_every: int = 1, n_pow: int = 30, x0=None, out=None, trace=None, stream=None):
        """sl1m_solve_stop: FISTA until the total error changes by <= tol (relative) OR the number of non-zero
        pixels by <= nnz_tol (relative), decided on the device; a negative tolerance switches that rule off.
        Returns (x, SolveInfo); SolveInfo.n_iter_done is the iteration it stopped at."""
        import torch
        if out is None:
            out = torch.empty(self.n_pix, dtype=torch.float32, device=vis.device)
        info = _SolveInfo()
        _check(load_library().sl1m_solve_stop(
            self._h, _dev_ptr(vis, torch.complex64, self.n_vis, "vis"), float(lam), float(L), int(n_pow),
            int(max_iter), float(tol), float(nnz_tol), int(check_every),
            _dev_ptr(x0, torch.float32, self.n_pix, "x0"), _dev_ptr(out, torch.float32, self.n_pix, "out"),
            _dev_ptr(trace, torch.float64, 3 * max(int(max_iter), 0), "trace") if trace is not None else None,
            ctypes.byref(info), _stream_ptr(stream)))
        return out, SolveInfo(info.n_iter_done, info.L_used, info.l2_term, info.l1_term, info.nnz)

    def solve_stop_batch(self, vis, lam, L, max_iter: int, tol: float = -1.0, nnz_tol: float = -1.0,
                         check_every: int = 1, n_pow: int = 30, x0=None, out=None, trace=None, stream=None):
        """sl1m_solve_stop_batch: every channel stops on its own.  Returns (x [n_chan][n_pix], [SolveInfo])."""
        import torch
        C = self.n_chan
        lam_a = np.ascontiguousarray(np.broadcast_to(np.asarray(lam, np.float32), (C,)))
        L_a = np.ascontiguousarray(np.broadcast_to(np.asarray(L, np.float32), (C,)))
        if out is None:
            out = torch.empty((C, self.n_pix), dtype=torch.float32, device=vis.device)
        infos = (_SolveInfo * C)()
        _check(load_library().sl1m_solve_stop_batch(
            self._h, _dev_ptr(vis, torch.complex64, C * self.n_vis, "vis"), _np_ptr(lam_a), _np_ptr(L_a), int(n_pow),
            int(max_iter), float(tol), float(nnz_tol), int(check_every),
            _dev_ptr(x0, torch.float32, C * self.n_pix, "x0"), _dev_ptr(out, torch.float32, C * self.n_pix, "out"),
            _dev_ptr(trace, torch.float64, C * 3 * max(int(max_iter), 1), "trace") if trace is not None else None,
            ctypes.cast(infos, ctypes.c_void_p), _stream_ptr(stream)))
        return out, [SolveInfo(i.n_iter_done, i.L_used, i.l2_term, i.l1_term, i.nnz) for i in infos]

    def fista_begin(self, vis, lam, L, x0=None, stream=None):
        """sl1m_fista_begin: start a stepped FISTA run.  `vis` is borrowed by the library: the binding keeps a
        reference so the tensor outlives the run."""
        import torch
        C = self.n_chan
        lam_a = np.ascontiguousarray(np.broadcast_to(np.asarray(lam, np.float32), (C,)))
        L_a = np.ascontiguousarray(np.broadcast_to(np.asarray(L, np.float32), (C,)))
        _check(load_library().sl1m_fista_begin(
            self._h, _dev_ptr(vis, torch.complex64, C * self.n_vis, "vis"), _np_ptr(lam_a), _np_ptr(L_a),
            _dev_ptr(x0, torch.float32, C * self.n_pix, "x0"), _stream_ptr(stream)))
        self._fista_vis = vis
        return self

    def fista_step(self, n_iter: int = 1, trace=None, stream=None):
        """sl1m_fista_step: n_iter more iterations of the run begun by fista_begin (asynchronous)."""
        import torch
        _check(load_library().sl1m_fista_step(
            self._h, int(n_iter),
            _dev_ptr(trace, torch.float64, self.n_chan * 3 * max(int(n_iter), 1), "trace") if trace is not None else None,
            _stream_ptr(stream)))
        return self

    def fista_image(self, out=None, stream=None):
        """sl1m_fista_image: (I_k, k) of the stepped run."""
        import torch
        if out is None:
            out = torch.empty(self._shape(self.n_pix), dtype=torch.float32, device="cuda")
        k = ctypes.c_int32(0)
        _check(load_library().sl1m_fista_image(self._h, _dev_ptr(out, torch.float32, self.n_chan * self.n_pix, "out"),
                                               ctypes.byref(k), _stream_ptr(stream)))
        return out, int(k.value)

    def dirty_image(self, vis, scale: float = None, out=None, stream=None):
        """sl1m_dirty_image: max(0, scale * Re M^H vis); scale defaults to 1/n_vis.  Batched plans: [n_chan][.]."""
        import torch
        if out is None:
            out = torch.empty(self._shape(self.n_pix), dtype=torch.float32, device=vis.device)
        _check(load_library().sl1m_dirty_image(
            self._h, _dev_ptr(vis, torch.complex64, self.n_chan * self.n_vis, "vis"),
            float(1.0 / self.n_vis if scale is None else scale),
            _dev_ptr(out, torch.float32, self.n_chan * self.n_pix, "out"), _stream_ptr(stream)))
        return out

    # ---- host-buffer calls (numpy / pinned torch CPU tensors) ----
    @staticmethod
    def _host_ptr(a, dtype, numel, name):
        import torch
        if a is None:
            return None
        if isinstance(a, torch.Tensor):
            if a.is_cuda or not a.is_contiguous() or a.numel() != numel:
                raise ValueError(f"{name}: need a contiguous CPU tensor with {numel} elements")
            return ctypes.c_void_p(a.data_ptr())
        if not (isinstance(a, np.ndarray) and a.dtype == dtype and a.flags.c_contiguous and a.size == numel):
            raise ValueError(f"{name}: need a contiguous {dtype} array with {numel} elements")
        return _np_ptr(a)

    def forward_host(self, x_host, out_host, stream=None):
        _check(load_library().sl1m_forward_host(self._h, self._host_ptr(x_host, np.float32, self.n_pix, "x"),
                                                self._host_ptr(out_host, np.complex64, self.n_vis, "out"),
                                                _stream_ptr(stream)))
        return out_host

    def adjoint_host(self, r_host, out_host, stream=None):
        _check(load_library().sl1m_adjoint_host(self._h, self._host_ptr(r_host, np.complex64, self.n_vis, "r"),
                                                self._host_ptr(out_host, np.float32, self.n_pix, "out"),
                                                _stream_ptr(stream)))
        return out_host

    def solve_host(self, vis_host, lam, L, n_iter, out_host, n_pow=30, x0_host=None, want_info=True, stream=None):
        info = _SolveInfo()
        _check(load_library().sl1m_solve_host(
            self._h, self._host_ptr(vis_host, np.complex64, self.n_vis, "vis"), float(lam), float(L), int(n_pow),
            int(n_iter), self._host_ptr(x0_host, np.float32, self.n_pix, "x0"),
            self._host_ptr(out_host, np.float32, self.n_pix, "out"),
            ctypes.byref(info) if want_info else None, _stream_ptr(stream)))
        res = SolveInfo(info.n_iter_done, info.L_used, info.l2_term, info.l1_term, info.nnz) if want_info else None
        return out_host, res

    def describe(self) -> dict:
        """sl1m_plan_describe: launch configuration and instruction mix."""
        info = _PlanInfo()
        _check(load_library().sl1m_plan_describe(self._h, ctypes.byref(info)))
        return {n: (float(getattr(info, n)) if n == "phase_span_rad" else int(getattr(info, n)))
                for n, _ in _PlanInfo._fields_}

    def forward_active_pixels(self, stream=None):
        """sl1m_forward_active_pixels: pixels the most recently packed forward input streams (per channel)."""
        out = np.zeros(self.n_chan, dtype=np.int64)
        _check(load_library().sl1m_forward_active_pixels(self._h, _np_ptr(out), _stream_ptr(stream)))
        return int(out[0]) if self.n_chan == 1 else out

    @property
    def launch_count(self) -> int:
        return int(load_library().sl1m_launch_count(self._h))
