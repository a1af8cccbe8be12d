"""fp64 CPU oracle for the SL1M hot path -- TEST INFRASTRUCTURE, not the product.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs
may import this package.  It shares nothing with `paper_1310_2078_b200/` (the CUDA path) and
never imports it.  The arithmetic lives in `sl1m_oracle.c` (plain C, `double complex`, literal
transcription of PAPER.md eqs (9), (16), (17), (18) and the FISTA listing); this file only
compiles it with gcc and marshals numpy arrays through ctypes.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sl1m_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """Compile sl1m_oracle.c -> liboracle.so (gcc -O2 -fopenmp, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fno-fast-math", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Problem(ctypes.Structure):
    _fields_ = [
        ("n_vis", ctypes.c_int64), ("uvw", ctypes.c_void_p),
        ("ant_p", ctypes.c_void_p), ("ant_q", ctypes.c_void_p),
        ("n_pix", ctypes.c_int64), ("l", ctypes.c_void_p), ("m", ctypes.c_void_p),
        ("sigma", ctypes.c_void_p), ("n_ant", ctypes.c_int32), ("gains", ctypes.c_void_p),
        ("gauss_model", ctypes.c_int32),
    ]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        P = ctypes.POINTER(_Problem)
        vp, i64, i32, f64 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_entry.argtypes = [P, i64, i64, vp]
        lib.oracle_forward.argtypes = [P, vp, i64, vp, vp]
        lib.oracle_adjoint.argtypes = [P, vp, i64, vp, vp]
        lib.oracle_max_eig.argtypes = [P, i32]
        lib.oracle_max_eig.restype = f64
        lib.oracle_threshold.argtypes = [f64, f64]
        lib.oracle_threshold.restype = f64
        lib.oracle_fista.argtypes = [P, vp, f64, f64, i32, vp, vp, vp, vp]
        lib.oracle_fista_tol.argtypes = [P, vp, f64, f64, i32, f64, f64, i32, vp, vp, vp, vp, vp]
        lib.oracle_fista_tol.restype = i32
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def threshold(x: float, d: float) -> float:
    """eq (18)."""
    return float(_load().oracle_threshold(float(x), float(d)))


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


class Oracle:
    """One measurement problem (uvw, antenna pairs, pixel list, sigma, gains, Gaussian model)."""

    def __init__(self, uvw, l, m, sigma=None, ant_p=None, ant_q=None, gains=None, gauss_model=1):
        self.uvw = np.ascontiguousarray(uvw, dtype=np.float64).reshape(-1, 3)
        self.l = np.ascontiguousarray(l, dtype=np.float64).ravel()
        self.m = np.ascontiguousarray(m, dtype=np.float64).ravel()
        self.n_vis, self.n_pix = self.uvw.shape[0], self.l.shape[0]
        assert self.m.shape[0] == self.n_pix
        self.sigma = None if sigma is None else np.ascontiguousarray(sigma, dtype=np.float64).ravel()
        self.gains = None
        self.ant_p = self.ant_q = None
        self.n_ant = 0
        if gains is not None:
            g = np.asarray(gains)
            assert g.ndim == 2 and g.shape[1] == self.n_pix and np.iscomplexobj(g)
            self.n_ant = g.shape[0]
            # exact widening of the caller's complex64 table; layout [n_ant][n_pix][2]
            self.gains = np.ascontiguousarray(g.astype(np.complex128)).view(np.float64)
            self.ant_p = np.ascontiguousarray(ant_p, dtype=np.int32)
            self.ant_q = np.ascontiguousarray(ant_q, dtype=np.int32)
            assert self.ant_p.shape[0] == self.n_vis and self.ant_q.shape[0] == self.n_vis
        self.gauss_model = int(gauss_model)
        self._c = _Problem(self.n_vis, _ptr(self.uvw), _ptr(self.ant_p), _ptr(self.ant_q),
                           self.n_pix, _ptr(self.l), _ptr(self.m), _ptr(self.sigma),
                           self.n_ant, _ptr(self.gains), self.gauss_model)

    @classmethod
    def from_workload(cls, wl):
        return cls(wl.uvw, wl.l, wl.m, wl.sigma, wl.ant_p, wl.ant_q, wl.gains, wl.gauss_model)

    # O1
    def entry(self, j: int, k: int) -> complex:
        out = np.zeros(2)
        _load().oracle_entry(ctypes.byref(self._c), int(j), int(k), _ptr(out))
        return complex(out[0], out[1])

    def dense(self) -> np.ndarray:
        """The full matrix M (tiny problems only)."""
        M = np.empty((self.n_vis, self.n_pix), dtype=np.complex128)
        for j in range(self.n_vis):
            for k in range(self.n_pix):
                M[j, k] = self.entry(j, k)
        return M

    # O2
    def forward(self, x, rows=None) -> np.ndarray:
        x = np.ascontiguousarray(x, dtype=np.float64).ravel()
        assert x.shape[0] == self.n_pix
        if rows is not None:
            rows = np.ascontiguousarray(rows, dtype=np.int64)
            n = rows.shape[0]
        else:
            n = self.n_vis
        v = np.zeros((n, 2))
        _load().oracle_forward(ctypes.byref(self._c), _ptr(x), n, _ptr(rows), _ptr(v))
        return v[:, 0] + 1j * v[:, 1]

    # O3
    def adjoint(self, r, cols=None) -> np.ndarray:
        r = np.ascontiguousarray(np.asarray(r, dtype=np.complex128)).view(np.float64)
        assert r.shape[0] == 2 * self.n_vis
        if cols is not None:
            cols = np.ascontiguousarray(cols, dtype=np.int64)
            n = cols.shape[0]
        else:
            n = self.n_pix
        g = np.zeros(n)
        _load().oracle_adjoint(ctypes.byref(self._c), _ptr(r), n, _ptr(cols), _ptr(g))
        return g

    # O4
    def max_eig(self, n_pow: int = 30) -> float:
        return float(_load().oracle_max_eig(ctypes.byref(self._c), int(n_pow)))

    # O5
    def fista(self, V, lam: float, L: float, n_iter: int, x0=None, want_trace: bool = False,
              want_info: bool = True):
        """want_info=False passes info3 = NULL: the C routine then skips its closing forward for
        ||M I_K - V||^2 (one whole apply at config 5)."""
        V = np.ascontiguousarray(np.asarray(V, dtype=np.complex128)).view(np.float64)
        assert V.shape[0] == 2 * self.n_vis
        x0a = None if x0 is None else np.ascontiguousarray(x0, dtype=np.float64)
        x = np.zeros(self.n_pix)
        trace = np.zeros((max(n_iter, 1), 3)) if want_trace else None
        info = np.zeros(3) if want_info else None
        _load().oracle_fista(ctypes.byref(self._c), _ptr(V), float(lam), float(L), int(n_iter),
                             _ptr(x0a), _ptr(x), _ptr(trace), _ptr(info))
        out = dict(x=x)
        if want_info:
            out.update(l2_term=float(info[0]), l1_term=float(info[1]), nnz=int(info[2]))
        if want_trace:
            out["trace"] = trace[:n_iter]
        return out

    # O5 + the termination rules of PAPER.md:194 / :239 (readings R21: total error; R24: number of non-zeros)
    def fista_tol(self, V, lam: float, L: float, max_iter: int, tol: float, check_every: int = 1, x0=None,
                  nnz_tol: float = -1.0):
        V = np.ascontiguousarray(np.asarray(V, dtype=np.complex128)).view(np.float64)
        assert V.shape[0] == 2 * self.n_vis
        x0a = None if x0 is None else np.ascontiguousarray(x0, dtype=np.float64)
        x = np.zeros(self.n_pix)
        trace = np.zeros((max(max_iter, 1), 3))
        info = np.zeros(3)
        E = np.zeros(max(max_iter, 1))
        n_done = _load().oracle_fista_tol(ctypes.byref(self._c), _ptr(V), float(lam), float(L), int(max_iter),
                                          float(tol), float(nnz_tol), int(check_every), _ptr(x0a), _ptr(x), _ptr(trace),
                                          _ptr(info), _ptr(E))
        return dict(x=x, n_iter_done=int(n_done), trace=trace[:n_done], E=E[:n_done], l2_term=float(info[0]),
                    l1_term=float(info[1]), nnz=int(info[2]))

    # PAPER.md:327 "use the dirty image as the initial condition": the back-projected data,
    # scaled and clipped to the positive orthant the solver lives in (reading R22).
    def dirty_image(self, V, scale: float):
        return np.maximum(0.0, float(scale) * self.adjoint(V))


# ---------------------------------------------------------------------------------------------
# NEXT-3: coarse-to-fine / adaptive quadtree driver, PAPER.md:329-339 (section 4.5, Fig. 10).
# "the system is solved at a low resolution, and pixels where emission is detected are then
#  subdivided.  This process continues until the resolution limit of the telescope is reached."
# Fig. 10: "refinement of all pixels greater than 1 per cent of the maximum", every level with the
# same lambda.  The paper fixes nothing else; reading R23 states what is assumed:
#   * a pixel is a square of side s_k centred on (l_k, m_k); it is refined iff
#     I_k > frac * max_j I_j and s_k / 2 >= min_side; a refined pixel is replaced IN PLACE by its
#     four children (side s_k/2, centres l_k -/+ s_k/4, m_k -/+ s_k/4, l fastest as in eqs (5)-(6));
#     all other pixels stay as they are (leaves of mixed size in one solve);
#   * "upscale the previously calculated solution": each child starts from I_k/4
#     (flux conserving), an unrefined pixel from I_k;
#   * frac < 0 refines every pixel: the plain coarse-to-fine strategy of PAPER.md:329;
#   * a pixel that can still be split (s_k / 2 >= min_side) is a Gaussian pixel of
#     sigma_k = sigma_factor * s_k (eq 16/17) -- a delta pixel at the centre of a square much larger
#     than the resolution does not describe the emission inside it; a pixel at the resolution
#     limit (s_k / 2 < min_side), and every pixel when sigma_factor == 0, is a delta pixel (eq 9);
#   * L is re-estimated at every level (n_pow rounds of O4, times L_safety).
# Plain Python loops on purpose: this is the definition, not an implementation.
# ---------------------------------------------------------------------------------------------
def quadtree_refine(l, m, side, I, frac: float, min_side: float):
    """One refinement step.  Returns (l, m, side, I0, parent, n_refined)."""
    l, m, side, I = (np.asarray(a, dtype=np.float64) for a in (l, m, side, I))
    top = float(I.max()) if I.size else 0.0
    thr = float(frac) * top
    lo, mo, so, xo, po = [], [], [], [], []
    n_refined = 0
    for k in range(I.shape[0]):
        half = side[k] / 2.0
        if top > 0.0 and I[k] > thr and half >= min_side:
            n_refined += 1
            q = side[k] / 4.0
            for dm in (-q, +q):
                for dl in (-q, +q):
                    lo.append(l[k] + dl)
                    mo.append(m[k] + dm)
                    so.append(half)
                    xo.append(I[k] / 4.0)
                    po.append(k)
        else:
            lo.append(l[k])
            mo.append(m[k])
            so.append(side[k])
            xo.append(I[k])
            po.append(k)
    return (np.array(lo), np.array(mo), np.array(so), np.array(xo), np.array(po, dtype=np.int64), n_refined)


def quadtree_solve(uvw, V, l0, m0, side0, n_levels: int, frac: float, min_side: float, lam: float,
                   n_pow: int, L_safety: float, max_iter: int, tol: float, check_every: int = 1,
                   sigma_factor: float = 0.0, gauss_model: int = 1, ant_p=None, ant_q=None, gains0=None):
    """The driver: solve, refine, warm-start, repeat (at most n_levels solves).
    gains0 [n_ant][n0] (with ant_p, ant_q): direction-dependent gains on the starting pixel list.  The paper says
    nothing about gains under refinement; reading R25: a child inherits the gain column of its parent
    (the beam is taken as constant over a pixel that is being split)."""
    l, m, side = (np.asarray(a, dtype=np.float64).copy() for a in (l0, m0, side0))
    gains = None if gains0 is None else np.asarray(gains0).astype(np.complex64)
    x0 = None
    levels = []
    for level in range(int(n_levels)):
        sigma = np.where(side / 2.0 >= min_side, sigma_factor * side, 0.0) if sigma_factor > 0 else None
        o = Oracle(uvw, l, m, sigma, ant_p, ant_q, gains, gauss_model=gauss_model)
        L = o.max_eig(n_pow) * L_safety
        r = o.fista_tol(V, lam, L, max_iter, tol, check_every, x0=x0)
        I = r["x"]
        levels.append(dict(n_pix=int(l.shape[0]), L=L, n_iter_done=r["n_iter_done"], l2_term=r["l2_term"],
                           l1_term=r["l1_term"], nnz=r["nnz"]))
        if level == n_levels - 1:
            break
        l2, m2, s2, x2, parent, n_ref = quadtree_refine(l, m, side, I, frac, min_side)
        if n_ref == 0:
            break
        l, m, side, x0 = l2, m2, s2, x2
        if gains is not None:
            gains = np.ascontiguousarray(gains[:, parent])            # reading R25
    return dict(l=l, m=m, side=side, x=I, levels=levels)
