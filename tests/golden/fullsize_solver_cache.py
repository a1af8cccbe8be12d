"""Full-size FISTA runs of the fp64 oracle on BASELINE.json's configs 2-5, cached for the GPU parity tests.

north_star asks for "full SL1M solves matching the fp64 oracle ... on all five configs"; SURVEY.md 8(d)
(SURVEY.md:520-528) fixes how: K = 50 / 25 / 5 full oracle iterations on configs 2 / 3 / 4 and K = 2 on config 5,
computed once OFFLINE on CPU cores and cached by a hash of the inputs, because one config-5 oracle apply is
4.3e11 terms (tens of minutes on a few cores).  The algorithm is the listing at PAPER.md:188-192 with eq (18),
PAPER.md:194-197.

This script imports ONLY `oracle` and `workloads` (plus numpy / hashlib): no value it stores has seen the CUDA path.

    python tests/golden/fullsize_solver_cache.py 2 3 4        # ~1 h on 8 cores
    python tests/golden/fullsize_solver_cache.py 5            # several hours on 8 cores

Per config it writes `tests/golden/solver_fullsize_config<c>.npz`:
    x        fp32 [n_pix]    the oracle's I_K (rounded once, 6e-8 relative: far below the 1e-3 tolerance)
    trace    fp64 [K][3]     per iteration {||M y_k - V||^2, sum I_k, nnz I_k}          (reading R20)
    V        complex64 [n_vis]  measured data V = M x_true (+ blobs) + noise, formed by the oracle
    lam, L, n_pow, K, input_hash, seconds_*, threads

Recipe (the same for every config):
    V    as in tests/test_gpu_parity.py::_measured (oracle forward of the truth, rounded to complex64)
    lam  workloads.fista_lambda (3 sigma_n sqrt(N_v)); the noiseless config 4: 0.01 max|Re M^H V|
    L    1.05 x oracle.max_eig(n_pow), n_pow = 30 / 30 / 10 / 2 for configs 2 / 3 / 4 / 5.  Power iteration
         approaches lambda_max from below, so the config-5 value (n_pow = 2: each round costs two full applies) is
         a stated step constant, not a converged one; for a K = 2 parity run only "both sides use the same L,
         of the right order" matters.
    K    workloads' n_iter: 50 / 25 / 5 / 2
`input_hash` = sha256 over the raw workload arrays (uvw, ant_p, ant_q, l, m, sigma, gains, x_true, blobs, noise) and
the recipe constants; the GPU tests recompute it from `make_workload` and FAIL when it differs (a changed input
recipe invalidates the cache).
"""
from __future__ import annotations

import hashlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

N_POW = {2: 30, 3: 30, 4: 10, 5: 2}
L_SAFETY = 1.05
LAMBDA_DIRTY_FRACTION = 0.01          # config 4 (noiseless): lambda = 0.01 max|Re M^H V|
RECIPE_VERSION = 1


def cache_path(cid: int) -> str:
    return os.path.join(HERE, f"solver_fullsize_config{cid}.npz")


def input_hash(wl) -> str:
    """sha256 of everything the cached run depends on (raw inputs + recipe constants)."""
    h = hashlib.sha256()
    h.update(f"v{RECIPE_VERSION} cid={wl.cid} K={wl.n_iter} n_pow={N_POW[wl.cid]} safety={L_SAFETY!r} "
             f"lamfrac={LAMBDA_DIRTY_FRACTION!r} sigma_n={wl.sigma_n!r} gauss_model={wl.gauss_model}".encode())
    arrays = [wl.uvw, wl.ant_p, wl.ant_q, wl.l, wl.m, wl.sigma, wl.gains, wl.x_true, wl.noise]
    if wl.truth_extra is not None:
        arrays += [wl.truth_extra[k] for k in ("l", "m", "sigma", "flux")]
    for a in arrays:
        if a is None:
            h.update(b"<none>")
        else:
            a = np.ascontiguousarray(a)
            h.update(str(a.dtype).encode() + str(a.shape).encode())
            h.update(a.tobytes())
    return h.hexdigest()


def measured(o, wl):
    """V = M x_true (+ blobs through a separate truth pixel list, eq 17) + noise, rounded to complex64."""
    import oracle
    V = o.forward(wl.x_true)
    if wl.truth_extra is not None:
        te = wl.truth_extra
        V = V + oracle.Oracle(wl.uvw, te["l"], te["m"], te["sigma"], gauss_model=1).forward(te["flux"])
    return (V + wl.noise).astype(np.complex64)


def run(cid: int) -> None:
    import oracle
    from workloads import fista_lambda, make_workload

    wl = make_workload(cid)
    o = oracle.Oracle.from_workload(wl)
    ih = input_hash(wl)
    part = cache_path(cid) + ".partial.npz"      # L survives an interrupted run (config 5: hours)
    print(f"[config {cid}] n_pix={wl.n_pix} n_vis={wl.n_vis} threads={oracle.num_threads()} hash={ih[:16]}", flush=True)
    t0 = time.time()
    V = measured(o, wl)
    t_v = time.time() - t0
    print(f"[config {cid}] V formed in {t_v:.1f} s", flush=True)

    L = None
    t_L = 0.0
    if os.path.exists(part):
        z = np.load(part)
        if str(z["input_hash"]) == ih:
            L, t_L = float(z["L"]), float(z["seconds_L"])
            print(f"[config {cid}] L = {L:.9g} taken from {os.path.basename(part)}", flush=True)
    if L is None:
        t0 = time.time()
        L = L_SAFETY * o.max_eig(N_POW[cid])
        t_L = time.time() - t0
        np.savez(part, input_hash=ih, L=L, seconds_L=t_L)
        print(f"[config {cid}] L = {L:.9g} ({N_POW[cid]} power rounds, {t_L:.1f} s)", flush=True)

    if wl.sigma_n > 0:
        lam = fista_lambda(wl)
    else:
        lam = LAMBDA_DIRTY_FRACTION * float(np.max(np.abs(o.adjoint(V))))
    print(f"[config {cid}] lambda = {lam:.9g}; running K = {wl.n_iter} oracle iterations", flush=True)

    t0 = time.time()
    ref = o.fista(V, lam, L, wl.n_iter, want_trace=True, want_info=False)
    t_s = time.time() - t0
    print(f"[config {cid}] solve {t_s:.1f} s; nnz(I_K) = {int(np.count_nonzero(ref['x']))}", flush=True)

    np.savez_compressed(
        cache_path(cid), x=ref["x"].astype(np.float32), trace=ref["trace"], V=V, lam=np.float64(lam),
        L=np.float64(L), n_pow=N_POW[cid], K=wl.n_iter, input_hash=ih, seconds_V=t_v, seconds_L=t_L,
        seconds_solve=t_s, threads=oracle.num_threads())
    os.remove(part)
    print(f"[config {cid}] wrote {cache_path(cid)} ({os.path.getsize(cache_path(cid)) / 1e6:.2f} MB)", flush=True)


if __name__ == "__main__":
    for c in (int(a) for a in sys.argv[1:]) if len(sys.argv) > 1 else (2, 3, 4):
        run(c)
