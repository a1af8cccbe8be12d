"""Pins for the oracle's solver pieces O4 (power iteration) and O5 (FISTA + T^d): hand values,
the textbook t-sequence, numpy eigenvalues, the DFT-lattice one-step case, KKT conditions, an
independent NNLS solve, the Beck-Teboulle bound, and sparse recovery.  CPU only."""
import math
import os

import numpy as np
import scipy.optimize

import oracle
from workloads import make_workload

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    out = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                out.append([float(t) for t in line.split()])
    return out


def test_threshold_hand_values():
    """eq (18), incl. the x = d tie and negatives (reading R12)."""
    for x, d, want in _rows("threshold_hand_values.txt"):
        assert oracle.threshold(x, d) == want


def test_momentum_follows_the_textbook_t_sequence():
    """Reading R8.  One pixel at the phase centre, N_v visibilities all equal to c: A = ones,
    Re A^H A = N_v.  With L = 2 N_v and lambda = 0 the gradient step is I_k = (y_k + c)/2, so
    the iterates follow from the momentum coefficients alone; those come from the golden
    t-sequence (Beck & Teboulle 2009a), not from the oracle."""
    gold = _rows("fista_t_sequence.txt")
    beta = [row[2] for row in gold]
    nv, c = 7, 3.0
    uvw = np.random.default_rng(2).uniform(-100, 100, (nv, 3))
    o = oracle.Oracle(uvw, [0.0], [0.0])
    V = np.full(nv, c, dtype=complex)
    I_prev, y = 0.0, 0.0
    for k in range(1, 5):
        I = (y + c) / 2
        got = o.fista(V, lam=0.0, L=2.0 * nv, n_iter=k)["x"][0]
        assert abs(got - I) < 2e-6 * c, (k, got, I)      # golden betas carry 6 digits
        y = I + beta[k - 1] * (I - I_prev)
        I_prev = I
    # t_2 is the golden ratio: exact check of the "/2" (the listing prints "/t_{k+1}")
    t2 = (1 + math.sqrt(5)) / 2
    assert abs(gold[1][1] - t2) < 1e-6


def _tiny(rng, n_vis=60, n_pix=40, wmax=50.0):
    uvw = rng.uniform(-1, 1, (n_vis, 3)) * np.array([400.0, 400.0, wmax])
    l = rng.uniform(-0.02, 0.02, n_pix)
    m = rng.uniform(-0.02, 0.02, n_pix)
    return oracle.Oracle(uvw, l, m)


def test_max_eig_against_numpy_eigvalsh_and_bounds():
    """Readings R10/R11: power iteration on x -> Re A^H A x converges FROM BELOW to
    lambda_max(Re M^H M) (numpy.linalg.eigvalsh); bounds max_k sum_j|M_jk|^2 <= L <= ||M||_F^2;
    a single-pixel plan gives L = sum_j |M_j0|^2 = N_v/n^2."""
    rng = np.random.default_rng(21)
    o = _tiny(rng)
    M = o.dense()
    H = (M.conj().T @ M).real
    lam_max = np.linalg.eigvalsh(H)[-1]
    L30 = o.max_eig(30)
    L400 = o.max_eig(400)
    assert L30 <= lam_max * (1 + 1e-12) and L400 <= lam_max * (1 + 1e-12)
    assert abs(L400 - lam_max) < 1e-6 * lam_max
    assert L30 > 0.9 * lam_max
    col = (np.abs(M) ** 2).sum(0)
    assert col.max() <= L400 * (1 + 1e-9) and L400 <= (np.abs(M) ** 2).sum() * (1 + 1e-12)
    # the complex lambda_max(M^H M) is larger: the distinction in R10 is not cosmetic
    assert np.linalg.eigvalsh(M.conj().T @ M)[-1] >= lam_max * (1 - 1e-12)
    l0, m0 = 0.3, -0.2
    o1 = oracle.Oracle(o.uvw, [l0], [m0])
    assert abs(o1.max_eig(3) - o.n_vis / (1 - l0 * l0 - m0 * m0)) < 1e-9


def test_fista_one_step_on_the_dft_lattice():
    """Reading R13: N x N grid, w = 0, full DFT lattice, gains g = sqrt(n) on both antennas
    (cancelling 1/n)  =>  Re A^H A = N^2 Id, L = N^2, and FISTA lands on the exact minimiser
    T^{lambda/L}(Re A^H V / L) in ONE iteration and stays there.  Expected value via numpy FFT."""
    N, delta = 8, 2e-3
    k = np.arange(N * N)
    l = (k % N - N // 2) * delta
    m = (k // N - N // 2) * delta
    a = np.arange(N)
    uu, vv = np.meshgrid(a, a, indexing="xy")
    uvw = np.stack([uu.ravel() / (N * delta), vv.ravel() / (N * delta), np.zeros(N * N)], 1)
    g = np.sqrt(np.sqrt(1 - l * l - m * m))
    gains = np.stack([g, g]).astype(np.complex64)
    p = np.zeros(N * N, np.int32)
    q = np.ones(N * N, np.int32)
    o = oracle.Oracle(uvw, l, m, ant_p=p, ant_q=q, gains=gains)
    assert abs(o.max_eig(5) - N * N) < 1e-4            # complex64 gains: n is cancelled to ~1e-7
    rng = np.random.default_rng(8)
    V = rng.standard_normal(N * N) + 1j * rng.standard_normal(N * N)
    lam = 3.0
    R = np.zeros((N, N), dtype=complex)
    R[vv.ravel(), uu.ravel()] = V * ((-1.0) ** (uu.ravel() + vv.ravel()))
    dirty = (np.fft.ifft2(R) * N * N).real.ravel()     # = Re A^H V up to the 1e-7 gain rounding
    want = np.where(dirty / N**2 > lam / N**2, dirty / N**2 - lam / N**2, 0.0)
    for K in (1, 2, 5):
        got = o.fista(V, lam=lam, L=float(N * N), n_iter=K)["x"]
        assert np.max(np.abs(got - want)) < 5e-6
    assert np.count_nonzero(want) > 5 and np.count_nonzero(want == 0) > 5


def test_fista_converges_to_kkt_point_and_matches_nnls():
    """Reading R9: the listing (step 1/L, threshold lambda/L) minimises
    F(I) = 1/2 ||V - A I||^2 + lambda sum I  s.t. I >= 0.
    (i) KKT with g = Re A^H (A I - V): I_k > 0 => g_k = -lambda; I_k = 0 => g_k >= -lambda.
    (ii) the same minimiser from scipy.optimize.nnls on the Cholesky-reduced problem
         (independent library routine).  (iii) Beck-Teboulle bound F(I_k) - F* <= 2 L |I*|^2/(k+1)^2."""
    rng = np.random.default_rng(31)
    o = _tiny(rng, n_vis=80, n_pix=30)
    x_true = np.zeros(o.n_pix)
    x_true[[3, 11, 17, 25]] = [1.0, 0.4, 2.5, 0.7]
    V = o.forward(x_true) + 0.01 * (rng.standard_normal(o.n_vis) + 1j * rng.standard_normal(o.n_vis))
    M = o.dense()
    H = (M.conj().T @ M).real
    L = np.linalg.eigvalsh(H)[-1] * 1.0001
    lam = 0.5
    res = o.fista(V, lam=lam, L=L, n_iter=4000)
    I = res["x"]
    assert np.all(I >= 0)
    grad = o.adjoint(o.forward(I) - V)
    on = I > 0
    assert np.max(np.abs(grad[on] + lam)) < 1e-6 * lam
    assert np.min(grad[~on] + lam) > -1e-6 * lam
    # (ii) NNLS: 1/2 x^T H x - b^T x, b = Re A^H V - lambda  ==  1/2 ||R x - R^-T b||^2 + const
    b = (M.conj().T @ V).real - lam
    Rch = np.linalg.cholesky(H).T
    x_nnls, _ = scipy.optimize.nnls(Rch, np.linalg.solve(Rch.T, b), maxiter=2000)
    assert np.max(np.abs(I - x_nnls)) < 1e-6

    # (iii)
    def F(x):
        return 0.5 * np.sum(np.abs(M @ x - V) ** 2) + lam * np.sum(x)
    Fstar = F(x_nnls)
    for k in (1, 5, 20, 100):
        Ik = o.fista(V, lam=lam, L=L, n_iter=k)["x"]
        assert F(Ik) - Fstar <= 2 * L * np.sum(x_nnls ** 2) / (k + 1) ** 2 + 1e-9
    # info terms (Table 1's separate L2 and L1 columns)
    assert abs(res["l2_term"] - np.sum(np.abs(M @ I - V) ** 2)) < 1e-9
    assert abs(res["l1_term"] - I.sum()) < 1e-12 and res["nnz"] == np.count_nonzero(I)


def test_fista_trace_and_warm_start():
    rng = np.random.default_rng(33)
    o = _tiny(rng, n_vis=40, n_pix=20)
    V = o.forward(rng.uniform(0, 1, o.n_pix))
    L = o.max_eig(100) * 1.05
    a = o.fista(V, lam=0.1, L=L, n_iter=6, want_trace=True)
    # trace[0] is ||A y_1 - V||^2 with y_1 = 0
    assert abs(a["trace"][0, 0] - np.sum(np.abs(V) ** 2)) < 1e-9
    assert abs(a["trace"][-1, 1] - a["x"].sum()) < 1e-12
    # warm start from x0 with K = 0 returns x0; from the converged point stays there
    conv = o.fista(V, lam=0.1, L=L, n_iter=3000)["x"]
    again = o.fista(V, lam=0.1, L=L, n_iter=3, x0=conv)["x"]
    assert np.max(np.abs(again - conv)) < 1e-8


def test_config1_noiseless_recovers_the_sparse_sky():
    """north_star: "recovering a known sparse positive sky on a tiny noiseless problem".
    Config 1 geometry (shrunk to 16x16 pixels so the CPU suite stays fast), noiseless,
    small lambda: support recovered exactly, fluxes to the O(lambda) shrinkage bias."""
    wl = make_workload(1, n_side=16, n_src=6)
    o = oracle.Oracle.from_workload(wl)
    V = o.forward(wl.x_true)
    L = o.max_eig(60) * 1.05
    lam = 1e-3 * np.max(np.abs(o.adjoint(V)))
    I = o.fista(V, lam=lam, L=L, n_iter=3000)["x"]
    assert np.all(I >= 0)
    sup_true = set(np.flatnonzero(wl.x_true))
    big = set(np.flatnonzero(I > 0.02))
    assert big == sup_true
    assert np.max(np.abs(I - wl.x_true)) < 0.02


def _dft_lattice(N=8, delta=2e-3):
    k = np.arange(N * N)
    l = (k % N - N // 2) * delta
    m = (k // N - N // 2) * delta
    a = np.arange(N)
    uu, vv = np.meshgrid(a, a, indexing="xy")
    uvw = np.stack([uu.ravel() / (N * delta), vv.ravel() / (N * delta), np.zeros(N * N)], 1)
    g = np.sqrt(np.sqrt(1 - l * l - m * m))
    gains = np.stack([g, g]).astype(np.complex64)
    return oracle.Oracle(uvw, l, m, ant_p=np.zeros(N * N, np.int32), ant_q=np.ones(N * N, np.int32), gains=gains)


def test_tolerance_stop_rule():
    """Reading R21: stop when the total error E of eq (10) changes by no more
    than `tol` relative, looked at every `check_every` iterations.
    (i)  DFT lattice: FISTA sits on the exact minimiser from I_1 on (closed form, reading R13).
         E_k carries the residual of y_k and y_1 = 0, y_2 = I_1, y_3 = I_2 = I_1: so E_1 != E_2 = E_3
         and the rule must fire at the first looked-at k >= 3, for any tol > 0.
    (ii) the stopping index is the first looked-at k whose |E_k - E_{k-1}| <= tol |E_k|, with E
         formed independently here from the fixed-K run's trace and the dense matrix.
    (iii) stopping only truncates: the result equals the fixed-K run at K = n_iter_done, tol < 0
         never stops, and a smaller tol never stops earlier."""
    o = _dft_lattice()
    rng = np.random.default_rng(8)
    V = rng.standard_normal(64) + 1j * rng.standard_normal(64)
    for every, want in ((1, 3), (2, 4), (3, 3), (4, 4)):
        r = o.fista_tol(V, lam=3.0, L=64.0, max_iter=50, tol=1e-4, check_every=every)
        assert r["n_iter_done"] == want
    # (ii), (iii) on a generic tiny problem
    rng = np.random.default_rng(35)
    o = _tiny(rng, n_vis=80, n_pix=30)
    x_true = np.zeros(o.n_pix)
    x_true[[3, 11, 17, 25]] = [1.0, 0.4, 2.5, 0.7]
    V = o.forward(x_true) + 0.01 * (rng.standard_normal(o.n_vis) + 1j * rng.standard_normal(o.n_vis))
    M = o.dense()
    L = np.linalg.eigvalsh((M.conj().T @ M).real)[-1] * 1.05
    lam, K = 0.5, 400
    full = o.fista(V, lam=lam, L=L, n_iter=K, want_trace=True)
    E = full["trace"][:, 0] + 2.0 * lam * full["trace"][:, 1]
    # trace[:, 0] really is ||M y_k - V||^2: rebuild y_2 from the first two iterates by hand
    I1 = o.fista(V, lam=lam, L=L, n_iter=1)["x"]
    I2 = o.fista(V, lam=lam, L=L, n_iter=2)["x"]
    t2 = (1 + math.sqrt(5)) / 2
    t3 = (1 + math.sqrt(1 + 4 * t2 * t2)) / 2
    y2 = I1                                   # beta_1 = (t_1 - 1)/t_2 = 0
    y3 = I2 + (t2 - 1) / t3 * (I2 - I1)
    assert abs(full["trace"][1, 0] - np.sum(np.abs(M @ y2 - V) ** 2)) < 1e-9
    assert abs(full["trace"][2, 0] - np.sum(np.abs(M @ y3 - V) ** 2)) < 1e-9
    last = 0
    for tol in (1e-2, 1e-4, 1e-6, 1e-8):
        for every in (1, 5):
            ks = [k for k in range(2, K + 1) if k % every == 0 and abs(E[k - 1] - E[k - 2]) <= tol * abs(E[k - 1])]
            want = ks[0] if ks else K
            r = o.fista_tol(V, lam=lam, L=L, max_iter=K, tol=tol, check_every=every)
            assert r["n_iter_done"] == want
            same = o.fista(V, lam=lam, L=L, n_iter=want)
            assert np.array_equal(r["x"], same["x"]) and r["l2_term"] == same["l2_term"]
        assert want >= last
        last = want
    assert 2 < last < K                       # the sweep really exercised early stops
    assert o.fista_tol(V, lam=lam, L=L, max_iter=37, tol=-1.0)["n_iter_done"] == 37


def test_total_error_weight_is_eq10_at_the_independent_minimiser():
    """Reading R21: the E the stopping rule looks at is eq (10) written for the
    listing's lambda, E = ||M y - V||^2 + 2 lambda sum I.  Pin without restating it: at convergence
    y_k = I_k = I*, so E_K must equal TWICE the minimum of F(I) = 1/2 ||V - M I||^2 + lambda sum I
    over I >= 0, and that minimum comes from scipy.optimize.nnls (an independent library solve,
    not from the oracle).  A `lambda` for `2 lambda` slip gives 2 F* - lambda sum I*, off by 10 %."""
    rng = np.random.default_rng(31)
    o = _tiny(rng, n_vis=80, n_pix=30)
    x_true = np.zeros(o.n_pix)
    x_true[[3, 11, 17, 25]] = [1.0, 0.4, 2.5, 0.7]
    V = o.forward(x_true) + 0.01 * (rng.standard_normal(o.n_vis) + 1j * rng.standard_normal(o.n_vis))
    M = o.dense()
    H = (M.conj().T @ M).real
    L = np.linalg.eigvalsh(H)[-1] * 1.0001
    lam = 0.5
    b = (M.conj().T @ V).real - lam
    Rch = np.linalg.cholesky(H).T
    x_nnls, _ = scipy.optimize.nnls(Rch, np.linalg.solve(Rch.T, b), maxiter=2000)
    Fstar = 0.5 * np.sum(np.abs(M @ x_nnls - V) ** 2) + lam * np.sum(x_nnls)
    r = o.fista_tol(V, lam=lam, L=L, max_iter=4000, tol=-1.0)
    assert r["n_iter_done"] == 4000 and r["E"].shape == (4000,)
    assert abs(r["E"][-1] - 2.0 * Fstar) < 1e-9 * Fstar
    assert lam * np.sum(x_nnls) > 0.05 * Fstar          # the L1 part is a visible share of E: the weight matters
    # and E_1 is the residual of y_1 = 0 plus the L1 part of I_1
    I1 = o.fista(V, lam=lam, L=L, n_iter=1)["x"]
    assert abs(r["E"][0] - (np.sum(np.abs(V) ** 2) + 2.0 * lam * I1.sum())) < 1e-9


def test_nnz_change_stop_rule():
    """Reading R24 ("... or when there is a sufficiently small change in the number of
    non-zero entries in I_k"): at the looked-at iterations k >= 2 stop iff |N_k - N_{k-1}| <= nnz_tol N_k.
    (i)  DFT lattice: the iterates are constant from I_1 on, so N_2 = N_1 and the rule fires at the
         first looked-at k >= 2 (the E rule needs k >= 3 there: y_2 != y_1).
    (ii) the stop index equals the one recomputed here from np.count_nonzero of the fixed-K iterates
         (the images themselves, not the oracle's own nnz column).
    (iii) "or": with both rules on, the run stops at the earlier of the two indices; only truncation."""
    o = _dft_lattice()
    rng = np.random.default_rng(8)
    V = rng.standard_normal(64) + 1j * rng.standard_normal(64)
    for every, want in ((1, 2), (2, 2), (3, 3), (5, 5)):
        r = o.fista_tol(V, lam=3.0, L=64.0, max_iter=50, tol=-1.0, nnz_tol=0.0, check_every=every)
        assert r["n_iter_done"] == want
    rng = np.random.default_rng(36)
    o = _tiny(rng, n_vis=60, n_pix=120)                      # more pixels than data: the support keeps moving
    x_true = np.zeros(o.n_pix)
    x_true[rng.choice(o.n_pix, 12, replace=False)] = rng.uniform(0.5, 3.0, 12)
    V = o.forward(x_true) + 0.05 * (rng.standard_normal(o.n_vis) + 1j * rng.standard_normal(o.n_vis))
    L = o.max_eig(200) * 1.05
    lam, K = 0.3, 120
    N = np.array([np.count_nonzero(o.fista(V, lam=lam, L=L, n_iter=k)["x"]) for k in range(1, K + 1)])
    assert len(set(N[:40].tolist())) > 3                     # the support size really changes early on
    seen = set()
    for nnz_tol in (0.2, 0.05, 0.0):
        for every in (1, 4):
            ks = [k for k in range(2, K + 1) if k % every == 0 and abs(int(N[k - 1]) - int(N[k - 2])) <= nnz_tol * N[k - 1]]
            want = ks[0] if ks else K
            r = o.fista_tol(V, lam=lam, L=L, max_iter=K, tol=-1.0, nnz_tol=nnz_tol, check_every=every)
            assert r["n_iter_done"] == want, (nnz_tol, every, r["n_iter_done"], want)
            assert np.array_equal(r["x"], o.fista(V, lam=lam, L=L, n_iter=want)["x"])
            seen.add(want)
    assert len(seen) >= 2 and min(seen) >= 2
    # (iii) either rule
    k_E = o.fista_tol(V, lam=lam, L=L, max_iter=K, tol=1e-5)["n_iter_done"]
    k_N = o.fista_tol(V, lam=lam, L=L, max_iter=K, tol=-1.0, nnz_tol=0.0)["n_iter_done"]
    k_any = o.fista_tol(V, lam=lam, L=L, max_iter=K, tol=1e-5, nnz_tol=0.0)["n_iter_done"]
    assert k_any == min(k_E, k_N) and k_E != k_N
    assert o.fista_tol(V, lam=lam, L=L, max_iter=23, tol=-1.0, nnz_tol=-1.0)["n_iter_done"] == 23


def test_dirty_image_start():
    """Reading R22: the dirty image max(0, s Re A^H V) as I_0.  On the DFT lattice
    Re A^H V / N^2 is numpy's inverse FFT; and FISTA's first iterate from zero is
    T^{lambda/L}(dirty/L), so starting from the dirty image must not change the fixed point."""
    N = 8
    o = _dft_lattice(N)
    rng = np.random.default_rng(9)
    V = rng.standard_normal(N * N) + 1j * rng.standard_normal(N * N)
    a = np.arange(N)
    uu, vv = np.meshgrid(a, a, indexing="xy")
    R = np.zeros((N, N), dtype=complex)
    R[vv.ravel(), uu.ravel()] = V * ((-1.0) ** (uu.ravel() + vv.ravel()))
    want = np.maximum(0.0, np.fft.ifft2(R).real.ravel())
    got = o.dirty_image(V, 1.0 / N**2)
    assert np.max(np.abs(got - want)) < 5e-6 and np.count_nonzero(got) > 5
    rng = np.random.default_rng(36)
    o = _tiny(rng, n_vis=80, n_pix=30)
    V = o.forward(rng.uniform(0, 1, o.n_pix))
    L = o.max_eig(200) * 1.05
    cold = o.fista(V, lam=0.2, L=L, n_iter=3000)["x"]
    warm = o.fista(V, lam=0.2, L=L, n_iter=3000, x0=o.dirty_image(V, 1.0 / o.n_vis))["x"]
    assert np.max(np.abs(cold - warm)) < 1e-7
