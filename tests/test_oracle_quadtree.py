"""Pins for the oracle's quadtree / coarse-to-fine driver (NEXT-3, DESIGN.md
reading R23): a hand-worked step, exact tiling by rasterisation, flux and area conservation, the
coarse-to-fine special case against the regular grid of eqs (5)-(6), and an end-to-end run that
must find a known sparse sky with a small fraction of the full grid's pixels.  CPU only."""
import os

import numpy as np

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _grid(N, delta):
    """eqs (5)-(6), written out here independently of oracle/ and workloads/."""
    k = np.arange(N * N)
    return (k % N - N / 2 + 0.5) * delta, (k // N - N / 2 + 0.5) * delta


def test_hand_worked_refinement_step():
    rows = [[float(t) for t in ln.split()] for ln in open(os.path.join(GOLD, "quadtree_hand_example.txt"))
            if ln.strip() and not ln.startswith("#")]
    want = np.array(rows)
    l = np.array([-0.5, 0.5, -0.5, 0.5])
    m = np.array([-0.5, -0.5, 0.5, 0.5])
    lo, mo, so, xo, po, n_ref = oracle.quadtree_refine(l, m, np.ones(4), np.array([0.0, 8.0, 0.05, 0.0]), 0.01, 0.5)
    assert n_ref == 1
    got = np.stack([lo, mo, so, xo, po.astype(float)], 1)
    assert got.shape == want.shape and np.array_equal(got, want)
    # min_side forbids the split; an all-zero image refines nothing
    assert oracle.quadtree_refine(l, m, np.ones(4), np.array([0.0, 8.0, 0.05, 0.0]), 0.01, 0.6)[5] == 0
    assert oracle.quadtree_refine(l, m, np.ones(4), np.zeros(4), 0.01, 0.1)[5] == 0


def test_leaves_tile_the_field_exactly_and_conserve_flux():
    """Three random refinement rounds from a 4 x 4 grid: rasterise every leaf onto the 32 x 32 lattice of
    finest cells with integer arithmetic; every cell must be covered exactly once."""
    rng = np.random.default_rng(5)
    N0, fine = 4, 32
    l, m = _grid(N0, 1.0)
    side = np.ones(N0 * N0)
    I = rng.uniform(0, 1, N0 * N0)
    flux0 = I.sum()
    for _ in range(3):
        l, m, side, I, parent, n_ref = oracle.quadtree_refine(l, m, side, I, 0.4, 0.0)
        assert n_ref > 0
        I = I * rng.uniform(0.5, 1.5, I.shape[0])
        flux0 = I.sum()
    cover = np.zeros((fine, fine), dtype=int)
    cell = N0 / fine
    for lk, mk, sk in zip(l, m, side):
        n = int(round(sk / cell))
        i0 = int(round((lk - sk / 2 + N0 / 2) / cell))
        j0 = int(round((mk - sk / 2 + N0 / 2) / cell))
        cover[j0:j0 + n, i0:i0 + n] += 1
    assert np.all(cover == 1)
    assert abs((side ** 2).sum() - N0 * N0) < 1e-12
    l2, m2, s2, I2, parent, _ = oracle.quadtree_refine(l, m, side, I, 0.2, 0.0)
    assert abs(I2.sum() - flux0) < 1e-12 * flux0                      # flux-conserving upscaling
    assert np.allclose(np.bincount(parent, weights=I2), I)            # children sum to their parent


def test_refine_all_is_the_coarse_to_fine_grid():
    """frac < 0 refines everything ("double the resolution and upscale"): the centres are
    exactly those of the regular grid with half the spacing."""
    N, d = 6, 0.01
    l, m = _grid(N, d)
    lo, mo, so, xo, _, n_ref = oracle.quadtree_refine(l, m, np.full(N * N, d), np.arange(N * N, dtype=float), -1.0, 0.0)
    assert n_ref == N * N and np.all(so == d / 2)
    lf, mf = _grid(2 * N, d / 2)
    key = lambda a, b: sorted(zip(np.round(a / (d / 4)).astype(int), np.round(b / (d / 4)).astype(int)))
    assert key(lo, mo) == key(lf, mf)


def test_quadtree_driver_finds_a_sparse_sky_with_few_pixels():
    """End to end on a noiseless toy: 6 point sources on a 64 x 64 fine grid, 16 antennas in a 1 km disk
    (config-1 style), start at 8 x 8 with Gaussian pixels of sigma = side above the resolution limit.  The driver must (i) end with every source inside a finest-level leaf
    that carries most of its flux, (ii) use far fewer leaves than the 4,096-pixel grid, (iii) fit the data."""
    rng = np.random.default_rng(77)
    Nf, field = 64, 0.05
    df = field / Nf
    ant = rng.uniform(-1, 1, (200, 2))
    ant = ant[(ant ** 2).sum(1) <= 1][:16] * 500.0 / 1.99862
    p, q = np.triu_indices(16, 1)
    base = ant[p] - ant[q]
    rot = [np.array([[np.cos(t), -np.sin(t)], [np.sin(t), np.cos(t)]]) for t in np.linspace(0, np.pi, 6, endpoint=False)]
    uv = np.concatenate([base @ R.T for R in rot])
    uvw = np.concatenate([uv, np.zeros((uv.shape[0], 1))], 1)
    lf, mf = _grid(Nf, df)
    src = rng.choice(np.flatnonzero((np.abs(lf) < 0.4 * field) & (np.abs(mf) < 0.4 * field)), 6, replace=False)
    flux = rng.uniform(1.0, 3.0, 6)
    x_true = np.zeros(Nf * Nf)
    x_true[src] = flux
    V = oracle.Oracle(uvw, lf, mf).forward(x_true)
    l0, m0 = _grid(8, field / 8)
    lam = 0.02 * np.abs(oracle.Oracle(uvw, l0, m0).adjoint(V)).max()
    res = oracle.quadtree_solve(uvw, V, l0, m0, np.full(64, field / 8), n_levels=4, frac=0.01, min_side=df * 0.999,
                                lam=lam, n_pow=30, L_safety=1.05, max_iter=400, tol=1e-7, check_every=10,
                                sigma_factor=1.0)
    assert len(res["levels"]) == 4 and res["l"].shape[0] < 0.25 * Nf * Nf
    assert [lv["n_pix"] for lv in res["levels"]] == sorted(lv["n_pix"] for lv in res["levels"])
    finest = np.isclose(res["side"], df)
    for s, f in zip(src, flux):
        hit = np.flatnonzero(finest & np.isclose(res["l"], lf[s]) & np.isclose(res["m"], mf[s]))
        assert hit.size == 1, "source pixel not refined to the finest level"
        assert abs(res["x"][hit[0]] - f) < 0.05 * f                  # O(lambda) shrinkage bias only
    assert res["levels"][-1]["l2_term"] < 1e-3 * np.sum(np.abs(V) ** 2)
    # delta pixels everywhere (sigma_factor = 0) cannot describe emission inside a coarse square: the fit is poor
    bad = oracle.quadtree_solve(uvw, V, l0, m0, np.full(64, field / 8), n_levels=4, frac=0.01, min_side=df * 0.999,
                                lam=lam, n_pow=30, L_safety=1.05, max_iter=400, tol=1e-7, check_every=10)
    assert bad["levels"][-1]["l2_term"] > 0.2 * np.sum(np.abs(V) ** 2)
