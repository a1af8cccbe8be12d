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


def test_quadtree_with_inherited_gains():
    """Reading R25: under refinement a child inherits the gain column of its parent.
    (i) gains constant over the sky, g_a(k) = c_a: then G_j = c_p conj(c_q) factors out of row j, so the driver on
        (V, gains) must walk exactly the tree, and return exactly the fluxes, of the unit-gain driver on the rows
        rescaled to unit gain -- here |c_a| = 1, so M_gain = D M with D unitary-diagonal and Re M^H D^H D M = Re M^H M:
        same L, same iterates, same splits, with V' = conj(G) V.
    (ii) a direction-dependent table: after one refine-all step the level-2 problem is the oracle's own operator
        on the children with gains[:, parent] -- checked against an explicitly built child table."""
    rng = np.random.default_rng(91)
    n_ant = 7
    ant = rng.uniform(-150, 150, (n_ant, 2))
    p, q = np.triu_indices(n_ant, 1)
    uv = np.concatenate([(ant[p] - ant[q]) @ np.array([[np.cos(t), -np.sin(t)], [np.sin(t), np.cos(t)]]).T
                         for t in (0.0, 0.7, 1.9)])
    uvw = np.concatenate([uv, rng.uniform(-5, 5, (uv.shape[0], 1))], 1)
    ap, aq = np.tile(p, 3).astype(np.int32), np.tile(q, 3).astype(np.int32)
    N, field = 4, 0.04
    l0, m0 = _grid(N, field / N)
    side0 = np.full(N * N, field / N)
    lf, mf = _grid(4 * N, field / (4 * N))
    x_true = np.zeros(16 * N * N)
    x_true[rng.choice(16 * N * N, 5, replace=False)] = rng.uniform(1, 3, 5)
    c = np.exp(1j * rng.uniform(-np.pi, np.pi, n_ant))
    G = c[ap] * np.conj(c[aq])
    V_unit = oracle.Oracle(uvw, lf, mf).forward(x_true)
    V = G * V_unit
    kw = dict(n_levels=3, frac=0.05, min_side=field / (4 * N) * 0.999, lam=0.05, n_pow=40, L_safety=1.05, max_iter=150,
              tol=1e-9, check_every=5, sigma_factor=1.0)
    a = oracle.quadtree_solve(uvw, V, l0, m0, side0, ant_p=ap, ant_q=aq, gains0=np.repeat(c[:, None], N * N, 1), **kw)
    b = oracle.quadtree_solve(uvw, V_unit, l0, m0, side0, **kw)
    assert [lv["n_pix"] for lv in a["levels"]] == [lv["n_pix"] for lv in b["levels"]] and len(a["levels"]) == 3
    assert np.array_equal(a["l"], b["l"]) and np.array_equal(a["side"], b["side"])
    assert np.max(np.abs(a["x"] - b["x"])) < 1e-6 * np.max(b["x"])
    # (ii)
    g0 = (1.0 + 0.3 * (rng.standard_normal((n_ant, N * N)) + 1j * rng.standard_normal((n_ant, N * N)))).astype(np.complex64)
    r = oracle.quadtree_solve(uvw, V, l0, m0, side0, n_levels=2, frac=-1.0, min_side=0.0, lam=0.05, n_pow=20,
                              L_safety=1.05, max_iter=40, tol=-1.0, ant_p=ap, ant_q=aq, gains0=g0)
    l1, m1, s1, x1, parent, _ = oracle.quadtree_refine(l0, m0, side0, oracle.Oracle(
        uvw, l0, m0, None, ap, aq, g0).fista_tol(V, 0.05, oracle.Oracle(uvw, l0, m0, None, ap, aq, g0).max_eig(20) * 1.05,
                                                 40, -1.0)["x"], -1.0, 0.0)
    child = oracle.Oracle(uvw, l1, m1, None, ap, aq, np.stack([g0[a_][parent] for a_ in range(n_ant)]))
    want = child.fista_tol(V, 0.05, child.max_eig(20) * 1.05, 40, -1.0, x0=x1)["x"]
    assert np.array_equal(r["l"], l1) and np.max(np.abs(r["x"] - want)) < 1e-9 * max(np.max(want), 1e-30)
