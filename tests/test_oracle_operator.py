"""Pins for the oracle's applies O2 (forward) and O3 (adjoint): an independent library routine
(numpy FFT on the DFT lattice), the adjoint identity, and dense brute force.  CPU only."""
import numpy as np
import pytest

import oracle
from workloads import make_workload


def _lattice(N, delta):
    """N x N pixel grid (eqs 5-6) and the full DFT lattice of visibilities
    u, v in {0..N-1}/(N delta), w = 0."""
    k = np.arange(N * N)
    l = (k % N - N // 2) * delta
    m = (k // N - N // 2) * delta
    a = np.arange(N)
    uu, vv = np.meshgrid(a, a, indexing="xy")          # u fastest
    uvw = np.stack([uu.ravel() / (N * delta), vv.ravel() / (N * delta), np.zeros(N * N)], axis=1)
    return l, m, uvw, uu.ravel(), vv.ravel()


def test_forward_equals_numpy_fft_on_the_dft_lattice():
    """eq (2)/(9) with w = 0 on a regular grid IS a 2-D DFT: compare the
    oracle's forward with numpy.fft.fft2 (independent library routine)."""
    N, delta = 16, 1e-3
    l, m, uvw, a, b = _lattice(N, delta)
    rng = np.random.default_rng(3)
    x = rng.uniform(0, 1, N * N)
    n = np.sqrt(1 - l * l - m * m)
    o = oracle.Oracle(uvw, l, m)
    got = o.forward(x)
    # v[a,b] = sum_{i,j} (x/n)[j,i] exp(-2 pi i (a (i-N/2) + b (j-N/2))/N) = (-1)^(a+b) FFT2(x/n)[b,a]
    F = np.fft.fft2((x / n).reshape(N, N))             # axes: [m index, l index]
    want = ((-1.0) ** (a + b)) * F[b, a]
    assert np.max(np.abs(got - want)) < 1e-11


def test_adjoint_equals_numpy_ifft_on_the_dft_lattice():
    N, delta = 16, 1e-3
    l, m, uvw, a, b = _lattice(N, delta)
    rng = np.random.default_rng(4)
    r = rng.standard_normal(N * N) + 1j * rng.standard_normal(N * N)
    n = np.sqrt(1 - l * l - m * m)
    o = oracle.Oracle(uvw, l, m)
    got = o.adjoint(r)
    # g[j,i] = Re (1/n) sum_{a,b} exp(+2 pi i (a(i-N/2)+b(j-N/2))/N) r[a,b]
    R = np.zeros((N, N), dtype=complex)
    R[b, a] = r * ((-1.0) ** (a + b))
    want = (np.fft.ifft2(R) * N * N).real.ravel() / n
    assert np.max(np.abs(got - want)) < 1e-10


def _random_problem(rng, n_vis=37, n_pix=53, gauss=False, gains=False, model=1, wmax=800.0):
    n_ant = 6
    uvw = rng.uniform(-1, 1, size=(n_vis, 3)) * np.array([900.0, 900.0, wmax])
    l = rng.uniform(-0.12, 0.12, n_pix)
    m = rng.uniform(-0.12, 0.12, n_pix)
    sigma = None
    if gauss:
        sigma = rng.uniform(0.0005, 0.004, n_pix)
        sigma[::5] = 0.0                              # mixed delta/Gaussian list (reading R15)
    kw = {}
    if gains:
        p = rng.integers(0, n_ant, n_vis)
        q = rng.integers(0, n_ant, n_vis)
        g = (rng.standard_normal((n_ant, n_pix)) + 1j * rng.standard_normal((n_ant, n_pix))).astype(np.complex64)
        kw = dict(ant_p=p, ant_q=q, gains=g)
    return oracle.Oracle(uvw, l, m, sigma, gauss_model=model, **kw)


@pytest.mark.parametrize("gauss,gains,model", [(False, False, 1), (True, False, 1), (True, False, 0),
                                               (False, True, 1), (True, True, 1)])
def test_adjoint_identity_1e12(gauss, gains, model):
    """north_star / reading R3: Re <A x, y> = <x, A^H y> for real x, complex y, to 1e-12."""
    rng = np.random.default_rng(11)
    o = _random_problem(rng, gauss=gauss, gains=gains, model=model)
    for _ in range(3):
        x = rng.standard_normal(o.n_pix)
        y = rng.standard_normal(o.n_vis) + 1j * rng.standard_normal(o.n_vis)
        lhs = np.real(np.vdot(o.forward(x), y))        # Re sum conj(Ax) y
        rhs = float(np.dot(x, o.adjoint(y)))
        assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), abs(rhs), 1.0)


@pytest.mark.parametrize("gauss,gains", [(False, False), (True, True)])
def test_applies_equal_dense_brute_force(gauss, gains):
    """O2/O3 loops (indices, conj, Re) against numpy matmul on the dense matrix of entries."""
    rng = np.random.default_rng(12)
    o = _random_problem(rng, n_vis=23, n_pix=31, gauss=gauss, gains=gains)
    M = o.dense()
    x = rng.uniform(0, 1, o.n_pix)
    x[::3] = 0.0
    r = rng.standard_normal(o.n_vis) + 1j * rng.standard_normal(o.n_vis)
    assert np.max(np.abs(o.forward(x) - M @ x)) < 1e-12
    assert np.max(np.abs(o.adjoint(r) - (M.conj().T @ r).real)) < 1e-12
    rows = np.array([5, 0, 22, 7])
    cols = np.array([30, 2, 2, 11])
    assert np.array_equal(o.forward(x, rows=rows), o.forward(x)[rows])
    assert np.array_equal(o.adjoint(r, cols=cols), o.adjoint(r)[cols])


def test_workload_shapes_match_baseline_configs():
    """BASELINE.json configs: sizes of the full workloads (no operator arithmetic involved)."""
    w1 = make_workload(1)
    assert (w1.n_pix, w1.n_vis, w1.n_ant) == (1024, 1000, 16) and np.all(w1.uvw[:, 2] == 0)
    assert abs(w1.l.min() + 0.05) < 1e-15 and np.count_nonzero(w1.x_true) == 10
    w2 = make_workload(2)
    assert (w2.n_pix, w2.n_vis) == (65536, 20160)
    w3 = make_workload(3)
    assert (w3.n_pix, w3.n_vis) == (86016, 20160) and w3.sigma is not None
    assert sorted(set(np.round(w3.sigma / w3.delta, 6))) == [0.5, 1.0, 2.0]
    w4 = make_workload(4, n_side=64, n_src=100)            # the full gain table is 256 MiB; shape logic only
    assert w4.gains.shape == (128, 4096) and w4.n_vis == 65024 and w4.sigma_n == 0.0
    w5 = make_workload(5, n_side=32, n_src=50)
    assert w5.n_vis == 406400 and np.abs(w5.uvw).max() <= 3000.0 / 1.99862 + 1
    # determinism
    assert np.array_equal(make_workload(2).uvw, w2.uvw)
