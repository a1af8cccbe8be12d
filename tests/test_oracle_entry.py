"""Pins for the oracle's matrix entry O1 (eqs 9, 16, 17) against what the paper and the
mathematics fix -- hand values, limits, and brute-force quadrature.  CPU only."""
import math
import os

import numpy as np
import pytest

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    out = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                out.append([float(t) for t in line.split()])
    return out


def _one(u, v, w, l, m, sigma=None, gp=None, gq=None, model=1):
    """Entry M_00 of a 1-visibility, 1-pixel problem."""
    kw = {}
    if gp is not None:
        kw = dict(ant_p=[0], ant_q=[1], gains=np.array([[gp], [gq]], dtype=np.complex64))
    o = oracle.Oracle([[u, v, w]], [l], [m], None if sigma is None else [sigma],
                      gauss_model=model, **kw)
    return o.entry(0, 0)


# --------------------------------------------------------------------------- eq (9)
def test_eq9_hand_values():
    """PAPER.md:117-120 eq (9): sign of the phase, u<->l / v<->m pairing, w(n-1), 1/n, gains."""
    for u, v, w, l, m, gpr, gpi, gqr, gqi, mre, mim in _rows("entry_hand_values.txt"):
        got = _one(u, v, w, l, m, gp=complex(gpr, gpi), gq=complex(gqr, gqi))
        assert abs(got - complex(mre, mim)) < 1e-12, (u, v, w, l, m, got)


def test_phase_centre_source_gives_constant_visibilities():
    """north_star: a unit point source at the phase centre gives V_j = 1 for every baseline."""
    rng = np.random.default_rng(0)
    uvw = rng.uniform(-2000, 2000, size=(50, 3))
    o = oracle.Oracle(uvw, [0.0, 0.01], [0.0, -0.02])
    v = o.forward([1.0, 0.0])
    assert np.max(np.abs(v - 1.0)) < 1e-14


def test_offset_source_closed_form_via_small_angle_series():
    """Offset source: |V| = 1/n0 and the phase equals the series -2 pi (u l + v m - w (r^2/2 + r^4/8
    + r^6/16 + 5 r^8/128)) -- the binomial series of n - 1, not a call to sqrt."""
    l0, m0 = 0.011, -0.007
    r2 = l0 * l0 + m0 * m0
    nm1 = -(r2 / 2 + r2 ** 2 / 8 + r2 ** 3 / 16 + 5 * r2 ** 4 / 128)
    inv_n = 1 + r2 / 2 + 3 * r2 ** 2 / 8 + 5 * r2 ** 3 / 16   # binomial series of (1-r2)^(-1/2)
    rng = np.random.default_rng(1)
    uvw = rng.uniform(-1500, 1500, size=(40, 3))
    o = oracle.Oracle(uvw, [l0], [m0])
    v = o.forward([2.5])
    ph = -2 * math.pi * (uvw[:, 0] * l0 + uvw[:, 1] * m0 + uvw[:, 2] * nm1)
    want = 2.5 * inv_n * np.exp(1j * ph)
    assert np.max(np.abs(v - want)) < 1e-9


# --------------------------------------------------------------------------- eq (16): quadrature
def _quad_eq15(u, v, w, l0, m0, s, npts=1601, half_widths=6.0):
    """Brute-force 2-D trapezoid of eq (15)'s integrand INCLUDING its 1/sigma^2:
    (1/s^2) exp(-pi((l-l0)^2+(m-m0)^2)/s^2) exp(i pi w (l^2+m^2)) exp(-2 pi i (u l + v m)).
    The Gaussian's standard deviation is s/sqrt(2 pi); the box is +-half_widths*s."""
    a = half_widths * s
    x = np.linspace(-a, a, npts)
    h = x[1] - x[0]
    wt = np.full(npts, h)
    wt[0] = wt[-1] = h / 2
    L = l0 + x[None, :]
    Mm = m0 + x[:, None]
    f = (1.0 / s ** 2) * np.exp(-math.pi * ((L - l0) ** 2 + (Mm - m0) ** 2) / s ** 2) \
        * np.exp(1j * math.pi * w * (L ** 2 + Mm ** 2)) * np.exp(-2j * math.pi * (u * L + v * Mm))
    return (wt[:, None] * wt[None, :] * f).sum()


@pytest.mark.parametrize("u,v,w,l0,m0,s", [
    (120.0, -80.0, 300.0, 0.010, 0.020, 0.002),
    (40.0, 25.0, 1000.0, -0.015, 0.005, 0.003),
    (300.0, 100.0, 0.0, 0.020, -0.010, 0.001),
    (-75.0, 60.0, -500.0, 0.000, 0.000, 0.004),
    (10.0, 5.0, 20000.0, 0.004, 0.003, 0.006),       # q = w s^2 = 0.72: strongly "defocused"
])
def test_eq16_is_the_analytic_integral_of_eq15(u, v, w, l0, m0, s):
    """PAPER.md:160 "This integral may be performed analytically": quadrature of eq (15) must
    equal the paraxial entry (times n, which eq (15) holds fixed at the pixel centre).  Pins
    readings R5 (no leftover 1/sigma^2) and R7 (the first exponential) and every sign in eq (16)."""
    n0 = math.sqrt(1 - l0 * l0 - m0 * m0)
    got = _one(u, v, w, l0, m0, sigma=s, model=0) * n0
    want = _quad_eq15(u, v, w, l0, m0, s)
    assert abs(got - want) < 1e-9, (got, want)


def test_gaussian_pixel_unit_integral_and_w0_limit():
    """PAPER.md:137 (unit integral) and :165 (w -> 0 gives the Fourier transform of a Gaussian):
    M(w=0) = exp(-2 pi i (u l + v m)) exp(-pi s^2 (u^2+v^2)) / n;  value 1/n at u = v = 0."""
    l0, m0, s = 0.02, -0.01, 0.003
    n0 = math.sqrt(1 - l0 * l0 - m0 * m0)
    for model in (0, 1):
        assert abs(_one(0, 0, 0, l0, m0, sigma=s, model=model) - 1 / n0) < 1e-14
    u, v = 90.0, -140.0
    want = np.exp(-2j * math.pi * (u * l0 + v * m0)) * math.exp(-math.pi * s * s * (u * u + v * v)) / n0
    assert abs(_one(u, v, 0.0, l0, m0, sigma=s, model=0) - want) < 1e-13


def test_sigma_to_zero_limits():
    """sigma -> 0 of eq (16) is the paraxial form of eq (4); of eq (17) it is
    eq (9) exactly (pins reading R6: the residual phase is n - 1 + r^2/2)."""
    u, v, w, l0, m0 = 210.0, -130.0, 800.0, 0.03, 0.02
    n0 = math.sqrt(1 - l0 * l0 - m0 * m0)
    delta = _one(u, v, w, l0, m0)
    wide = _one(u, v, w, l0, m0, sigma=1e-9, model=1)
    assert abs(wide - delta) < 1e-11
    parax = _one(u, v, w, l0, m0, sigma=1e-9, model=0)
    want = np.exp(-2j * math.pi * (u * l0 + v * m0)) * np.exp(1j * math.pi * w * (l0 * l0 + m0 * m0)) / n0
    assert abs(parax - want) < 1e-11
    # and sigma == 0 exactly always means eq (9), whatever the model (reading R15)
    assert _one(u, v, w, l0, m0, sigma=0.0, model=0) == delta
    assert _one(u, v, w, l0, m0, sigma=0.0, model=1) == delta


def test_eq13_residual_phase_matches_papers_expansion():
    """PAPER.md:142-147 eq (13): M17/M16 = exp(-2 pi i w (n-1+r^2/2)) ~= 1 + i pi w r^4/4.
    With the sign as PRINTED inside eqs (12)/(17) the ratio would be about -0.31+0.95i."""
    for l0, m0, w, rre, rim in _rows("eq13_residual_phase.txt"):
        ratio = _one(50.0, 60.0, w, l0, m0, sigma=0.001, model=1) / _one(50.0, 60.0, w, l0, m0, sigma=0.001, model=0)
        assert abs(ratio - complex(rre, rim)) < 5e-6      # O(eps^6) terms + the rhs's own truncation
        assert abs(abs(ratio) - 1.0) < 1e-14


# --------------------------------------------------------------------------- eq (17) vs exact eq (4)
def _quad_eq4_gaussian(u, v, w, l0, m0, s, npts=1601, half_widths=6.0):
    """Brute-force quadrature of the EXACT integrand of eq (4) for one unit-flux Gaussian pixel
    eq (11), unit gains:  f_k(l,m)/n(l,m) * exp(-2 pi i (u l + v m + w (n(l,m) - 1)))."""
    a = half_widths * s
    x = np.linspace(-a, a, npts)
    h = x[1] - x[0]
    wt = np.full(npts, h)
    wt[0] = wt[-1] = h / 2
    L = l0 + x[None, :]
    Mm = m0 + x[:, None]
    n = np.sqrt(1 - L ** 2 - Mm ** 2)
    f = (1.0 / s ** 2) * np.exp(-math.pi * ((L - l0) ** 2 + (Mm - m0) ** 2) / s ** 2) / n \
        * np.exp(-2j * math.pi * (u * L + v * Mm + w * (n - 1)))
    return (wt[:, None] * wt[None, :] * f).sum()


@pytest.mark.parametrize("u,v,w,l0,m0,s,tol", [
    (120.0, -80.0, 300.0, 0.010, 0.020, 0.002, 1e-5),
    (200.0, 150.0, 1000.0, 0.10, 0.12, 0.001, 2e-3),     # wide angle, large w
    (30.0, 10.0, 100.0, 0.20, -0.15, 0.002, 2e-3),
])
def test_eq17_approximates_the_exact_integral(u, v, w, l0, m0, s, tol):
    """eq (17) "will be suitable for any field of view" as long as the pixel is
    small; the oracle implements the approximation, this quantifies it (reading R18)."""
    got = _one(u, v, w, l0, m0, sigma=s, model=1)
    want = _quad_eq4_gaussian(u, v, w, l0, m0, s)
    assert abs(got - want) < tol, (got, want)


def test_eq16_fails_at_wide_angle_where_eq17_holds():
    """eq (13) "limits the field of view"; at l=.10, m=.12, w=1000 the paraxial
    form is far off while the wide-field form is not."""
    u, v, w, l0, m0, s = 200.0, 150.0, 1000.0, 0.10, 0.12, 0.001
    exact = _quad_eq4_gaussian(u, v, w, l0, m0, s)
    assert abs(_one(u, v, w, l0, m0, sigma=s, model=0) - exact) > 0.1
    assert abs(_one(u, v, w, l0, m0, sigma=s, model=1) - exact) < 2e-3


# --------------------------------------------------------------------------- real-arithmetic form
def test_real_form_identity_used_by_the_cuda_kernels():
    """with q = w s^2, den = 1+q^2,
    A = -pi s^2 ((u-wl)^2+(v-wm)^2)/den,   M = (1/(n den)) (1+iq) exp(A) exp(-i(X - q A)),
    X = 2 pi (u l + v m + w n'), n' = n-1 (eq 17) or -r^2/2 (eq 16).  The oracle uses the literal
    complex-denominator form; this test pins the derivation the GPU relies on."""
    rng = np.random.default_rng(5)
    for _ in range(200):
        u, v = rng.uniform(-1500, 1500, 2)
        w = rng.uniform(-1500, 1500)
        l0, m0 = rng.uniform(-0.2, 0.2, 2)
        s = 10 ** rng.uniform(-5, -1.7)
        n0 = math.sqrt(1 - l0 * l0 - m0 * m0)
        r2 = l0 * l0 + m0 * m0
        q = w * s * s
        den = 1 + q * q
        A = -math.pi * s * s * ((u - w * l0) ** 2 + (v - w * m0) ** 2) / den
        for model, npr in ((1, n0 - 1), (0, -r2 / 2)):
            X = 2 * math.pi * (u * l0 + v * m0 + w * npr)
            want = (1 + 1j * q) / (n0 * den) * math.exp(A) * np.exp(-1j * (X - q * A))
            got = _one(u, v, w, l0, m0, sigma=s, model=model)
            assert abs(got - want) <= 1e-9 * max(abs(want), 1e-30) + 1e-15, (got, want, q)


def test_gains_factorisation_cases():
    """Reading R4: constant-per-antenna gains scale V_j by c_p conj(c_q);
    one real beam shared by all antennas is the unit-gain apply of b^2 x."""
    rng = np.random.default_rng(7)
    n_ant, n_pix = 5, 30
    p, q = np.triu_indices(n_ant, 1)
    uvw = rng.uniform(-300, 300, size=(len(p), 3))
    l = rng.uniform(-0.05, 0.05, n_pix)
    m = rng.uniform(-0.05, 0.05, n_pix)
    x = rng.uniform(0, 1, n_pix)
    unit = oracle.Oracle(uvw, l, m)
    c = (rng.standard_normal(n_ant) + 1j * rng.standard_normal(n_ant)).astype(np.complex64)
    g = np.repeat(c[:, None], n_pix, axis=1)
    o = oracle.Oracle(uvw, l, m, ant_p=p, ant_q=q, gains=g)
    want = unit.forward(x) * (c[p].astype(np.complex128) * np.conj(c[q].astype(np.complex128)))
    assert np.max(np.abs(o.forward(x) - want)) < 1e-12
    b = rng.uniform(0.5, 1.0, n_pix).astype(np.float32)
    o2 = oracle.Oracle(uvw, l, m, ant_p=p, ant_q=q, gains=np.repeat(b[None, :], n_ant, 0).astype(np.complex64))
    want2 = unit.forward(b.astype(np.float64) ** 2 * x)
    assert np.max(np.abs(o2.forward(x) - want2)) < 1e-12


def test_polar_identities_used_by_the_cuda_kernels():
    """DESIGN.md section 6, pinned against the oracle's literal complex arithmetic (delta and Gaussian entries, both models):
    (i)  polar gains: with G = g_p conj(g_q) = |G| e^{i gamma}, the entry with gains is |G| times the unit-gain entry
         evaluated with its phase shifted by -gamma, i.e. M_gain = |G| e^{i gamma} M_unit (a real weight and a phase shift);
    (ii) one-cosine adjoint: Re(conj(M) r) = |M| |r| cos(arg r - arg M); for a delta pixel arg M = gamma - X, so the term
         is (|G|/n) |r| cos(X - gamma + arg r);
    (iii) Gaussian: A cos X' + B sin X' = R cos(X' - psi) with A = r_re + q r_im, B = q r_re - r_im, (R, psi) = polar(A, B)."""
    rng = np.random.default_rng(17)
    n_ant, n_pix = 4, 6
    p, q = np.triu_indices(n_ant, 1)
    uvw = rng.uniform(-800, 800, size=(len(p), 3))
    l = rng.uniform(-0.1, 0.1, n_pix)
    m = rng.uniform(-0.1, 0.1, n_pix)
    sig = np.where(rng.uniform(size=n_pix) < 0.5, 0.0, 10 ** rng.uniform(-4, -2, n_pix))
    g = (rng.standard_normal((n_ant, n_pix)) + 1j * rng.standard_normal((n_ant, n_pix))).astype(np.complex64)
    g[0, 0] = 0.0                       # a zero gain: amplitude 0, phase 0
    g[1, 1] = -2.0                      # phase pi
    g[2, 2] = 3.0j                      # phase pi/2
    for model in (0, 1):
        unit = oracle.Oracle(uvw, l, m, sigma=sig, gauss_model=model)
        og = oracle.Oracle(uvw, l, m, sigma=sig, ant_p=p, ant_q=q, gains=g, gauss_model=model)
        g64 = g.astype(np.complex128)
        amp, ph = np.abs(g64), np.angle(g64)
        for j in range(len(p)):
            r = complex(rng.standard_normal(), rng.standard_normal())
            for k in range(n_pix):
                Mu, Mg = unit.entry(j, k), og.entry(j, k)
                G_amp = amp[p[j], k] * amp[q[j], k]
                gamma = ph[p[j], k] - ph[q[j], k]
                assert abs(Mg - G_amp * np.exp(1j * gamma) * Mu) <= 1e-13 * max(abs(Mu) * max(G_amp, 1), 1e-30)      # (i)
                want = (np.conj(Mg) * r).real
                got = abs(Mg) * abs(r) * math.cos(np.angle(r) - np.angle(Mg)) if abs(Mg) > 0 else 0.0
                assert abs(got - want) <= 1e-12 * max(abs(Mg) * abs(r), 1e-30)                                         # (ii)
                if sig[k] == 0.0:      # delta pixel: the phase the kernel forms explicitly
                    n0 = math.sqrt(1 - l[k] ** 2 - m[k] ** 2)
                    X = 2 * math.pi * (uvw[j, 0] * l[k] + uvw[j, 1] * m[k] + uvw[j, 2] * (n0 - 1))
                    got2 = G_amp / n0 * abs(r) * math.cos(X - gamma + np.angle(r))
                    assert abs(got2 - want) <= 1e-9 * max(abs(Mg) * abs(r), 1e-30)
    for _ in range(200):                                                                                              # (iii)
        qq, Xp = rng.uniform(-3, 3), rng.uniform(-50, 50)
        r = complex(rng.standard_normal(), rng.standard_normal())
        A, B = r.real + qq * r.imag, qq * r.real - r.imag
        R, psi = math.hypot(A, B), math.atan2(B, A)
        lhs = A * math.cos(Xp) + B * math.sin(Xp)
        assert abs(lhs - R * math.cos(Xp - psi)) <= 1e-12 * max(R, 1e-30)
        # and A cos X' + B sin X' is Re((1 + iq) conj(c - i s) ... ) of the kernels' entry form: Re conj((1+iq)(c - is)) r
        c, s = math.cos(Xp), math.sin(Xp)
        assert abs(lhs - (np.conj((1 + 1j * qq) * (c - 1j * s)) * r).real) <= 1e-12 * max(R, 1e-30)
