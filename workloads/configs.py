"""The five BASELINE.json configurations as seeded synthetic inputs.

Recipe (stated in DESIGN.md §"Input recipe"; items marked [reading] are this repo's reading of
an under-specified config and are fixed):

* RNG: ``numpy.random.default_rng(1310207800 + config_id)``; draw order: antennas, pixel
  jitter, source pixels, fluxes, blob parameters, gain coefficients, noise.
* 150 MHz, uvw in wavelengths (section 2).
* Antennas uniform in a disk whose stated size is its DIAMETER [reading].
* Configs 2-5: textbook Earth-rotation synthesis, latitude -26.7 deg, declination -30 deg,
  hour angles ``linspace(-H, +H, n_steps)`` inclusive [reading]; time-major record order, then
  (p, q) lexicographic with p < q.
* Config 1: coplanar snapshot baselines rotated by ``pi*s/9``, s = 0..8, first 1,000 kept, w = 0.
* Pixel grids follow eqs (5)-(6): ``l_k = (k mod N - N/2) D``,
  ``m_k = (floor(k/N) - N/2) D`` with ``D = 2 sin(FOV/2)/N`` [reading] (config 1: 0.1/32).
* Fluxes ``clip(0.1 (1 + Lomax(1.5)), 0.1, 10)`` Jy, i.e. Pareto(alpha=1.5) with minimum 0.1.
* Sources sit on distinct pixels of the (finest) grid drawn from its inner 80 % [reading].

These inputs STAND IN for the paper's simulated ASKAP observations and the CASA-tutorial VLA
datasets, none of which is available here.

No operator arithmetic lives here: measured data ``V = A x_true + noise`` is assembled by the
caller (tests use the oracle's A, bench.py uses the CUDA A).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

C_LIGHT = 299792458.0
FREQ_HZ = 150e6
WAVELENGTH = C_LIGHT / FREQ_HZ
LATITUDE = math.radians(-26.7)
DECLINATION = math.radians(-30.0)

CONFIG_IDS = (1, 2, 3, 4, 5)

GAUSS_PARAXIAL = 0  # eq (16)
GAUSS_WIDEFIELD = 1  # eq (17)


@dataclasses.dataclass
class Workload:
    cid: int
    name: str
    uvw: np.ndarray            # [n_vis, 3] float64, wavelengths
    ant_p: np.ndarray          # [n_vis] int32
    ant_q: np.ndarray          # [n_vis] int32
    n_ant: int
    l: np.ndarray              # [n_pix] float64 direction cosines
    m: np.ndarray              # [n_pix] float64
    sigma: Optional[np.ndarray]   # [n_pix] float64 (paper's sigma_k, eq 11) or None = delta pixels
    gains: Optional[np.ndarray]   # [n_ant, n_pix] complex64 or None = unit gains
    gauss_model: int
    x_true: np.ndarray         # [n_pix] float64, sparse positive sky on the pixel list
    truth_extra: Optional[dict]   # config 3: blobs as a separate truth pixel list {l, m, sigma, flux}
    noise: np.ndarray          # [n_vis] complex128, already scaled by sigma_n
    sigma_n: float
    n_iter: int                # solver iteration count used by parity tests / bench
    delta: float               # fine grid spacing
    meta: dict

    @property
    def n_vis(self) -> int:
        return int(self.uvw.shape[0])

    @property
    def n_pix(self) -> int:
        return int(self.l.shape[0])


# ----------------------------------------------------------------------------- geometry
def _antennas(rng: np.random.Generator, n_ant: int, diameter_m: float) -> np.ndarray:
    u1 = rng.random(n_ant)
    u2 = rng.random(n_ant)
    r = 0.5 * diameter_m * np.sqrt(u1)
    th = 2.0 * np.pi * u2
    return np.stack([r * np.cos(th), r * np.sin(th), np.zeros(n_ant)], axis=1)  # E, N, Up


def _pairs(n_ant: int):
    p, q = np.triu_indices(n_ant, k=1)
    return p.astype(np.int32), q.astype(np.int32)


def _uvw_synthesis(enu: np.ndarray, h_max_hours: float, n_steps: int):
    """Earth-rotation synthesis, time-major then (p,q) lexicographic."""
    sl, cl = math.sin(LATITUDE), math.cos(LATITUDE)
    e, n, up = enu[:, 0], enu[:, 1], enu[:, 2]
    xyz = np.stack([-sl * n + cl * up, e, cl * n + sl * up], axis=1)
    p, q = _pairs(enu.shape[0])
    b = (xyz[p] - xyz[q]) / WAVELENGTH
    bx, by, bz = b[:, 0], b[:, 1], b[:, 2]
    sd, cd = math.sin(DECLINATION), math.cos(DECLINATION)
    hs = np.linspace(-h_max_hours, h_max_hours, n_steps) * (math.pi / 12.0)
    out, ps, qs = [], [], []
    for h in hs:
        sh, ch = math.sin(h), math.cos(h)
        u = sh * bx + ch * by
        v = -sd * ch * bx + sd * sh * by + cd * bz
        w = cd * ch * bx - cd * sh * by + sd * bz
        out.append(np.stack([u, v, w], axis=1))
        ps.append(p)
        qs.append(q)
    return np.concatenate(out), np.concatenate(ps), np.concatenate(qs)


def _uvw_coplanar(enu: np.ndarray, n_keep: int):
    p, q = _pairs(enu.shape[0])
    de = (enu[p, 0] - enu[q, 0]) / WAVELENGTH
    dn = (enu[p, 1] - enu[q, 1]) / WAVELENGTH
    out, ps, qs = [], [], []
    for s in range(9):
        th = math.pi * s / 9.0
        c, sn = math.cos(th), math.sin(th)
        out.append(np.stack([c * de - sn * dn, sn * de + c * dn, np.zeros_like(de)], axis=1))
        ps.append(p)
        qs.append(q)
    uvw = np.concatenate(out)[:n_keep]
    return uvw, np.concatenate(ps)[:n_keep], np.concatenate(qs)[:n_keep]


def _grid(n_side: int, delta: float, offset: float = 0.0):
    k = np.arange(n_side * n_side)
    l = (k % n_side - n_side // 2) * delta + offset
    m = (k // n_side - n_side // 2) * delta + offset
    return l.astype(np.float64), m.astype(np.float64)


def _inner_pixels(n_side: int) -> np.ndarray:
    """Linear indices of the inner 80 % of an n_side x n_side grid."""
    lo = int(round(0.1 * n_side))
    hi = n_side - lo
    ii = np.arange(lo, hi)
    return (ii[:, None] * n_side + ii[None, :]).ravel()


def _fluxes(rng: np.random.Generator, n: int) -> np.ndarray:
    return np.clip(0.1 * (1.0 + rng.pareto(1.5, size=n)), 0.1, 10.0)


def _noise(rng: np.random.Generator, n_vis: int, sigma_n: float) -> np.ndarray:
    re = rng.standard_normal(n_vis)
    im = rng.standard_normal(n_vis)
    return sigma_n * (re + 1j * im)


def fista_lambda(wl: Workload) -> float:
    """lambda = 3 sigma_n sqrt(N_v) [reading]; the noiseless config 4 takes its lambda from the
    dirty image, which needs the operator, so the caller computes it."""
    return 3.0 * wl.sigma_n * math.sqrt(wl.n_vis)


# ----------------------------------------------------------------------------- configs
_DEFAULTS = {
    1: dict(n_side=32, n_ant=16, n_vis=1000, n_src=10, sigma_n=0.01, n_iter=200, diameter=1000.0),
    2: dict(n_side=256, n_ant=64, n_steps=10, h_max=2.0, fov_deg=2.0, n_src=200, sigma_n=0.05,
            n_iter=50, diameter=3000.0),
    3: dict(n_side=256, n_ant=64, n_steps=10, h_max=2.0, fov_deg=2.0, n_src=100, n_blob=20,
            sigma_n=0.05, n_iter=25, diameter=3000.0, gauss_model=GAUSS_WIDEFIELD),
    4: dict(n_side=512, n_ant=128, n_steps=8, h_max=2.0, fov_deg=20.0, n_src=1000, sigma_n=0.0,
            n_iter=5, diameter=3000.0),
    5: dict(n_side=1024, n_ant=128, n_steps=50, h_max=3.0, fov_deg=30.0, n_src=5000, sigma_n=0.1,
            n_iter=2, diameter=3000.0),
}

_NAMES = {
    1: "tiny-coplanar",
    2: "narrow-noncoplanar",
    3: "multiscale-gaussian",
    4: "ddgains-widefield",
    5: "paper-scale-widefield",
}


def make_workload(cid: int, **overrides) -> Workload:
    """Build config `cid` (1..5).  `overrides` shrink a config for tests (e.g. n_side=64,
    n_ant=16, n_steps=4, n_src=50); the draw order and formulas are unchanged."""
    if cid not in _DEFAULTS:
        raise ValueError(f"unknown config {cid}")
    prm = dict(_DEFAULTS[cid])
    unknown = set(overrides) - set(prm)
    if unknown:
        raise ValueError(f"unknown override(s) {sorted(unknown)} for config {cid}")
    prm.update(overrides)
    rng = np.random.default_rng(1310207800 + cid)
    n_side, n_ant = int(prm["n_side"]), int(prm["n_ant"])

    # 1. antennas
    enu = _antennas(rng, n_ant, prm["diameter"])
    if cid == 1:
        uvw, ant_p, ant_q = _uvw_coplanar(enu, int(prm["n_vis"]))
        delta = 0.1 / n_side
    else:
        uvw, ant_p, ant_q = _uvw_synthesis(enu, prm["h_max"], int(prm["n_steps"]))
        delta = 2.0 * math.sin(math.radians(prm["fov_deg"]) / 2.0) / n_side

    # 2. pixel list (+ jitter for config 4)
    sigma = None
    if cid == 3:
        ls, ms, ss = [], [], []
        for s, sig in enumerate((0.5, 1.0, 2.0)):
            ns = n_side >> s
            step = delta * (1 << s)
            ll, mm = _grid(ns, step, offset=((1 << s) - 1) * delta / 2.0)
            ls.append(ll)
            ms.append(mm)
            ss.append(np.full(ns * ns, sig * delta))
        l, m, sigma = np.concatenate(ls), np.concatenate(ms), np.concatenate(ss)
    else:
        l, m = _grid(n_side, delta)
    if cid == 4:
        l = l + rng.uniform(-0.3, 0.3, size=l.shape) * delta
        m = m + rng.uniform(-0.3, 0.3, size=m.shape) * delta

    # 3. source pixels, 4. fluxes  (on the finest grid, which is the first n_side^2 pixels)
    inner = _inner_pixels(n_side)
    n_src = int(prm["n_src"])
    src = rng.choice(inner, size=n_src, replace=False)
    x_true = np.zeros(l.shape[0], dtype=np.float64)
    x_true[src] = _fluxes(rng, n_src)

    # 5. blobs (config 3): a separate truth pixel list evaluated with eq (17)
    truth_extra = None
    if cid == 3:
        nb = int(prm["n_blob"])
        half = 0.4 * n_side * delta
        bl = rng.uniform(-half, half, size=nb)
        bm = rng.uniform(-half, half, size=nb)
        bs = rng.uniform(1.0, 8.0, size=nb) * delta
        bf = _fluxes(rng, nb)
        truth_extra = dict(l=bl, m=bm, sigma=bs, flux=bf)

    # 6. gains (config 4): Gaussian primary beam x smooth per-antenna complex perturbation
    gains = None
    if cid == 4:
        z = (rng.standard_normal((n_ant, 3)) + 1j * rng.standard_normal((n_ant, 3))) / math.sqrt(2.0)
        theta = np.arcsin(np.sqrt(l * l + m * m))
        b_pow = np.exp(-4.0 * math.log(2.0) * (theta / math.radians(25.0)) ** 2)
        b_amp = np.sqrt(b_pow)
        l_max = 0.5 * n_side * delta
        pert = z[:, 0:1] + z[:, 1:2] * (l / l_max)[None, :] + z[:, 2:3] * (m / l_max)[None, :]
        gains = (b_amp[None, :] * (1.0 + 0.05 * pert)).astype(np.complex64)

    # 7. noise
    noise = _noise(rng, uvw.shape[0], float(prm["sigma_n"]))

    return Workload(
        cid=cid, name=_NAMES[cid], uvw=np.ascontiguousarray(uvw, dtype=np.float64),
        ant_p=np.ascontiguousarray(ant_p, dtype=np.int32),
        ant_q=np.ascontiguousarray(ant_q, dtype=np.int32), n_ant=n_ant,
        l=np.ascontiguousarray(l), m=np.ascontiguousarray(m), sigma=sigma, gains=gains,
        gauss_model=int(prm.get("gauss_model", GAUSS_WIDEFIELD)), x_true=x_true,
        truth_extra=truth_extra, noise=noise, sigma_n=float(prm["sigma_n"]),
        n_iter=int(prm["n_iter"]), delta=float(delta), meta=prm,
    )
