"""Seeded synthetic inputs shared by the CUDA path's tests/bench and the oracle.

This module holds NO arithmetic of the method (no Legendre functions, no FFT, no kernels): only
random draws and the geometry of the workloads.  Recipes follow BASELINE.json `configs` and
SURVEY.md 8(d); see DESIGN.md "Input recipe".

* points uniform on the sphere: theta = arccos(U[-1,1]), phi ~ U[0, 2 pi)
* CMB-lensing-like points (config 2): an equi-angular ring grid and, per pixel, an iid Gaussian
  deflection (sigma = 2.5 arcmin per component => |alpha| ~ Rayleigh(sigma)); the displaced
  positions (arXiv 2406.14542 Eq. C1) are NOT computed here but by
  nusht_pointing / oracle.pointing from these draws.  The paper's real deflection fields
   are not available offline, this stands in for them.
* a_lm: complex, m >= 0, real-field convention, m-major triangular layout
  idx(l, m) = m (2 lmax + 1 - m)/2 + l; white (C_l = 1) or C_l = 1/(l+1)^2.
"""
from __future__ import annotations

import numpy as np

ARCMIN = np.pi / 180.0 / 60.0


def nlm(lmax: int, mmax: int) -> int:
    return (mmax + 1) * (lmax + 1) - mmax * (mmax + 1) // 2


def lm_index(lmax: int, l, m):
    return m * (2 * lmax + 1 - m) // 2 + l


def uniform_sphere_points(npts: int, seed: int):
    rng = np.random.default_rng(seed)
    theta = np.arccos(rng.uniform(-1.0, 1.0, size=npts))
    phi = rng.uniform(0.0, 2.0 * np.pi, size=npts)
    return theta, phi


def random_alm(lmax: int, mmax: int, seed: int, spectrum: str = "white"):
    """Complex alm with E|a_lm|^2 = C_l.  'white': Re, Im ~ N(0,1) for m > 0 and a_l0 ~ N(0,1) real
    (BASELINE.json configs 1 and 3).  'inv_l2': C_l = 1/(l+1)^2, Re, Im variance C_l/2, a_l0 real
    with variance C_l (configs 2 and 4)."""
    rng = np.random.default_rng(seed + 1000003)
    n = nlm(lmax, mmax)
    re = rng.standard_normal(n)
    im = rng.standard_normal(n)
    alm = np.empty(n, dtype=np.complex128)
    if spectrum == "white":
        alm.real, alm.imag = re, im
        alm[: lmax + 1] = re[: lmax + 1]
    elif spectrum == "inv_l2":
        for m in range(mmax + 1):
            lo = lm_index(lmax, m, m)
            l = np.arange(m, lmax + 1)
            amp = 1.0 / (l + 1.0)
            sl = slice(lo, lo + lmax - m + 1)
            if m == 0:
                alm[sl] = re[sl] * amp
            else:
                alm[sl] = (re[sl] + 1j * im[sl]) * (amp / np.sqrt(2.0))
    else:
        raise ValueError(spectrum)
    return alm


def random_map(npts: int, seed: int):
    rng = np.random.default_rng(seed + 2000003)
    return rng.standard_normal(npts)


def lensing_grid_and_deflection(nrings: int, npix: int, seed: int, sigma: float = 2.5 * ARCMIN):
    """The undeflected nrings x npix equi-angular grid theta_i = pi (i + 1/2)/nrings, phi_j = 2 pi j/npix (ring-major
    order) and an iid Gaussian deflection (alpha_theta, alpha_phi) per pixel, each component N(0, sigma^2), so that
    |alpha| ~ Rayleigh(sigma) along a uniformly random direction (BASELINE.json configs[1]).  Random draws only: the
    deflected positions of Eq. C1 are computed by nusht_pointing on the CUDA side and by
    oracle.pointing on the checker's side, each from these same arrays."""
    rng = np.random.default_rng(seed)
    th = np.pi * (np.arange(nrings) + 0.5) / nrings
    ph = 2.0 * np.pi * np.arange(npix) / npix
    theta = np.repeat(th, npix)
    phi = np.tile(ph, nrings)
    a_t = rng.normal(0.0, sigma, size=theta.shape[0])
    a_p = rng.normal(0.0, sigma, size=theta.shape[0])
    return theta, phi, a_t, a_p


# BASELINE.json `configs`, in order.  npts / spectrum / eps / dtype per config.
CONFIGS = {
    1: dict(lmax=63, mmax=63, eps=1e-10, dtype="f64", npts=16384, points="uniform", spectrum="white", seed=0),
    2: dict(lmax=1023, mmax=1023, eps=1e-10, dtype="f64", npts=2048 * 2048, points="lensing", spectrum="inv_l2", seed=2),
    3: dict(lmax=4095, mmax=4095, eps=1e-10, dtype="f64", npts=4 * 4096 * 4096, points="uniform", spectrum="white", seed=3),
    4: dict(lmax=8191, mmax=8191, eps=1e-8, dtype="f64", npts=2 * 8192 * 8192, points="uniform", spectrum="inv_l2", seed=4),
    # not a BASELINE.json config: twice the band limit of the largest one (the paper's A100 limit is lmax ~ 9000,
    # PAPER.md:156), 2 (lmax + 1)^2 points as in config 4; 108 GB of plan workspace at sigma = 2
    6: dict(lmax=16383, mmax=16383, eps=1e-10, dtype="f64", npts=2 * 16384 * 16384, points="uniform", spectrum="inv_l2", seed=6),
}


def make_config(i: int, npts: int | None = None):
    """(cfg, theta, phi, alm, x) for BASELINE config i; `npts` overrides the point count (tests).
    For the lensing-like config the returned (theta, phi) is the UNDEFLECTED pixel grid and cfg["deflection"] holds
    (alpha_theta, alpha_phi): the caller turns them into the point set with Eq. C1, through nusht_pointing (CUDA
    path) or oracle.pointing (checker).  cfg["deflection"] is None for the other configs."""
    cfg = dict(CONFIGS[i])
    cfg["deflection"] = None
    if npts is not None:
        cfg["npts"] = int(npts)
    if cfg["points"] == "uniform":
        theta, phi = uniform_sphere_points(cfg["npts"], cfg["seed"])
    else:
        side = int(round(np.sqrt(cfg["npts"])))
        theta, phi, a_t, a_p = lensing_grid_and_deflection(side, side, cfg["seed"])
        cfg["deflection"] = (a_t, a_p)
        cfg["npts"] = side * side
    alm = random_alm(cfg["lmax"], cfg["mmax"], cfg["seed"], cfg["spectrum"])
    x = random_map(cfg["npts"], cfg["seed"])
    return cfg, theta, phi, alm, x


def healpix_ring_layout(nside: int):
    """Ring layout of the HEALPix pixelisation (Gorski et al. 2005; "standard pixelization schemes such as
    HEALPix"), restated from its definition: 4 nside - 1 rings; polar caps with 4 i pixels on ring i at
    cos(theta) = 1 - i^2 / (3 nside^2), first pixel at pi / (4 i); equatorial belt with 4 nside pixels at
    cos(theta) = 4/3 - 2 i / (3 nside), shifted by half a pixel on every other ring.  Returns (theta, nphi, phi0,
    weight) with the equal-area weight 4 pi / npix.  Geometry only: no transform arithmetic."""
    theta, nphi, phi0 = [], [], []
    for i in range(1, 4 * nside):
        if i < nside:
            z, n, p0 = 1 - i * i / (3.0 * nside * nside), 4 * i, np.pi / (4 * i)
        elif i <= 3 * nside:
            z, n = 4.0 / 3 - 2.0 * i / (3 * nside), 4 * nside
            p0 = ((i - nside + 1) % 2) * np.pi / (4 * nside)
        else:
            k = 4 * nside - i
            z, n, p0 = -(1 - k * k / (3.0 * nside * nside)), 4 * k, np.pi / (4 * k)
        theta.append(np.arccos(z))
        nphi.append(n)
        phi0.append(p0)
    theta = np.array(theta)
    half = len(theta) // 2                      # exact mirror symmetry of the colatitudes
    theta[len(theta) - half:] = np.pi - theta[:half][::-1]
    nphi = np.array(nphi, dtype=np.int64)
    return theta, nphi, np.array(phi0), np.full(len(theta), 4 * np.pi / float(nphi.sum()))

