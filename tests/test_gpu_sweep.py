"""Seeded sweeps over the argument space of the two plan types: band limits from 0 up, mmax < lmax, both dtypes, both
up-sampling factors, every accuracy the plan accepts, point sets from none to clustered / degenerate ones, ring grids
with poles, single-pixel rings and every FFT route.  Each case is checked against the CPU oracle (Eq. 3 / Eq. 2 by
their direct sums).  Fixed seeds: the same cases every run."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2406_14542_b200 import inputs  # noqa: E402


@pytest.fixture(scope="module")
def nusht():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2406_14542_b200 import nusht as n
    return n


def cu(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def field_rms(alm, L):
    """rms over the sphere of the field with these coefficients: sqrt(sum_lm w_m |a_lm|^2 / 4 pi).  The accuracy of
    the nuFFT is relative to this scale, not to the value at one point (a single output can be small by cancellation)."""
    wm = np.where(np.arange(len(alm)) <= L, 1.0, 2.0)
    return np.sqrt(np.sum(wm * np.abs(alm) ** 2) / (4 * np.pi)) + 1e-300


def test_nusht_argument_sweep(nusht, oracle):
    rng = np.random.default_rng(20240614)
    for case in range(300):
        L = int(rng.choice([0, 1, 2, 3, 5, 17, 31, 32, 63, 64, 100, 127, 128, 200, 255, 300]))
        M = int(rng.integers(0, L + 1)) if rng.random() < 0.5 else L
        dtype = "f32" if rng.random() < 0.3 else "f64"
        sigma = 1.25 if rng.random() < 0.3 else None
        if dtype == "f64":
            eps = float(rng.choice([1e-2, 1e-4, 1e-6, 1e-8, 1e-10] + ([1e-12, 1e-13] if sigma is None else [])))
        else:
            eps = float(rng.choice([1e-1, 1e-3, 1e-5] + ([1e-6] if sigma is None else [])))
        npts = int(rng.choice([0, 1, 2, 31, 32, 33, 500, 3000]))
        kind = int(rng.integers(0, 4))
        if kind == 0:
            theta, phi = inputs.uniform_sphere_points(npts, int(rng.integers(1 << 30)))
        elif kind == 1:                                   # clustered at a pole
            theta, phi = np.abs(rng.normal(0, 1e-3, npts)), rng.uniform(0, 2 * np.pi, npts)
            if rng.random() < 0.5:
                theta = np.pi - theta
        elif kind == 2:                                   # one small patch across the phi = 0 seam
            theta = 1.0 + rng.uniform(0, 1e-4, npts)
            phi = (6.2831 + rng.uniform(0, 1e-3, npts)) % (2 * np.pi)
        else:                                             # exact special values
            theta = rng.choice([0.0, np.pi, np.pi / 2, 1e-300, np.pi - 1e-16], npts)
            phi = rng.choice([0.0, 2 * np.pi - 1e-16, np.pi, 1e-300], npts)
        theta = np.clip(theta, 0, np.pi)
        tag = (case, L, M, dtype, sigma, eps, npts, kind)
        plan = nusht.Plan(L, M, cu(theta) if npts else None, cu(phi) if npts else None, eps, dtype=dtype, sigma=sigma)
        cd, rd = (np.complex128, np.float64) if dtype == "f64" else (np.complex64, np.float32)
        alm = inputs.random_alm(L, M, int(rng.integers(1 << 30)))
        x = inputs.random_map(npts, int(rng.integers(1 << 30))).astype(rd)
        f = plan.synthesis(cu(alm.astype(cd))).cpu().numpy().astype(np.float64)
        c = plan.adjoint(cu(x)).cpu().numpy().astype(np.complex128)
        plan.destroy()
        assert np.all(np.isfinite(f)) and np.all(np.isfinite(c.view(np.float64))), tag
        if npts == 0:
            assert f.size == 0 and np.all(c == 0), tag
            continue
        bar = 10 * eps if dtype == "f64" else max(10 * eps, 1e-4)
        ns = min(npts, 300)
        f_ref = oracle.synthesis(L, M, theta[:ns], phi[:ns], alm, "ld")
        assert np.linalg.norm(f[:ns] - f_ref) <= bar * np.sqrt(ns) * field_rms(alm, L), tag
        c_ref = oracle.adjoint(L, M, theta, phi, x.astype(np.float64), "ld")
        # (the adjoint's error is relative to the scale of the input map; c itself can be small by cancellation,
        # e.g. m > 0 coefficients of points at a pole: hence the factor 10)
        assert np.linalg.norm(c - c_ref) <= 10 * bar * np.linalg.norm(c_ref) + 1e-300, tag


def test_ring_plan_argument_sweep(nusht, oracle, monkeypatch):
    rng = np.random.default_rng(20240615)
    for case in range(300):
        L = int(rng.choice([0, 1, 2, 5, 17, 40, 63, 100, 150]))
        M = int(rng.integers(0, L + 1)) if rng.random() < 0.5 else L
        nr = int(rng.choice([1, 2, 3, 8, 17, 40]))
        theta = np.arccos(rng.uniform(-1, 1, nr))
        if rng.random() < 0.3:
            theta[0] = 0.0
        if rng.random() < 0.3 and nr > 1:
            theta[1] = np.pi - theta[0]
        style = int(rng.integers(0, 3))
        nphi = (rng.integers(1, 300, nr) if style == 0 else
                np.full(nr, int(rng.choice([1, 2, 7, 64, 96, 255]))) if style == 1 else 4 * (1 + np.arange(nr)))
        phi0, w = rng.uniform(-7, 7, nr), rng.uniform(0.1, 2, nr)
        dtype = "f32" if rng.random() < 0.25 else "f64"
        mode = str(rng.choice(["0", "all", ""]))
        if mode:
            monkeypatch.setenv("NUSHT_RING_POOL", mode)
        else:
            monkeypatch.delenv("NUSHT_RING_POOL", raising=False)
        tag = (case, L, M, nr, style, dtype, mode)
        plan = nusht.RingPlan(L, M, theta, nphi, phi0, w, dtype=dtype)
        th = np.repeat(theta, nphi)
        ph = np.concatenate([p0 + 2 * np.pi * np.arange(n) / n for n, p0 in zip(nphi, phi0)])
        cd, rd = (np.complex128, np.float64) if dtype == "f64" else (np.complex64, np.float32)
        alm = inputs.random_alm(L, M, int(rng.integers(1 << 30)))
        x = inputs.random_map(len(th), int(rng.integers(1 << 30))).astype(rd)
        f = plan.synthesis(cu(alm.astype(cd))).cpu().numpy().astype(np.float64)
        c = plan.analysis(cu(x)).cpu().numpy().astype(np.complex128)
        plan.destroy()
        f_ref = oracle.synthesis(L, M, th, ph, alm, "ld")
        c_ref = oracle.adjoint(L, M, th, ph, np.repeat(w, nphi) * x.astype(np.float64), "ld")
        bar = 1e-12 if dtype == "f64" else 5e-6
        assert np.linalg.norm(f - f_ref) <= bar * np.sqrt(len(th)) * field_rms(alm, L), tag
        assert np.linalg.norm(c - c_ref) <= 10 * bar * np.linalg.norm(c_ref) + 1e-300, tag
