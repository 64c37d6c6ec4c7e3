"""GPU parity of the pointing kernel (Eq. C1; csrc/pointing.cu) against oracle.pointing
(numpy long double).  FP64 on both sides; the bar is a few ulp of the angles: |d theta'| <= 4e-15 and
sin(theta') |d phi'| <= 4e-15 (phi' itself is ill-conditioned next to the poles: the error of the POSITION is
what is bounded), phi' compared modulo 2 pi."""
import ctypes

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

ARCMIN = np.pi / (180 * 60)


@pytest.fixture(scope="module")
def nusht():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2406_14542_b200 import nusht as n
    return n


def cu(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def check(nusht, oracle, th, ph, at, ap, tol=4e-15):
    t2, p2 = nusht.nusht_pointing(cu(th), cu(ph), cu(at), cu(ap))
    t2, p2 = t2.cpu().numpy(), p2.cpu().numpy()
    tr, pr = oracle.pointing(th, ph, at, ap)
    assert np.all((t2 >= 0) & (t2 <= np.pi) & (p2 >= 0) & (p2 < 2 * np.pi))
    dt = np.abs(np.asarray(np.longdouble(t2) - tr, dtype=np.float64))
    dp = np.abs(np.asarray(np.longdouble(p2) - pr, dtype=np.float64))
    dp = np.minimum(dp, 2 * np.pi - dp)
    assert dt.max() <= tol, dt.max()
    assert (np.sin(np.asarray(tr, dtype=np.float64)) * dp).max() <= tol, (np.sin(np.asarray(tr, dtype=np.float64)) * dp).max()
    return t2, p2


@pytest.mark.parametrize("nrings,npix", [(64, 64), (1000, 777)])
def test_lensing_like_deflections_on_a_ring_grid(nusht, oracle, nrings, npix):
    """Config-2 recipe: equi-angular rings, iid deflections of 2.5 arcmin rms; several
    CTAs and a ragged tail."""
    rng = np.random.default_rng(41)
    th = np.repeat(np.pi * (np.arange(nrings) + 0.5) / nrings, npix)
    ph = np.tile(2 * np.pi * np.arange(npix) / npix, nrings)
    at, ap = rng.normal(0, 2.5 * ARCMIN, th.size), rng.normal(0, 2.5 * ARCMIN, th.size)
    check(nusht, oracle, th, ph, at, ap)


def test_large_deflections_poles_and_zero(nusht, oracle):
    rng = np.random.default_rng(42)
    n = 100003
    th, ph = np.arccos(rng.uniform(-1, 1, n)), rng.uniform(0, 2 * np.pi, n)
    at, ap = rng.normal(0, 0.5, n), rng.normal(0, 0.5, n)
    th[:6] = [0.0, np.pi, 1e-12, np.pi - 1e-12, 0.5, 0.5]
    at[4], ap[4] = 0.0, 0.0                        # zero deflection: the identity
    at[5], ap[5] = 1e-300, 0.0                     # sin(a)/a at a tiny a
    ph[6], at[6], ap[6] = 2 * np.pi - 1e-9, 0.0, 1e-3    # phi' wraps through 2 pi
    ph[7], at[7], ap[7] = 1e-9, 0.0, -1e-3               # and through 0
    t2, p2 = check(nusht, oracle, th, ph, at, ap)
    assert t2[4] == th[4] and abs(p2[4] - ph[4]) <= 1e-15
    # a = pi/2 .. pi: the far side of the sphere
    at2 = rng.uniform(1.5, 3.1, n)
    check(nusht, oracle, th, ph, at2, np.zeros(n))


def test_pointed_positions_feed_the_transform(nusht, oracle):
    """The use the paper makes of it: synthesis at the deflected positions equals the oracle's
    direct sum at the oracle's deflected positions."""
    from paper_2406_14542_b200 import inputs
    L, eps = 63, 1e-10
    rng = np.random.default_rng(43)
    th = np.repeat(np.pi * (np.arange(96) + 0.5) / 96, 128)
    ph = np.tile(2 * np.pi * np.arange(128) / 128, 96)
    at, ap = rng.normal(0, 20 * ARCMIN, th.size), rng.normal(0, 20 * ARCMIN, th.size)
    t2, p2 = nusht.nusht_pointing(cu(th), cu(ph), cu(at), cu(ap))
    alm = inputs.random_alm(L, L, 43)
    plan = nusht.Plan(L, L, t2, p2, eps)
    f = plan.synthesis(cu(alm)).cpu().numpy()
    tr, pr = oracle.pointing(th, ph, at, ap)
    f_ref = oracle.synthesis(L, L, np.asarray(tr, dtype=np.float64), np.asarray(pr, dtype=np.float64), alm, "ld")
    assert np.linalg.norm(f - f_ref) / np.linalg.norm(f_ref) <= 10 * eps
    plan.destroy()


def test_pointing_argument_checks(nusht):
    lib = nusht.lib
    assert lib.nusht_pointing(0, None, None, None, None, None, None, None) == 0       # npts = 0: no-op
    assert lib.nusht_pointing(-1, None, None, None, None, None, None, None) == -1
    assert lib.nusht_pointing(8, None, None, None, None, None, None, None) == -1      # NULL arrays
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    t2, p2 = nusht.nusht_pointing(e, e, e, e)
    assert t2.numel() == 0 and p2.numel() == 0
