"""Pins for the CPU oracle (oracle/): everything here is CPU-only and checks the oracle against
things OTHER than itself -- closed forms, library routines (mpmath, scipy), invariants.

Citations: arXiv 2406.14542 Eq. 1-3, fn. 4; readings G1-G3, G12
and pins P1-P8 in DESIGN.md / SURVEY.md 8(c).
"""
import os

import numpy as np
import pytest

from paper_2406_14542_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "plm_mpmath.txt")


def single_alm(lmax, mmax, l, m, val):
    a = np.zeros(inputs.nlm(lmax, mmax), dtype=np.complex128)
    a[inputs.lm_index(lmax, l, m)] = val
    return a


def closed_form(l, m, th, ph):
    """Orthonormal, Condon-Shortley Y_lm for l <= 2 (textbook table)."""
    s, c = np.sin(th), np.cos(th)
    e = np.exp(1j * m * ph)
    tab = {
        (0, 0): np.sqrt(1 / (4 * np.pi)) * np.ones_like(th),
        (1, 0): np.sqrt(3 / (4 * np.pi)) * c,
        (1, 1): -np.sqrt(3 / (8 * np.pi)) * s,
        (2, 0): np.sqrt(5 / (16 * np.pi)) * (3 * c * c - 1),
        (2, 1): -np.sqrt(15 / (8 * np.pi)) * s * c,
        (2, 2): np.sqrt(15 / (32 * np.pi)) * s * s,
    }
    return tab[(l, m)] * e


# ---- P1: closed forms, through the full synthesis entry point (layout, w_m, phase) ------------
@pytest.mark.parametrize("l,m", [(0, 0), (1, 0), (1, 1), (2, 0), (2, 1), (2, 2)])
@pytest.mark.parametrize("prec", ["d", "ld"])
def test_closed_forms_synthesis(oracle, l, m, prec):
    rng = np.random.default_rng(l * 10 + m)
    th = np.arccos(rng.uniform(-1, 1, 200))
    ph = rng.uniform(0, 2 * np.pi, 200)
    lmax, mmax = 5, 4
    a = 0.7 - 1.3j if m > 0 else 0.7 + 0j
    f = oracle.synthesis(lmax, mmax, th, ph, single_alm(lmax, mmax, l, m, a), prec)
    wm = 1.0 if m == 0 else 2.0
    ref = wm * np.real(a * closed_form(l, m, th, ph))
    assert np.max(np.abs(f - ref)) < 2e-15


def test_im_al0_ignored(oracle):
    th, ph = inputs.uniform_sphere_points(50, 1)
    a = inputs.random_alm(6, 6, 1)
    b = a.copy()
    b[:7] += 1j * np.arange(1, 8)
    assert np.array_equal(oracle.synthesis(6, 6, th, ph, a), oracle.synthesis(6, 6, th, ph, b))


# ---- P5: mpmath library values (stored; generator beside the file) ---------------------------
def _golden():
    rows = []
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        l, m, thx, frac, ex = line.split()
        rows.append((int(l), int(m), float.fromhex(thx), float(frac), int(ex)))
    return rows


@pytest.mark.parametrize("prec,eps", [("ld", 2.0 ** -64), ("d", 2.0 ** -53)])
def test_plm_vs_mpmath_golden(oracle, prec, eps):
    for l, m, th, frac, ex in _golden():
        mant, e2 = oracle.plm(l, m, th, prec)
        # same binary exponent, or off by one when the fraction sits at the 0.5/1 boundary
        assert abs(e2 - ex) <= 1, (l, m, th)
        got = mant * 2.0 ** (e2 - ex)
        # near a zero of Pbar (equator, odd l+m) the value is set by cos(theta) rounding: skip rel check
        if abs(np.cos(th)) < 1e-15:
            continue
        # rounding of cos(theta) moves theta by eps/sin(theta); dPbar/dtheta ~ l Pbar; plus O(l) steps
        tol = eps * (2000.0 + 8.0 * l / max(np.sin(th), 1e-3))
        assert abs(got / frac - 1.0) < tol, (l, m, th, got / frac - 1.0, tol)


def test_plm_vs_mpmath_live(oracle):
    mp = pytest.importorskip("mpmath")
    mp.mp.dps = 40
    rng = np.random.default_rng(7)
    for _ in range(60):
        l = int(rng.integers(0, 300))
        m = int(rng.integers(0, l + 1))
        th = float(np.arccos(rng.uniform(-1, 1)))
        ref = mp.re(mp.spherharm(l, m, mp.mpf(th), 0, maxprec=100000))
        got = oracle.plm_value(l, m, th, "ld")
        scale = np.sqrt((2 * l + 1) / (4 * np.pi))
        assert abs(got - float(ref)) < 1e-14 * scale, (l, m, th)


# ---- P6: scipy library cross-check through synthesis and adjoint -----------------------------
def test_vs_scipy_sph_harm(oracle):
    sp = pytest.importorskip("scipy.special")
    if not hasattr(sp, "sph_harm_y"):
        pytest.skip("scipy without sph_harm_y")
    lmax = mmax = 40
    th, ph = inputs.uniform_sphere_points(300, 11)
    a = inputs.random_alm(lmax, mmax, 11)
    ref = np.zeros(300)
    for m in range(mmax + 1):
        for l in range(m, lmax + 1):
            y = sp.sph_harm_y(l, m, th, ph)
            c = a[inputs.lm_index(lmax, l, m)]
            ref += (c.real * y.real) if m == 0 else 2 * np.real(c * y)
    f = oracle.synthesis(lmax, mmax, th, ph, a)
    assert np.linalg.norm(f - ref) / np.linalg.norm(ref) < 5e-14
    # adjoint: c_lm = sum_j x_j conj(Y_lm)
    x = inputs.random_map(300, 11)
    c = oracle.adjoint(lmax, mmax, th, ph, x)
    for (l, m) in [(0, 0), (7, 0), (7, 3), (40, 40), (39, 1), (40, 0)]:
        r = np.sum(x * np.conj(sp.sph_harm_y(l, m, th, ph)))
        if m == 0:
            r = r.real
        assert abs(c[inputs.lm_index(lmax, l, m)] - r) < 1e-12


# ---- P2: addition theorem sum_m |Y_lm|^2 = (2l+1)/4pi, incl. near-pole and large l -----------
@pytest.mark.parametrize("l", [0, 1, 15, 200, 1023, 4095])
@pytest.mark.parametrize("theta", [1e-3, 0.05, 0.9, np.pi / 2, 3.0])
def test_addition_theorem(oracle, l, theta):
    tot = oracle.plm_value(l, 0, theta) ** 2
    for m in range(1, l + 1):
        tot += 2 * oracle.plm_value(l, m, theta) ** 2
    tol = 2e-10 if l > 1000 else 1e-11
    assert abs(tot / ((2 * l + 1) / (4 * np.pi)) - 1) < tol


# ---- parity Pbar_lm(pi - theta) = (-1)^(l+m) Pbar_lm(theta) ------------------------------------
def test_parity(oracle):
    for (l, m, th) in [(5, 2, 0.4), (6, 2, 0.4), (101, 50, 1.1), (100, 50, 1.1)]:
        a = oracle.plm_value(l, m, th, "ld")
        b = oracle.plm_value(l, m, np.pi - th, "ld")
        assert abs(b - (-1) ** (l + m) * a) < 1e-13 * (1 + abs(a))


# ---- P3: orthonormality under Gauss-Legendre quadrature ---------------------------------------
@pytest.mark.parametrize("lmax,mmax", [(0, 0), (7, 7), (24, 24), (32, 20)])
def test_gauss_legendre_orthonormality(oracle, lmax, mmax):
    xg, wg = np.polynomial.legendre.leggauss(lmax + 1)
    nph = 2 * lmax + 2
    th = np.repeat(np.arccos(xg), nph)
    ph = np.tile(2 * np.pi * np.arange(nph) / nph, lmax + 1)
    w = np.repeat(wg, nph) * (2 * np.pi / nph)
    a = inputs.random_alm(lmax, mmax, 5)
    f = oracle.synthesis(lmax, mmax, th, ph, a)
    back = oracle.adjoint(lmax, mmax, th, ph, w * f)
    assert np.max(np.abs(back - a)) < 1e-13 * max(1.0, np.max(np.abs(a))) * (lmax + 1)


# ---- P4: adjoint identity with the G3 inner product -------------------------------------------
@pytest.mark.parametrize("lmax,mmax,npts", [(12, 12, 500), (63, 63, 2000), (63, 17, 1000)])
def test_adjoint_identity(oracle, lmax, mmax, npts):
    th, ph = inputs.uniform_sphere_points(npts, 3)
    a = inputs.random_alm(lmax, mmax, 3)
    x = inputs.random_map(npts, 3)
    f = oracle.synthesis(lmax, mmax, th, ph, a)
    c = oracle.adjoint(lmax, mmax, th, ph, x)
    lhs = float(np.sum(np.longdouble(f) * np.longdouble(x)))
    rhs = oracle.inner_alm(lmax, mmax, a, c)
    assert abs(lhs - rhs) < 1e-13 * np.linalg.norm(f) * np.linalg.norm(x)


def test_adjoint_m0_imag_zero(oracle):
    th, ph = inputs.uniform_sphere_points(100, 4)
    c = oracle.adjoint(8, 8, th, ph, inputs.random_map(100, 4))
    assert np.all(c[:9].imag == 0.0)


# ---- P8: special cases ------------------------------------------------------------------------
def test_lmax_zero(oracle):
    th, ph = inputs.uniform_sphere_points(20, 5)
    f = oracle.synthesis(0, 0, th, ph, np.array([2.5 + 0j]))
    assert np.allclose(f, 2.5 / np.sqrt(4 * np.pi), rtol=0, atol=3e-16)


def test_poles_exact(oracle):
    # theta = 0 or pi: only m = 0 contributes; Pbar_l0(0) = sqrt((2l+1)/4pi), (-1)^l at pi
    lmax = 20
    a = inputs.random_alm(lmax, lmax, 6)
    th = np.array([0.0, np.pi])
    ph = np.array([0.3, 1.7])
    f = oracle.synthesis(lmax, lmax, th, ph, a)
    l = np.arange(lmax + 1)
    n = np.sqrt((2 * l + 1) / (4 * np.pi))
    assert abs(f[0] - np.sum(a[: lmax + 1].real * n)) < 1e-13
    # theta = pi is the binary64 nearest pi: sin = 1.2e-16, so m >= 1 terms are ~1e-16
    assert abs(f[1] - np.sum(a[: lmax + 1].real * n * (-1.0) ** l)) < 1e-13


def test_single_point_adjoint(oracle):
    sp = pytest.importorskip("scipy.special")
    th, ph = np.array([1.234]), np.array([4.321])
    c = oracle.adjoint(9, 9, th, ph, np.array([1.7]))
    for (l, m) in [(0, 0), (3, 2), (9, 9), (9, 0)]:
        r = 1.7 * np.conj(sp.sph_harm_y(l, m, th[0], ph[0]))
        r = r.real if m == 0 else r
        assert abs(c[inputs.lm_index(9, l, m)] - r) < 1e-14


def test_ring_sum_matches_synthesis(oracle):
    lmax = mmax = 30
    m = 7
    a = inputs.random_alm(lmax, mmax, 8)
    lo = inputs.lm_index(lmax, m, m)
    am = a[lo: lo + lmax - m + 1]
    th = np.linspace(0.0, np.pi, 17)
    F = oracle.ring_sum(lmax, m, th, am)
    only = np.zeros_like(a)
    only[lo: lo + lmax - m + 1] = am
    ph = np.full_like(th, 0.37)
    f = oracle.synthesis(lmax, mmax, th, ph, only)
    assert np.max(np.abs(f - 2 * np.real(F * np.exp(1j * m * ph)))) < 1e-14


def test_columns_match_full_adjoint(oracle):
    lmax = 25
    th, ph = inputs.uniform_sphere_points(300, 9)
    x = inputs.random_map(300, 9)
    c = oracle.adjoint(lmax, lmax, th, ph, x)
    cols = oracle.adjoint_columns(lmax, [0, 3, 25], th, ph, x)
    for q, m in enumerate([0, 3, 25]):
        lo = inputs.lm_index(lmax, m, m)
        assert np.array_equal(cols[q, m:], c[lo: lo + lmax - m + 1])
        assert np.all(cols[q, :m] == 0)


def test_double_vs_long_double(oracle):
    lmax = 200
    th, ph = inputs.uniform_sphere_points(200, 10)
    a = inputs.random_alm(lmax, lmax, 10)
    fd = oracle.synthesis(lmax, lmax, th, ph, a, "d")
    fl = oracle.synthesis(lmax, lmax, th, ph, a, "ld")
    assert np.linalg.norm(fd - fl) / np.linalg.norm(fl) < 1e-13


def test_large_lmax_rescaling_synthesis_vs_mpmath(oracle):
    """One high-l coefficient whose Pbar underflows binary64 at the seed: the synthesis entry point
    must reproduce w_m Re(a Y_lm) with Y_lm from mpmath (exercises O2 inside the real code path)."""
    mp = pytest.importorskip("mpmath")
    mp.mp.dps = 40
    lmax = mmax = 2100
    l, m = 2100, 2000            # Pbar_mm(0.4) ~ sin(0.4)^2000 ~ 1e-820
    th = np.array([0.4, 1.2, 2.9])
    ph = np.array([0.1, 2.2, 5.0])
    a = single_alm(lmax, mmax, l, m, 1.0 + 0.5j)
    f = oracle.synthesis(lmax, mmax, th, ph, a)
    for j in range(3):
        y = mp.spherharm(l, m, mp.mpf(float(th[j])), mp.mpf(float(ph[j])), maxprec=400000)
        ref = 2 * float(mp.re(mp.mpc(1.0, 0.5) * y))
        assert abs(f[j] - ref) < 5e-12 * max(abs(ref), 1e-30) + 1e-300


# ---- pointing (Eq. C1) ---------------------------------------------------------
def _unit(theta, phi):
    return np.stack([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)])


def test_pointing_zero_deflection_is_identity(oracle):
    rng = np.random.default_rng(5)
    th, ph = np.arccos(rng.uniform(-1, 1, 1000)), rng.uniform(0, 2 * np.pi, 1000)
    t2, p2 = oracle.pointing(th, ph, np.zeros(1000), np.zeros(1000))
    assert np.max(np.abs(t2 - th)) < 1e-17 + 2e-19 * 10 and np.max(np.abs(np.asarray(p2, dtype=np.float64) - ph)) < 1e-15


def test_pointing_along_the_meridian_and_along_the_equator(oracle):
    """Closed forms: alpha_phi = 0 is a rotation about e_phi, i.e. theta' = theta + alpha_theta at the same phi
    (fixes the sign and direction of e_theta); on the equator alpha_theta = 0 is a rotation about the z axis,
    phi' = phi + alpha_phi at theta' = pi/2 (fixes e_phi)."""
    rng = np.random.default_rng(6)
    th, ph = rng.uniform(0.3, 2.8, 500), rng.uniform(0.3, 6.0, 500)
    a = rng.uniform(-0.2, 0.2, 500)
    t2, p2 = oracle.pointing(th, ph, a, np.zeros(500))
    assert np.max(np.abs(np.asarray(t2 - (np.longdouble(1) * th + a), dtype=np.float64))) < 1e-17
    assert np.max(np.abs(np.asarray(p2, dtype=np.float64) - ph)) < 1e-15
    t3, p3 = oracle.pointing(np.full(500, np.pi / 2), ph, np.zeros(500), a)
    assert np.max(np.abs(np.asarray(t3, dtype=np.float64) - np.pi / 2)) < 1e-15     # pi/2 itself is rounded in binary64
    assert np.max(np.abs(np.asarray(p3, dtype=np.float64) - (ph + a))) < 1e-15


def test_pointing_moves_by_alpha_on_a_great_circle_and_obeys_the_cosine_rule(oracle):
    """Invariants: n' is the unit vector at angular distance alpha from n, and with psi the angle of the
    deflection from e_theta (alpha_theta = alpha cos psi) the spherical triangle (pole, n, n') gives
    cos theta' = cos alpha cos theta - sin alpha sin theta cos psi."""
    rng = np.random.default_rng(7)
    n = 2000
    th, ph = np.arccos(rng.uniform(-1, 1, n)), rng.uniform(0, 2 * np.pi, n)
    alpha, psi = rng.uniform(1e-6, 0.5, n), rng.uniform(0, 2 * np.pi, n)
    t2, p2 = oracle.pointing(th, ph, alpha * np.cos(psi), alpha * np.sin(psi))
    t2, p2 = np.asarray(t2, dtype=np.float64), np.asarray(p2, dtype=np.float64)
    assert np.all((t2 >= 0) & (t2 <= np.pi) & (p2 >= 0) & (p2 < 2 * np.pi))
    cosd = np.sum(_unit(th, ph) * _unit(t2, p2), axis=0)
    assert np.max(np.abs(cosd - np.cos(alpha))) < 5e-16
    assert np.max(np.abs(np.cos(t2) - (np.cos(alpha) * np.cos(th) - np.sin(alpha) * np.sin(th) * np.cos(psi)))) < 5e-16
    # a deflection with a positive alpha_phi moves east: the z component of n x n' is positive
    t4, p4 = oracle.pointing(th, ph, np.zeros(n), alpha)
    u, v = _unit(th, ph), _unit(np.asarray(t4, dtype=np.float64), np.asarray(p4, dtype=np.float64))
    assert np.all((u[0] * v[1] - u[1] * v[0])[np.sin(th) > 1e-3] > 0)


# ---- the exponent-rescaling regime (O2): where the full-size GPU tests use the oracle as truth ----------------
# At lmax >= ~1000 most (m, theta) start with Pbar_mm ~ sin^m(theta) far below binary64 range; the value comes back
# into range through the `renorm` / `sc` refresh inside each copy of the l loop (ring_sum, synthesis,
# adjoint_columns).  The pins above run at lmax <= 63 (or through oracle_plm / oracle_synthesis only), so a slip in
# the ring_sum or adjoint copy of that bookkeeping would go unseen; these run every copy in that regime.
def _near_pole_points(n, seed):
    rng = np.random.default_rng(seed)
    th = np.arccos(rng.uniform(-1, 1, n))
    k = n // 2
    cap = rng.uniform(0.02, 0.6, k)
    th[:k] = np.where(rng.random(k) < 0.5, cap, np.pi - cap)
    th[k] = 1e-3
    return th, rng.uniform(0, 2 * np.pi, n)


@pytest.mark.parametrize("prec,tol", [("d", 1e-14), ("ld", 1e-14)])
def test_adjoint_identity_rescaling_regime(oracle, prec, tol):
    """P4 at lmax = mmax = 1500 with half of the points at theta in [0.02, 0.6] and the mirrored cap: sin^m theta
    leaves the binary64 range for most m there and returns through the sc refresh of BOTH loops (synthesis,
    adjoint_columns).  <S a, x> = <a, S^T x> in the G3 inner product (Eq. 2-3)."""
    L = M = 1500
    th, ph = _near_pole_points(100, 17)
    a = inputs.random_alm(L, M, 17)
    x = inputs.random_map(100, 17)
    f = oracle.synthesis(L, M, th, ph, a, prec)
    c = oracle.adjoint(L, M, th, ph, x, prec)
    lhs = float(np.sum(np.longdouble(f) * np.longdouble(x)))
    rhs = oracle.inner_alm(L, M, a, c)
    assert abs(lhs - rhs) <= tol * np.linalg.norm(f) * np.linalg.norm(x)


@pytest.mark.parametrize("l,m,theta", [(2100, 2000, 0.4), (2100, 300, 0.05), (2100, 2100, 2.9)])
def test_single_point_adjoint_columns_vs_mpmath_rescaling(oracle, l, m, theta):
    """Eq. 2 for one point is c_lm = x conj(Y_lm(theta, phi)); Y_lm from the library routine mpmath.spherharm.
    The seeds are sin(0.4)^2000 ~ 1e-820, sin(0.05)^300 ~ 1e-390 and sin(2.9)^2100 ~ 1e-1300: the value only
    exists through the rescaling of oracle_adjoint_columns (both precisions)."""
    mp = pytest.importorskip("mpmath")
    mp.mp.dps = 40
    phi, xval = 2.2, 1.7
    y = mp.spherharm(l, m, mp.mpf(float(theta)), mp.mpf(float(phi)), maxprec=400000)
    ref = xval * complex(float(mp.re(y)), -float(mp.im(y)))
    for prec, tol in (("d", 5e-12), ("ld", 5e-13)):
        col = oracle.adjoint_columns(l, [m], np.array([theta]), np.array([phi]), np.array([xval]), prec)
        assert abs(col[0, l] - ref) <= tol * abs(ref), (prec, col[0, l], ref)
        # a column of the full adjoint is the same numbers
        assert np.all(col[0, :m] == 0)


@pytest.mark.parametrize("m", [300, 900, 1500])
def test_ring_sum_matches_synthesis_rescaling_regime(oracle, m):
    """ring_sum (the truth of the Legendre stage tests at lmax = 4095 / 8191) against the synthesis entry point
    (itself pinned to mpmath in that regime above) at lmax = 1500 on rings that include the neighbourhood of both
    poles: f = 2 Re(F_m e^{i m phi}) for a_lm supported on one m."""
    L = M = 1500
    a = inputs.random_alm(L, M, 18)
    lo = inputs.lm_index(L, m, m)
    am = a[lo: lo + L - m + 1]
    th = np.concatenate([np.pi * np.arange(0, 1502, 7) / 1501, [0.02, 0.05, 0.3, np.pi - 0.02, np.pi - 0.3]])
    only = np.zeros_like(a)
    only[lo: lo + L - m + 1] = am
    ph = np.full_like(th, 0.37)
    for prec in ("d", "ld"):
        F = oracle.ring_sum(L, m, th, am, prec)
        f = oracle.synthesis(L, M, th, ph, only, prec)
        ref = 2 * np.real(F * np.exp(1j * np.asarray(np.longdouble(m) * np.longdouble(ph), dtype=np.float64)))
        assert np.max(np.abs(f - ref)) <= 2e-13 * np.max(np.abs(f)), (m, prec)
        assert np.max(np.abs(F)) > 0.1      # the column is not all underflow


def test_ring_sum_single_coefficient_vs_mpmath_golden(oracle):
    """ring_sum with one non-zero a_lm must return a Pbar_lm(theta): against the stored mpmath values at l = 4095
    and 8191 (tests/golden/plm_mpmath.txt) wherever the value is representable in binary64.  Seeds: sin(1)^2000 ~
    1e-150, sin(0.08)^300 ~ 1e-330, sin(1)^4000 ~ 1e-300, sin(1.2)^8000 ~ 1e-245, sin(0.02)^100 ~ 1e-170."""
    a = 1.3 - 0.4j
    n = 0
    for l, m, th, frac, ex in _golden():
        if l < 4095 or ex < -1000:
            continue
        am = np.zeros(l - m + 1, dtype=np.complex128)
        am[-1] = a
        ref = a * frac * 2.0 ** ex
        for prec, eps in (("d", 2.0 ** -53), ("ld", 2.0 ** -64)):
            F = oracle.ring_sum(l, m, np.array([th]), am, prec)[0]
            tol = eps * (2000.0 + 8.0 * l / max(np.sin(th), 1e-3)) + 2.0 ** -52
            assert abs(F - ref) <= tol * abs(ref), (l, m, th, prec, F, ref)
        n += 1
    assert n >= 8


# ---- gradient of the lensing potential (Eq. C2) --------------------------------------------------
def _grad_closed_form(l, m, a, th, ph):
    """(d/dtheta, (1/sin theta) d/dphi) of w_m Re(a Y_lm), from the textbook table of Y_lm for l <= 2."""
    s, c = np.sin(th), np.cos(th)
    e = np.exp(1j * m * ph)
    dtab = {     # (P(theta), dP/dtheta) with Y_lm = P e^{i m phi}
        (1, 0): (np.sqrt(3 / (4 * np.pi)) * c, -np.sqrt(3 / (4 * np.pi)) * s),
        (1, 1): (-np.sqrt(3 / (8 * np.pi)) * s, -np.sqrt(3 / (8 * np.pi)) * c),
        (2, 0): (np.sqrt(5 / (16 * np.pi)) * (3 * c * c - 1), -np.sqrt(5 / (16 * np.pi)) * 6 * c * s),
        (2, 1): (-np.sqrt(15 / (8 * np.pi)) * s * c, -np.sqrt(15 / (8 * np.pi)) * (c * c - s * s)),
        (2, 2): (np.sqrt(15 / (32 * np.pi)) * s * s, np.sqrt(15 / (32 * np.pi)) * 2 * s * c),
    }
    P, dP = dtab[(l, m)]
    wm = 1.0 if m == 0 else 2.0
    return wm * np.real(a * dP * e), wm * np.real(a * 1j * m * P * e) / s


@pytest.mark.parametrize("l,m", [(1, 0), (1, 1), (2, 0), (2, 1), (2, 2)])
@pytest.mark.parametrize("prec", ["d", "ld"])
def test_gradient_closed_forms(oracle, l, m, prec):
    rng = np.random.default_rng(40 + l * 3 + m)
    th = np.arccos(rng.uniform(-0.999, 0.999, 300))
    ph = rng.uniform(0, 2 * np.pi, 300)
    a = 0.7 - 1.3j if m > 0 else 0.7 + 0j
    gt, gp = oracle.gradient(5, 4, th, ph, single_alm(5, 4, l, m, a), prec)
    rt, rp = _grad_closed_form(l, m, a, th, ph)
    assert np.max(np.abs(gt - rt)) < 5e-15 and np.max(np.abs((gp - rp) * np.sin(th))) < 5e-15


def test_gradient_vs_finite_differences_of_synthesis(oracle):
    """alpha_theta = dPhi/dtheta and alpha_phi = (1/sin theta) dPhi/dphi against 5-point central differences (h = 1e-4:
    truncation ~ h^4 l^5 / 30, round-off ~ 1e-16 / h) of the oracle's synthesis, itself pinned above."""
    lmax, mmax = 40, 33
    a = inputs.random_alm(lmax, mmax, 44)
    rng = np.random.default_rng(45)
    th = np.arccos(rng.uniform(-0.98, 0.98, 400))
    ph = rng.uniform(0.1, 6.1, 400)
    h = 1e-4

    def d5(f):
        return (f(-2 * h) - 8 * f(-h) + 8 * f(h) - f(2 * h)) / (12 * h)
    dt = d5(lambda e: oracle.synthesis(lmax, mmax, th + e, ph, a, "ld"))
    dph = d5(lambda e: oracle.synthesis(lmax, mmax, th, ph + e, a, "ld")) / np.sin(th)
    gt, gp = oracle.gradient(lmax, mmax, th, ph, a, "ld")
    scale = np.sqrt(np.mean(gt ** 2))
    assert np.max(np.abs(gt - dt)) < 2e-8 * scale
    assert np.max(np.abs((gp - dph) * np.sin(th))) < 2e-8 * scale


@pytest.mark.parametrize("prec", ["d", "ld"])
def test_gradient_rescaling_regime_vs_coefficient_identity(oracle, prec):
    """lmax = 1500 with near-pole points: sin^m theta underflows and the gradient's copy of the l loop goes through
    its own exponent refresh.  Pin: the ladder identity sin(theta) dPbar_lm/dtheta = l c_{l+1} Pbar_{l+1,m} -
    (l+1) c_l Pbar_{l-1,m}, c_l^2 = (l^2 - m^2)/(4 l^2 - 1) (a DIFFERENT relation from the one the oracle sums), turns
    sin(theta) dPhi/dtheta into a plain synthesis at band limit lmax + 1, evaluated by oracle.synthesis (pinned to
    mpmath in this regime above); likewise dPhi/dphi is the synthesis of i m Phi_lm."""
    L = M = 1500
    th, ph = _near_pole_points(60, 46)
    phl = inputs.random_alm(L, M, 46, "inv_l2")
    gt, gp = oracle.gradient(L, M, th, ph, phl, prec)
    L1 = L + 1
    a1 = np.zeros(inputs.nlm(L1, M), dtype=np.complex128)
    b1 = np.zeros(inputs.nlm(L1, M), dtype=np.complex128)
    for m in range(M + 1):
        l = np.arange(m, L + 1, dtype=np.float64)
        p = phl[inputs.lm_index(L, m, m): inputs.lm_index(L, m, m) + L - m + 1]
        c = lambda ll: np.sqrt((ll * ll - m * m) / (4 * ll * ll - 1))        # noqa: E731
        o1 = inputs.lm_index(L1, m, m)
        # Phi_lm contributes l c_{l+1} to l' = l + 1 and -(l + 1) c_l to l' = l - 1
        a1[o1 + 1: o1 + 1 + len(l)] += l * c(l + 1) * p
        a1[o1: o1 + len(l) - 1] += (-(l + 1) * c(l) * p)[1:]
        b1[o1: o1 + len(l)] = 1j * m * p
    if True:
        a1[: L1 + 1] = a1[: L1 + 1].real
    st = oracle.synthesis(L1, M, th, ph, a1, prec)
    sp = oracle.synthesis(L1, M, th, ph, b1, prec)
    scale = np.sqrt(np.mean(st ** 2))
    tol = 2e-11 if prec == "d" else 2e-13
    assert np.max(np.abs(gt * np.sin(th) - st)) <= tol * scale
    assert np.max(np.abs(gp * np.sin(th) - sp)) <= tol * scale
