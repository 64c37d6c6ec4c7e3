"""ctypes loader for the CPU oracle (oracle/nusht_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py.  Nothing under paper_2406_14542_b200/
imports this module, and this module imports nothing from there.

The functions are the plain definitions of arXiv 2406.14542 Eq. 3 (synthesis)
and Eq. 2 (adjoint); see the C source for the step-by-step statement.
`precision="ld"` selects the x86 80-bit long double instantiation.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(_HERE, "nusht_oracle.c"), os.path.join(_HERE, "nusht_oracle_impl.inc")]
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile liboracle.so with gcc (no -ffast-math) if missing or older than its sources."""
    stale = force or not os.path.exists(_LIB) or any(
        os.path.getmtime(s) > os.path.getmtime(_LIB) for s in _SRC)
    if stale:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC[0], "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        for suf in ("_d", "_ld"):
            f = getattr(_lib, "oracle_plm" + suf)
            f.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_double, dp, ctypes.POINTER(ctypes.c_long)]
            f.restype = None
            f = getattr(_lib, "oracle_ring_sum" + suf)
            f.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_long, dp, dp, dp]
            f.restype = None
            f = getattr(_lib, "oracle_synthesis" + suf)
            f.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_long, dp, dp, dp, dp]
            f.restype = None
            f = getattr(_lib, "oracle_adjoint" + suf)
            f.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_long, dp, dp, dp, dp]
            f.restype = None
            f = getattr(_lib, "oracle_adjoint_columns" + suf)
            f.argtypes = [ctypes.c_int, ctypes.c_int, ip, ctypes.c_long, dp, dp, dp, dp]
            f.restype = None
        for suf in ("_d", "_ld"):
            f = getattr(_lib, "oracle_gradient" + suf)
            f.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_long, dp, dp, dp, dp, dp]
            f.restype = None
        _lib.oracle_num_threads.restype = ctypes.c_int
        _lib.oracle_long_double_bits.restype = ctypes.c_int
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _suf(precision):
    if precision not in ("d", "ld"):
        raise ValueError("precision must be 'd' or 'ld'")
    return "_" + precision


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def long_double_mantissa_bits() -> int:
    return int(_load().oracle_long_double_bits()) % 1000


def nlm(lmax: int, mmax: int) -> int:
    """Number of stored coefficients, m-major triangular layout (G2)."""
    return (mmax + 1) * (lmax + 1) - mmax * (mmax + 1) // 2


def lm_index(lmax: int, l, m):
    """idx(l, m) = m (2 lmax + 1 - m)/2 + l."""
    return m * (2 * lmax + 1 - m) // 2 + l


def plm(l: int, m: int, theta: float, precision: str = "d"):
    """Pbar_lm(theta) = Y_lm(theta, 0) as (mantissa in [0.5,1) with sign, binary exponent)."""
    mant = ctypes.c_double()
    ex = ctypes.c_long()
    getattr(_load(), "oracle_plm" + _suf(precision))(l, m, float(theta), ctypes.byref(mant), ctypes.byref(ex))
    return mant.value, ex.value


def plm_value(l: int, m: int, theta: float, precision: str = "d") -> float:
    mant, ex = plm(l, m, theta, precision)
    return float(np.ldexp(mant, ex))


def ring_sum(lmax: int, m: int, theta, alm_m, precision: str = "d"):
    """F_m(theta_k) = sum_{l=m}^{lmax} a_lm Pbar_lm(theta_k); alm_m complex, l = m..lmax."""
    theta = _f64(theta)
    a = np.ascontiguousarray(alm_m, dtype=np.complex128)
    if a.shape != (lmax - m + 1,):
        raise ValueError("alm_m must have lmax-m+1 entries")
    out = np.empty(theta.shape[0], dtype=np.complex128)
    getattr(_load(), "oracle_ring_sum" + _suf(precision))(
        lmax, m, theta.shape[0], _dp(theta), _dp(a.view(np.float64)), _dp(out.view(np.float64)))
    return out


def synthesis(lmax: int, mmax: int, theta, phi, alm, precision: str = "d"):
    """Eq. 3: real map values at (theta_j, phi_j) from complex alm (m >= 0, real field)."""
    theta, phi = _f64(theta), _f64(phi)
    a = np.ascontiguousarray(alm, dtype=np.complex128)
    if a.shape != (nlm(lmax, mmax),):
        raise ValueError("alm has wrong length")
    if theta.shape != phi.shape or theta.ndim != 1:
        raise ValueError("theta/phi must be 1-D and equal length")
    out = np.empty(theta.shape[0], dtype=np.float64)
    getattr(_load(), "oracle_synthesis" + _suf(precision))(
        lmax, mmax, theta.shape[0], _dp(theta), _dp(phi), _dp(a.view(np.float64)), _dp(out))
    return out


def adjoint(lmax: int, mmax: int, theta, phi, x, precision: str = "d"):
    """Eq. 2: c_lm = sum_j x_j Pbar_lm(theta_j) e^{-i m phi_j}, all (l, m); Im c_l0 = 0."""
    theta, phi, x = _f64(theta), _f64(phi), _f64(x)
    out = np.zeros(nlm(lmax, mmax), dtype=np.complex128)
    getattr(_load(), "oracle_adjoint" + _suf(precision))(
        lmax, mmax, theta.shape[0], _dp(theta), _dp(phi), _dp(x), _dp(out.view(np.float64)))
    return out


def adjoint_columns(lmax: int, mlist, theta, phi, x, precision: str = "d"):
    """Eq. 2 restricted to the listed m: returns complex array [len(mlist), lmax+1] indexed by l
    (entries l < m are zero)."""
    theta, phi, x = _f64(theta), _f64(phi), _f64(x)
    ml = np.ascontiguousarray(mlist, dtype=np.int32)
    out = np.zeros((ml.shape[0], lmax + 1), dtype=np.complex128)
    getattr(_load(), "oracle_adjoint_columns" + _suf(precision))(
        lmax, ml.shape[0], ml.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), theta.shape[0],
        _dp(theta), _dp(phi), _dp(x), _dp(out.view(np.float64)))
    return out


def gradient(lmax: int, mmax: int, theta, phi, philm, precision: str = "d"):
    """Eq. C2: (alpha_theta, alpha_phi) = (d/dtheta, (1/sin theta) d/dphi) of
    Phi = sum_lm Phi_lm Y_lm at the points, by the direct sum (see the C source).  Points at a pole give NaN / Inf."""
    theta, phi = _f64(theta), _f64(phi)
    a = np.ascontiguousarray(philm, dtype=np.complex128)
    if a.shape != (nlm(lmax, mmax),):
        raise ValueError("philm has wrong length")
    if theta.shape != phi.shape or theta.ndim != 1:
        raise ValueError("theta/phi must be 1-D and equal length")
    a_t = np.empty(theta.shape[0], dtype=np.float64)
    a_p = np.empty(theta.shape[0], dtype=np.float64)
    getattr(_load(), "oracle_gradient" + _suf(precision))(
        lmax, mmax, theta.shape[0], _dp(theta), _dp(phi), _dp(a.view(np.float64)), _dp(a_t), _dp(a_p))
    return a_t, a_p


def inner_alm(lmax: int, mmax: int, a, c) -> float:
    """Real inner product on m >= 0 storage (G3):
    <a, c> = sum_l a_l0 c_l0 + 2 sum_{m>=1} Re(a_lm conj(c_lm)), with Im of m=0 entries ignored."""
    a = np.asarray(a, dtype=np.complex128)
    c = np.asarray(c, dtype=np.complex128)
    n0 = lmax + 1
    s0 = float(np.sum(np.longdouble(a[:n0].real) * np.longdouble(c[:n0].real)))
    prod = np.longdouble(a[n0:].real) * np.longdouble(c[n0:].real) + \
        np.longdouble(a[n0:].imag) * np.longdouble(c[n0:].imag)
    return s0 + 2.0 * float(np.sum(prod))


def pointing(theta, phi, alpha_theta, alpha_phi):
    """Deflected positions of arXiv 2406.14542 Eq. C1, written out in numpy long double:

        n' = cos(a) n + (sin(a)/a) (a_theta e_theta + a_phi e_phi),   a = sqrt(a_theta^2 + a_phi^2),

    with n = (sin t cos p, sin t sin p, cos t) and the right-handed basis e_theta = dn/dtheta =
    (cos t cos p, cos t sin p, -sin t), e_phi = (-sin p, cos p, 0).  Returns the angles of n':
    theta' = atan2(|n'_xy|, n'_z) in [0, pi] (the polar angle, written so that it keeps its accuracy next to the
    poles, where arccos does not) and phi' = atan2(n'_y, n'_x) mod 2 pi; sin(a)/a := 1 at a = 0.
    Pins (tests/test_oracle_pins.py): a = 0 is the identity, a_phi = 0 moves along the meridian by a_theta,
    on the equator a_theta = 0 moves along the equator by a_phi, |n'| = 1 and the angle between n and n' is a,
    and the spherical-triangle cosine rule for theta'."""
    ld = np.longdouble
    t, p = np.asarray(theta, dtype=ld), np.asarray(phi, dtype=ld)
    at, ap = np.asarray(alpha_theta, dtype=ld), np.asarray(alpha_phi, dtype=ld)
    a = np.sqrt(at * at + ap * ap)
    st, ct, sp, cp = np.sin(t), np.cos(t), np.sin(p), np.cos(p)
    n = (st * cp, st * sp, ct)
    e_t = (ct * cp, ct * sp, -st)
    e_p = (-sp, cp, np.zeros_like(sp))
    with np.errstate(invalid="ignore", divide="ignore"):
        sinc = np.where(a > 0, np.sin(a) / np.where(a > 0, a, ld(1)), ld(1))
    ca = np.cos(a)
    nx, ny, nz = (ca * n[k] + sinc * (at * e_t[k] + ap * e_p[k]) for k in range(3))
    two_pi = 2 * np.arctan2(ld(0), ld(-1))
    theta2 = np.arctan2(np.sqrt(nx * nx + ny * ny), nz)
    phi2 = np.arctan2(ny, nx)
    phi2 = np.where(phi2 < 0, phi2 + two_pi, phi2)
    phi2 = np.where(phi2 >= two_pi, phi2 - two_pi, phi2)
    return theta2, phi2
