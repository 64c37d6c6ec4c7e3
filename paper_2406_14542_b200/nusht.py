"""Thin ctypes binding of libnusht.so (include/nusht.h): same names, argument marshalling only.

Every step of the transform runs in the CUDA library; torch is used for device memory and streams.
There is no CPU fallback: if the library has not been built, importing this module raises.
"""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libnusht.so")

NUSHT_F64, NUSHT_F32 = 0, 1
NUSHT_OK = 0
NUM_STAGES = 7
SYN_STAGES = ["alm_prep", "legendre", "fft_theta", "deconv_pad", "fft_fine_theta", "fft_fine_phi", "interp"]
ADJ_STAGES = ["spread", "fft_fine_phi", "fft_fine_theta", "deconv_trunc", "fft_theta", "legendre", "alm_post"]
EXPORTS = [
    "nusht_plan", "nusht_synthesis", "nusht_adjoint", "nusht_destroy", "nusht_synthesis_host",
    "nusht_adjoint_host", "nusht_host_sync", "nusht_stage_legendre_synthesis", "nusht_stage_legendre_adjoint",
    "nusht_stage_interp", "nusht_stage_spread", "nusht_set_stage_timing", "nusht_stage_times",
    "nusht_plan_info", "nusht_strerror", "nusht_version", "nusht_pointing", "nusht_host_reserve",
    "nusht_stage_fourier_synthesis", "nusht_stage_fourier_adjoint", "nusht_launch_count", "nusht_probe_fp64",
    "nusht_ring_plan", "nusht_ring_synthesis", "nusht_ring_analysis", "nusht_ring_gradient", "nusht_ring_info",
    "nusht_ring_destroy", "nusht_ring_pairing", "nusht_plan_ex", "nusht_static_scratch",
    "nusht_stage_legendre_adjoint_static", "nusht_set_points",
]


class NushtInfo(ctypes.Structure):
    _fields_ = [
        ("lmax", ctypes.c_int), ("mmax", ctypes.c_int), ("dtype", ctypes.c_int),
        ("npts", ctypes.c_int64), ("nlm", ctypes.c_int64), ("eps", ctypes.c_double),
        ("n_rings", ctypes.c_int), ("n_theta", ctypes.c_int), ("n_theta_fine", ctypes.c_int),
        ("n_phi_fine", ctypes.c_int), ("kernel_width", ctypes.c_int), ("kernel_degree", ctypes.c_int),
        ("kernel_beta", ctypes.c_double), ("sigma", ctypes.c_double),
        ("workspace_bytes", ctypes.c_int64), ("plan_ms", ctypes.c_double), ("sort_ms", ctypes.c_double),
        ("legendre_fma_synthesis", ctypes.c_int64), ("legendre_fma_adjoint", ctypes.c_int64),
        ("set_points_ms", ctypes.c_double),
    ]


class NushtRingInfo(ctypes.Structure):
    _fields_ = [
        ("lmax", ctypes.c_int), ("mmax", ctypes.c_int), ("dtype", ctypes.c_int), ("nrings", ctypes.c_int),
        ("npairs", ctypes.c_int), ("nruns", ctypes.c_int),
        ("npix", ctypes.c_int64), ("nlm", ctypes.c_int64), ("workspace_bytes", ctypes.c_int64),
        ("plan_ms", ctypes.c_double),
    ]


class NushtOpts(ctypes.Structure):
    _fields_ = [("sigma", ctypes.c_double), ("reserved", ctypes.c_int * 6)]


class NushtError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("nusht error %d: %s" % (code, msg))
        self.code = code


def _load():
    if not os.path.exists(_LIBPATH):
        raise ImportError(
            "libnusht.so is not built (run `python -m paper_2406_14542_b200.build`); there is no CPU fallback")
    lib = ctypes.CDLL(_LIBPATH)
    vp, ip = ctypes.c_void_p, ctypes.c_int
    lib.nusht_plan.argtypes = [ctypes.POINTER(vp), ip, ip, ctypes.c_int64, vp, vp, ctypes.c_double, ip]
    for name in ("nusht_synthesis", "nusht_adjoint", "nusht_synthesis_host", "nusht_adjoint_host",
                 "nusht_stage_legendre_synthesis", "nusht_stage_legendre_adjoint", "nusht_stage_interp",
                 "nusht_stage_spread", "nusht_stage_fourier_synthesis", "nusht_stage_fourier_adjoint",
                 "nusht_stage_legendre_adjoint_static"):
        getattr(lib, name).argtypes = [vp, vp, vp, vp]
        getattr(lib, name).restype = ip
    lib.nusht_plan.restype = ip
    lib.nusht_plan_ex.argtypes = [ctypes.POINTER(vp), ip, ip, ctypes.c_int64, vp, vp, ctypes.c_double, ip,
                                  ctypes.POINTER(NushtOpts)]
    lib.nusht_plan_ex.restype = ip
    lib.nusht_destroy.argtypes = [vp]
    lib.nusht_destroy.restype = ip
    lib.nusht_host_sync.argtypes = [vp]
    lib.nusht_host_sync.restype = ip
    lib.nusht_host_reserve.argtypes = [vp]
    lib.nusht_host_reserve.restype = ip
    lib.nusht_set_points.argtypes = [vp, ctypes.c_int64, vp, vp]
    lib.nusht_set_points.restype = ip
    lib.nusht_static_scratch.argtypes = [ctypes.POINTER(ctypes.c_int64)]
    lib.nusht_static_scratch.restype = ip
    lib.nusht_launch_count.argtypes = []
    lib.nusht_launch_count.restype = ctypes.c_int64
    lib.nusht_probe_fp64.argtypes = [ip, ctypes.POINTER(ctypes.c_double)]
    lib.nusht_probe_fp64.restype = ip
    lib.nusht_set_stage_timing.argtypes = [vp, ip]
    lib.nusht_set_stage_timing.restype = ip
    lib.nusht_stage_times.argtypes = [vp, ip, ctypes.POINTER(ctypes.c_float), ip]
    lib.nusht_stage_times.restype = ip
    lib.nusht_plan_info.argtypes = [vp, ctypes.POINTER(NushtInfo)]
    lib.nusht_plan_info.restype = ip
    lib.nusht_pointing.argtypes = [ctypes.c_int64, vp, vp, vp, vp, vp, vp, vp]
    lib.nusht_pointing.restype = ip
    dp, lp = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int64)
    lib.nusht_ring_plan.argtypes = [ctypes.POINTER(vp), ip, ip, ip, dp, lp, dp, dp, ip]
    lib.nusht_ring_plan.restype = ip
    for name in ("nusht_ring_synthesis", "nusht_ring_analysis"):
        getattr(lib, name).argtypes = [vp, vp, vp, vp]
        getattr(lib, name).restype = ip
    lib.nusht_ring_gradient.argtypes = [vp, vp, vp, vp, vp]
    lib.nusht_ring_gradient.restype = ip
    lib.nusht_ring_info.argtypes = [vp, ctypes.POINTER(NushtRingInfo)]
    lib.nusht_ring_info.restype = ip
    lib.nusht_ring_destroy.argtypes = [vp]
    lib.nusht_ring_destroy.restype = ip
    lib.nusht_ring_pairing.argtypes = [ip, dp, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int)]
    lib.nusht_ring_pairing.restype = ip
    lib.nusht_strerror.argtypes = [ip]
    lib.nusht_strerror.restype = ctypes.c_char_p
    lib.nusht_version.restype = ctypes.c_char_p
    return lib


lib = _load()


def _check(code):
    if code != NUSHT_OK:
        raise NushtError(code, lib.nusht_strerror(code).decode())


def version() -> str:
    return lib.nusht_version().decode()


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


class Plan:
    """nusht_plan(lmax, mmax, npts, theta, phi, eps, dtype): theta/phi are CUDA float64 tensors.
    sigma (nusht_plan_ex): up-sampling factor of the nuFFT grid, 2 (default) or 1.25."""

    def __init__(self, lmax, mmax, theta, phi, eps, dtype="f64", sigma=None):
        self._h = ctypes.c_void_p()
        if dtype in ("f64", NUSHT_F64):
            self.dtype = NUSHT_F64
        elif dtype in ("f32", NUSHT_F32):
            self.dtype = NUSHT_F32
        else:
            raise ValueError("dtype must be 'f64' or 'f32'")
        npts = 0 if theta is None else int(theta.numel())
        if npts:
            if phi is None or int(phi.numel()) != npts:
                raise ValueError("theta and phi must have the same number of entries")
            if not (theta.is_cuda and phi.is_cuda and theta.dtype == torch.float64 and phi.dtype == torch.float64):
                raise TypeError("theta/phi must be CUDA float64 tensors")
            theta, phi = theta.contiguous(), phi.contiguous()
            tp, pp = theta.data_ptr(), phi.data_ptr()
        else:
            tp = pp = None
        if sigma is None:
            _check(lib.nusht_plan(ctypes.byref(self._h), int(lmax), int(mmax), npts, tp, pp, float(eps), self.dtype))
        else:
            opts = NushtOpts()
            opts.sigma = float(sigma)
            _check(lib.nusht_plan_ex(ctypes.byref(self._h), int(lmax), int(mmax), npts, tp, pp, float(eps), self.dtype,
                                     ctypes.byref(opts)))
        self.info = NushtInfo()
        _check(lib.nusht_plan_info(self._h, ctypes.byref(self.info)))
        self.lmax, self.mmax, self.npts, self.nlm = int(lmax), int(mmax), npts, int(self.info.nlm)
        self.rdtype = torch.float64 if self.dtype == NUSHT_F64 else torch.float32
        self.cdtype = torch.complex128 if self.dtype == NUSHT_F64 else torch.complex64

    def set_points(self, theta, phi):
        """nusht_set_points: a new point set for the same (lmax, mmax, eps, dtype, sigma); only the point sort runs."""
        npts = 0 if theta is None else int(theta.numel())
        if npts:
            if phi is None or int(phi.numel()) != npts:
                raise ValueError("theta and phi must have the same number of entries")
            if not (theta.is_cuda and phi.is_cuda and theta.dtype == torch.float64 and phi.dtype == torch.float64):
                raise TypeError("theta/phi must be CUDA float64 tensors")
            theta, phi = theta.contiguous(), phi.contiguous()
            tp, pp = theta.data_ptr(), phi.data_ptr()
        else:
            tp = pp = None
        code = lib.nusht_set_points(self._h, npts, tp, pp)
        _check(lib.nusht_plan_info(self._h, ctypes.byref(self.info)))
        self.npts = int(self.info.npts)
        _check(code)

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib.nusht_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # ---- marshalling helpers ----
    def _alm_arg(self, alm, device=True):
        if alm.dtype != self.cdtype or alm.numel() != self.nlm or alm.is_cuda != device or not alm.is_contiguous():
            raise TypeError("alm must be a contiguous %s tensor of %d entries on %s"
                            % (self.cdtype, self.nlm, "cuda" if device else "cpu"))
        return alm.data_ptr()

    def _map_arg(self, m, device=True):
        if m.dtype != self.rdtype or m.numel() != self.npts or m.is_cuda != device or not m.is_contiguous():
            raise TypeError("map must be a contiguous %s tensor of %d entries on %s"
                            % (self.rdtype, self.npts, "cuda" if device else "cpu"))
        return m.data_ptr() if self.npts else None

    # ---- transforms ----
    def synthesis(self, alm, out=None, stream=None):
        if out is None:
            out = torch.empty(self.npts, dtype=self.rdtype, device=alm.device)
        _check(lib.nusht_synthesis(self._h, self._alm_arg(alm), self._map_arg(out), _stream_ptr(stream)))
        return out

    def adjoint(self, x, out=None, stream=None):
        if out is None:
            out = torch.empty(self.nlm, dtype=self.cdtype, device="cuda")
        _check(lib.nusht_adjoint(self._h, self._map_arg(x), self._alm_arg(out), _stream_ptr(stream)))
        return out

    def synthesis_host(self, alm_host, out_host, stream=None):
        _check(lib.nusht_synthesis_host(self._h, self._alm_arg(alm_host, False), self._map_arg(out_host, False),
                                        _stream_ptr(stream)))
        return out_host

    def adjoint_host(self, x_host, out_host, stream=None):
        _check(lib.nusht_adjoint_host(self._h, self._map_arg(x_host, False), self._alm_arg(out_host, False),
                                      _stream_ptr(stream)))
        return out_host

    def host_reserve(self):
        """Allocate the staging buffers of the host-buffer calls now (nusht_host_reserve)."""
        _check(lib.nusht_host_reserve(self._h))

    def host_sync(self):
        """Wait until every host-buffer transform issued so far has delivered its output."""
        _check(lib.nusht_host_sync(self._h))

    # ---- stages ----
    def stage_legendre_synthesis(self, alm, stream=None):
        out = torch.empty((self.mmax + 1, self.info.n_theta), dtype=torch.complex128, device="cuda")
        _check(lib.nusht_stage_legendre_synthesis(self._h, self._alm_arg(alm), out.data_ptr(), _stream_ptr(stream)))
        return out

    def stage_legendre_adjoint(self, gt, stream=None):
        if gt.dtype != torch.complex128 or tuple(gt.shape) != (self.mmax + 1, self.info.n_theta) or not gt.is_cuda:
            raise TypeError("gtilde must be CUDA complex128 [(mmax+1), n_theta]")
        out = torch.empty(self.nlm, dtype=self.cdtype, device="cuda")
        _check(lib.nusht_stage_legendre_adjoint(self._h, gt.contiguous().data_ptr(), out.data_ptr(),
                                                _stream_ptr(stream)))
        return out

    def stage_legendre_adjoint_static(self, gt, out, stream=None):
        """nusht_stage_legendre_adjoint_static: the same result through the library's static scratch array; the C
        call allocates nothing (hence `out` is the caller's).  Plans up to lmax = mmax = 1023; calls that overlap
        on the GPU race on the one array (include/nusht.h)."""
        if gt.dtype != torch.complex128 or tuple(gt.shape) != (self.mmax + 1, self.info.n_theta) or not gt.is_cuda \
                or not gt.is_contiguous():
            raise TypeError("gtilde must be contiguous CUDA complex128 [(mmax+1), n_theta]")
        if out.dtype != self.cdtype or tuple(out.shape) != (self.nlm,) or not out.is_cuda or not out.is_contiguous():
            raise TypeError("out must be contiguous CUDA %s [nlm]" % self.cdtype)
        _check(lib.nusht_stage_legendre_adjoint_static(self._h, gt.data_ptr(), out.data_ptr(), _stream_ptr(stream)))
        return out

    def grid_shape(self):
        return (self.info.n_theta_fine // 2 + 1, self.info.n_phi_fine)

    def stage_fourier_synthesis(self, ft, stream=None):
        if ft.dtype != torch.complex128 or tuple(ft.shape) != (self.mmax + 1, self.info.n_theta) or not ft.is_cuda:
            raise TypeError("ftilde must be CUDA complex128 [(mmax+1), n_theta]")
        out = torch.empty(self.grid_shape(), dtype=self.rdtype, device="cuda")
        _check(lib.nusht_stage_fourier_synthesis(self._h, ft.contiguous().data_ptr(), out.data_ptr(),
                                                 _stream_ptr(stream)))
        return out

    def stage_fourier_adjoint(self, grid, stream=None):
        if grid.dtype != self.rdtype or tuple(grid.shape) != self.grid_shape() or not grid.is_cuda:
            raise TypeError("grid must be CUDA %s %s" % (self.rdtype, self.grid_shape()))
        out = torch.empty((self.mmax + 1, self.info.n_theta), dtype=torch.complex128, device="cuda")
        _check(lib.nusht_stage_fourier_adjoint(self._h, grid.contiguous().data_ptr(), out.data_ptr(),
                                               _stream_ptr(stream)))
        return out

    def stage_interp(self, grid, stream=None):
        if grid.dtype != self.rdtype or tuple(grid.shape) != self.grid_shape() or not grid.is_cuda:
            raise TypeError("grid must be CUDA %s %s" % (self.rdtype, self.grid_shape()))
        out = torch.empty(self.npts, dtype=self.rdtype, device="cuda")
        _check(lib.nusht_stage_interp(self._h, grid.contiguous().data_ptr(), self._map_arg(out), _stream_ptr(stream)))
        return out

    def stage_spread(self, x, stream=None):
        out = torch.empty(self.grid_shape(), dtype=self.rdtype, device="cuda")
        _check(lib.nusht_stage_spread(self._h, self._map_arg(x), out.data_ptr(), _stream_ptr(stream)))
        return out

    # ---- timing ----
    def set_stage_timing(self, enable=True):
        _check(lib.nusht_set_stage_timing(self._h, 1 if enable else 0))

    def stage_times(self, which):
        buf = (ctypes.c_float * NUM_STAGES)()
        _check(lib.nusht_stage_times(self._h, 0 if which in (0, "synthesis") else 1, buf, NUM_STAGES))
        names = SYN_STAGES if which in (0, "synthesis") else ADJ_STAGES
        return {n: float(buf[i]) for i, n in enumerate(names)}


class RingPlan:
    """nusht_ring_plan(lmax, mmax, nrings, theta, nphi, phi0, weight, dtype): transforms on a ring grid.  theta, nphi,
    phi0, weight are HOST sequences (numpy arrays / lists) of one entry per ring; maps are CUDA tensors of npix reals."""

    def __init__(self, lmax, mmax, theta, nphi, phi0=None, weight=None, dtype="f64"):
        import numpy as np
        self._h = ctypes.c_void_p()
        if dtype in ("f64", NUSHT_F64):
            self.dtype = NUSHT_F64
        elif dtype in ("f32", NUSHT_F32):
            self.dtype = NUSHT_F32
        else:
            raise ValueError("dtype must be 'f64' or 'f32'")
        th = np.ascontiguousarray(theta, dtype=np.float64)
        n = np.ascontiguousarray(nphi, dtype=np.int64)
        if th.ndim != 1 or n.shape != th.shape:
            raise ValueError("theta and nphi must be 1-D with one entry per ring")
        dp, lp = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int64)

        def opt(a):
            if a is None:
                return None, None
            a = np.ascontiguousarray(a, dtype=np.float64)
            if a.shape != th.shape:
                raise ValueError("phi0 / weight must have one entry per ring")
            return a, a.ctypes.data_as(dp)
        p0, p0p = opt(phi0)
        w, wp = opt(weight)
        _check(lib.nusht_ring_plan(ctypes.byref(self._h), int(lmax), int(mmax), int(th.shape[0]), th.ctypes.data_as(dp),
                                   n.ctypes.data_as(lp), p0p, wp, self.dtype))
        self.info = NushtRingInfo()
        _check(lib.nusht_ring_info(self._h, ctypes.byref(self.info)))
        self.lmax, self.mmax, self.npix, self.nlm = int(lmax), int(mmax), int(self.info.npix), int(self.info.nlm)
        self.rdtype = torch.float64 if self.dtype == NUSHT_F64 else torch.float32
        self.cdtype = torch.complex128 if self.dtype == NUSHT_F64 else torch.complex64

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib.nusht_ring_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def _alm_arg(self, alm):
        if alm.dtype != self.cdtype or alm.numel() != self.nlm or not alm.is_cuda or not alm.is_contiguous():
            raise TypeError("alm must be a contiguous CUDA %s tensor of %d entries" % (self.cdtype, self.nlm))
        return alm.data_ptr()

    def _map_arg(self, m):
        if m.dtype != self.rdtype or m.numel() != self.npix or not m.is_cuda or not m.is_contiguous():
            raise TypeError("map must be a contiguous CUDA %s tensor of %d entries" % (self.rdtype, self.npix))
        return m.data_ptr()

    def synthesis(self, alm, out=None, stream=None):
        if out is None:
            out = torch.empty(self.npix, dtype=self.rdtype, device="cuda")
        _check(lib.nusht_ring_synthesis(self._h, self._alm_arg(alm), self._map_arg(out), _stream_ptr(stream)))
        return out

    def analysis(self, m, out=None, stream=None):
        if out is None:
            out = torch.empty(self.nlm, dtype=self.cdtype, device="cuda")
        _check(lib.nusht_ring_analysis(self._h, self._map_arg(m), self._alm_arg(out), _stream_ptr(stream)))
        return out

    def gradient(self, philm, stream=None):
        a_t = torch.empty(self.npix, dtype=self.rdtype, device="cuda")
        a_p = torch.empty(self.npix, dtype=self.rdtype, device="cuda")
        _check(lib.nusht_ring_gradient(self._h, self._alm_arg(philm), a_t.data_ptr(), a_p.data_ptr(),
                                       _stream_ptr(stream)))
        return a_t, a_p


def ring_pairing(theta):
    """Pairs of mirror rings as the ring plan forms them (nusht_ring_pairing; host only): list of (north, south | -1)."""
    import numpy as np
    th = np.ascontiguousarray(theta, dtype=np.float64)
    pn = np.empty(len(th), dtype=np.int32)
    ps = np.empty(len(th), dtype=np.int32)
    ip = ctypes.POINTER(ctypes.c_int)
    n = lib.nusht_ring_pairing(len(th), th.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), pn.ctypes.data_as(ip),
                               ps.ctypes.data_as(ip))
    if n < 0:
        _check(n)
    return [(int(pn[j]), int(ps[j])) for j in range(n)]


def launch_count() -> int:
    """Kernels of this library launched so far in this process (nusht_launch_count)."""
    return int(lib.nusht_launch_count())


def static_scratch() -> int:
    """Resolve the static scratch array of nusht_stage_legendre_adjoint_static on the current device (set-up step,
    outside graph capture) and return its capacity in bytes (nusht_static_scratch)."""
    v = ctypes.c_int64()
    _check(lib.nusht_static_scratch(ctypes.byref(v)))
    return int(v.value)


def probe_fp64(kind: str) -> float:
    """Measured FP64 throughput of the current device in TFLOP/s: kind 'dfma' or 'dmma' (nusht_probe_fp64)."""
    v = ctypes.c_double()
    _check(lib.nusht_probe_fp64({"dfma": 0, "dmma": 1}[kind], ctypes.byref(v)))
    return float(v.value)


def nusht_plan(lmax, mmax, npts, theta, phi, eps, dtype="f64"):
    assert npts == (0 if theta is None else theta.numel())
    return Plan(lmax, mmax, theta, phi, eps, dtype)


def nusht_synthesis(plan, alm, map_out=None, stream=None):
    return plan.synthesis(alm, map_out, stream)


def nusht_adjoint(plan, x, alm_out=None, stream=None):
    return plan.adjoint(x, alm_out, stream)


def nusht_destroy(plan):
    plan.destroy()


def nusht_pointing(theta, phi, alpha_theta, alpha_phi, stream=None):
    """Eq. C1: deflected positions (theta', phi') of CUDA float64 points; argument marshalling
    only, the arithmetic is k_pointing (csrc/pointing.cu)."""
    n = theta.numel()
    for a in (theta, phi, alpha_theta, alpha_phi):
        if not a.is_cuda or a.dtype != torch.float64 or a.numel() != n or not a.is_contiguous():
            raise TypeError("theta, phi, alpha_theta, alpha_phi must be contiguous CUDA float64 of one length")
    t2, p2 = torch.empty_like(theta), torch.empty_like(phi)
    _check(lib.nusht_pointing(n, theta.data_ptr(), phi.data_ptr(), alpha_theta.data_ptr(), alpha_phi.data_ptr(),
                              t2.data_ptr(), p2.data_ptr(), _stream_ptr(stream)))
    return t2, p2
