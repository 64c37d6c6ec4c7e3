"""CPU-only checks of the boundary: the C-ABI library loads and exports every symbol that
include/nusht.h declares; plan-argument validation that needs no device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2406_14542_b200 import build
    return ctypes.CDLL(build.build())


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "nusht.h")).read()
    return sorted(set(re.findall(r"NUSHT_API\s+[\w\s\*]+?\b(nusht_\w+)\s*\(", src)))


def test_header_declares_the_four_north_star_calls():
    syms = declared_symbols()
    for s in ("nusht_plan", "nusht_synthesis", "nusht_adjoint", "nusht_destroy"):
        assert s in syms


def test_library_exports_every_declared_symbol(lib):
    syms = declared_symbols()
    assert len(syms) >= 15
    for s in syms:
        assert hasattr(lib, s), s


def test_binding_lists_same_symbols():
    from paper_2406_14542_b200 import nusht
    assert sorted(nusht.EXPORTS) == declared_symbols()


def test_strerror_and_version(lib):
    lib.nusht_strerror.restype = ctypes.c_char_p
    lib.nusht_version.restype = ctypes.c_char_p
    assert lib.nusht_strerror(0) == b"ok"
    assert b"invalid" in lib.nusht_strerror(-1)
    assert b"sm_100a" in lib.nusht_version()


def test_plan_rejects_bad_arguments_without_device(lib):
    lib.nusht_plan.argtypes = [ctypes.POINTER(ctypes.c_void_p), ctypes.c_int, ctypes.c_int, ctypes.c_int64,
                               ctypes.c_void_p, ctypes.c_void_p, ctypes.c_double, ctypes.c_int]
    h = ctypes.c_void_p()
    assert lib.nusht_plan(ctypes.byref(h), -1, 0, 0, None, None, 1e-6, 0) == -1     # lmax < 0
    assert lib.nusht_plan(ctypes.byref(h), 4, 5, 0, None, None, 1e-6, 0) == -1      # mmax > lmax
    assert lib.nusht_plan(ctypes.byref(h), 4, 4, 0, None, None, 1e-15, 0) == -1     # eps too small
    assert lib.nusht_plan(ctypes.byref(h), 4, 4, 0, None, None, 1e-8, 1) == -1      # eps too small for F32
    assert lib.nusht_plan(ctypes.byref(h), 4, 4, 0, None, None, 1e-6, 7) == -1      # dtype
    assert lib.nusht_plan(ctypes.byref(h), 4, 4, 10, None, None, 1e-6, 0) == -1     # NULL points
    assert lib.nusht_plan(None, 4, 4, 0, None, None, 1e-6, 0) == -1
    assert h.value is None


def test_no_device_is_a_loud_error(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    lib.nusht_plan.argtypes = [ctypes.POINTER(ctypes.c_void_p), ctypes.c_int, ctypes.c_int, ctypes.c_int64,
                               ctypes.c_void_p, ctypes.c_void_p, ctypes.c_double, ctypes.c_int]
    h = ctypes.c_void_p()
    assert lib.nusht_plan(ctypes.byref(h), 4, 4, 0, None, None, 1e-6, 0) == -3      # NUSHT_ERR_CUDA, no fallback
    assert lib.nusht_destroy(None) == 0


def test_plan_ex_rejects_bad_options_without_device(lib):
    class Opts(ctypes.Structure):
        _fields_ = [("sigma", ctypes.c_double), ("reserved", ctypes.c_int * 6)]
    lib.nusht_plan_ex.argtypes = [ctypes.POINTER(ctypes.c_void_p), ctypes.c_int, ctypes.c_int, ctypes.c_int64,
                                  ctypes.c_void_p, ctypes.c_void_p, ctypes.c_double, ctypes.c_int, ctypes.POINTER(Opts)]
    h = ctypes.c_void_p()
    o = Opts()
    o.sigma = 1.5
    assert lib.nusht_plan_ex(ctypes.byref(h), 4, 4, 0, None, None, 1e-6, 0, ctypes.byref(o)) == -1     # unsupported sigma
    o.sigma = 1.25
    assert lib.nusht_plan_ex(ctypes.byref(h), 4, 4, 0, None, None, 1e-11, 0, ctypes.byref(o)) == -1    # below the 1e-10 floor
    o.reserved[2] = 7
    assert lib.nusht_plan_ex(ctypes.byref(h), 4, 4, 0, None, None, 1e-6, 0, ctypes.byref(o)) == -1     # reserved must be zero
    assert h.value is None


def test_ring_plan_rejects_bad_arguments_without_device(lib):
    dp, lp = ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int64)
    lib.nusht_ring_plan.argtypes = [ctypes.POINTER(ctypes.c_void_p), ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, lp, dp,
                                    dp, ctypes.c_int]
    h = ctypes.c_void_p()
    th = (ctypes.c_double * 2)(0.5, 4.0)
    n = (ctypes.c_int64 * 2)(8, 8)
    assert lib.nusht_ring_plan(ctypes.byref(h), 4, 4, 2, th, n, None, None, 0) == -6       # theta outside [0, pi]
    th[1] = 2.0
    n[1] = 0
    assert lib.nusht_ring_plan(ctypes.byref(h), 4, 4, 2, th, n, None, None, 0) == -1       # empty ring
    n[1] = 8
    assert lib.nusht_ring_plan(ctypes.byref(h), 4, 5, 2, th, n, None, None, 0) == -1       # mmax > lmax
    assert lib.nusht_ring_plan(ctypes.byref(h), 4, 4, 0, th, n, None, None, 0) == -1       # no rings
    assert h.value is None
    assert lib.nusht_ring_destroy(None) == 0


def test_round2_entry_points_reject_null_plans_without_device(lib):
    vp = ctypes.c_void_p
    lib.nusht_set_points.argtypes = [vp, ctypes.c_int64, vp, vp]
    lib.nusht_stage_legendre_adjoint_static.argtypes = [vp, vp, vp, vp]
    lib.nusht_static_scratch.argtypes = [ctypes.POINTER(ctypes.c_int64)]
    lib.nusht_strerror.restype = ctypes.c_char_p
    assert lib.nusht_set_points(None, 0, None, None) == -1
    assert lib.nusht_stage_legendre_adjoint_static(None, None, None, None) == -1
    assert b"static scratch" in lib.nusht_strerror(-7)          # NUSHT_ERR_TOO_LARGE names the entry point and the limit
    import torch
    if not torch.cuda.is_available():
        n = ctypes.c_int64(-1)
        assert lib.nusht_static_scratch(ctypes.byref(n)) == -3   # NUSHT_ERR_CUDA: the array lives on a device
