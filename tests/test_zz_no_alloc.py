"""nusht_stage_legendre_adjoint_static (include/nusht.h): the transpose of the Legendre stage (
PAPER.md:80-86) with its accumulators in the library's file-scope static device array, for callers that may not
allocate.  Checked against nusht_stage_legendre_adjoint, the existing path with the accumulators in the plan's
workspace: the same kernels run, the sums are global floating-point reductions whose order is not fixed, so the two
agree to rounding (the bar is the one test_gpu_parity.py uses for this stage), and call after call must agree too
(the array keeps the previous call's sums: a missing clear would show on the second call).

This file is collected last on purpose (pytest -x: a failure here hides nothing after it)."""
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


def rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def random_gtilde(M, nth2, seed):
    rng = np.random.default_rng(seed)
    return torch.from_numpy(rng.standard_normal((M + 1, nth2)) + 1j * rng.standard_normal((M + 1, nth2))).cuda()


@pytest.mark.parametrize("L,M,dtype", [(255, 200, "f64"), (1023, 1023, "f64"), (63, 63, "f32"), (0, 0, "f64")])
def test_static_scratch_adjoint_matches_the_plan_workspace_path(nusht, L, M, dtype):
    assert nusht.static_scratch() == 8404992                # set-up: resolves the array's address on this device
    plan = nusht.Plan(L, M, None, None, 1e-5 if dtype == "f32" else 1e-10, dtype=dtype)
    nth2 = plan.info.n_theta
    tol = 1e-6 if dtype == "f32" else 2e-12 * max(1.0, L / 100.0)
    before = torch.cuda.memory_allocated()
    for call in range(2):                                    # two calls in a row, different inputs
        gt = random_gtilde(M, nth2, 900 + call)
        ref = plan.stage_legendre_adjoint(gt)
        out = torch.full((plan.nlm,), float("nan"), dtype=plan.cdtype, device="cuda")
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        got = plan.stage_legendre_adjoint_static(gt, out)
        assert got.data_ptr() == out.data_ptr()
        torch.cuda.synchronize()
        if call == 1:                                        # (call 0 may still load kernels lazily)
            assert torch.cuda.mem_get_info()[0] == free_before       # the driver handed out no device memory
        a, b = got.cpu().numpy().astype(np.complex128), ref.cpu().numpy().astype(np.complex128)
        assert np.all(np.isfinite(a.view(np.float64)))
        assert rel(a, b) <= tol, (call, rel(a, b))
        assert np.max(np.abs(a - b)) <= 50 * tol * np.sqrt(np.mean(np.abs(b) ** 2)), call
        assert np.all(a[: L + 1].imag == 0)                  # m = 0 coefficients are real, as on the existing path
        del gt, ref, out, got
    assert torch.cuda.memory_allocated() == before
    plan.destroy()


def test_static_scratch_same_input_twice_and_after_a_larger_plan(nusht):
    """The array is shared by every plan on the device: a small plan after a large one must not see its sums."""
    big = nusht.Plan(700, 700, None, None, 1e-10)
    small = nusht.Plan(40, 17, None, None, 1e-10)
    g_big = random_gtilde(700, big.info.n_theta, 910)
    g_small = random_gtilde(17, small.info.n_theta, 911)
    out_big = torch.empty(big.nlm, dtype=torch.complex128, device="cuda")
    out_small = torch.empty(small.nlm, dtype=torch.complex128, device="cuda")
    big.stage_legendre_adjoint_static(g_big, out_big)
    first = small.stage_legendre_adjoint_static(g_small, out_small).cpu().numpy().copy()
    second = small.stage_legendre_adjoint_static(g_small, out_small).cpu().numpy()
    ref = small.stage_legendre_adjoint(g_small).cpu().numpy()
    assert rel(first, ref) <= 2e-12 and rel(second, ref) <= 2e-12
    assert rel(out_big.cpu().numpy(), big.stage_legendre_adjoint(g_big).cpu().numpy()) <= 2e-12 * 7
    big.destroy()
    small.destroy()


def test_static_scratch_rejects_plans_beyond_its_capacity(nusht):
    plan = nusht.Plan(1024, 1024, None, None, 1e-10)         # 263,169 accumulators > 262,656
    gt = random_gtilde(1024, plan.info.n_theta, 920)
    out = torch.full((plan.nlm,), 7.0 + 0j, dtype=torch.complex128, device="cuda")
    with pytest.raises(nusht.NushtError) as e:
        plan.stage_legendre_adjoint_static(gt, out)
    assert e.value.code == -7 and "static scratch" in str(e.value)
    torch.cuda.synchronize()
    assert bool(torch.all(out == 7.0 + 0j))                  # nothing was enqueued
    plan.destroy()
    plan = nusht.Plan(1100, 500, None, None, 1e-10)          # 213,301 accumulators: fits although lmax > 1023
    gt = random_gtilde(500, plan.info.n_theta, 921)
    out = torch.empty(plan.nlm, dtype=torch.complex128, device="cuda")
    got = plan.stage_legendre_adjoint_static(gt, out).cpu().numpy()
    assert rel(got, plan.stage_legendre_adjoint(gt).cpu().numpy()) <= 2e-12 * 11
    plan.destroy()
