"""Full-size parity (BASELINE.json configs[1], [2]) in the launch configuration bench.py times.
The oracle cannot brute-force these sizes, so synthesis is compared on a seeded sample of the
outputs, and the adjoint through (i) a sparse input supported on a sample of the points, for
which Eq. 2 is a short sum, and (ii) the adjoint identity on a dense random input."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2406_14542_b200 import inputs  # noqa: E402


def cu(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.mark.parametrize("config,nsample", [(2, 1500), (3, 300), (4, 100)])
def test_fullsize_sampled(oracle, config, nsample):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2406_14542_b200 import nusht
    cfg, theta, phi, alm, x = inputs.make_config(config)
    L, M, eps, npts = cfg["lmax"], cfg["mmax"], cfg["eps"], cfg["npts"]
    plan = nusht.Plan(L, M, cu(theta), cu(phi), eps)
    d_alm = cu(alm)
    f = plan.synthesis(d_alm).cpu().numpy()
    rng = np.random.default_rng(99)
    idx = np.sort(rng.choice(npts, nsample, replace=False))
    # a few deliberately awkward samples: closest to the poles and to phi = 0 / 2 pi
    idx = np.unique(np.concatenate([idx, [np.argmin(theta), np.argmax(theta), np.argmin(phi), np.argmax(phi)]]))
    f_ref = oracle.synthesis(L, M, theta[idx], phi[idx], alm, "ld")
    assert rel(f[idx], f_ref) <= 10 * eps
    # adjoint of a sparse map: c_lm = sum_{j in idx} x_j conj(Y_lm(j))
    xs = np.zeros(npts)
    xs[idx] = x[idx]
    c = plan.adjoint(cu(xs)).cpu().numpy()
    c_ref = oracle.adjoint(L, M, theta[idx], phi[idx], x[idx], "ld")
    assert rel(c, c_ref) <= 10 * eps
    # adjoint identity on the dense input, accumulated in extended precision
    cd = plan.adjoint(cu(x)).cpu().numpy()
    lhs = float(np.sum(np.longdouble(f) * np.longdouble(x)))
    rhs = oracle.inner_alm(L, M, alm, cd)
    assert abs(lhs - rhs) <= 1e-12 * np.linalg.norm(f) * np.linalg.norm(x)
    # the same identity with x = S a (inner product ||f||^2, no cancellation): a bar on the operator pair
    cf = plan.adjoint(cu(f)).cpu().numpy()
    lhs = float(np.sum(np.longdouble(f) * np.longdouble(f)))
    assert abs(lhs - oracle.inner_alm(L, M, alm, cf)) <= 1e-12 * lhs
    plan.destroy()


@pytest.mark.parametrize("eps", [1e-4, 1e-6])
def test_fullsize_fp32_sampled(oracle, monkeypatch, eps):
    """BASELINE.json configs[4], FP32 rows: lmax = 4095 on 67 M points, in the configuration bench.py --eps-sweep
    times: the gather interpolation with the L2-blocked un-permutation at its default bucket size (16 buckets
    here).  Sampled outputs against the long-double oracle at the north_star bar for the FP32 path (1e-4 at
    eps >= 1e-5; at 1e-6 binary32 itself limits the result, 3e-4 as in test_fp32_path), the whole map against the
    register-window kernel with its direct scatter to binary32 rounding, and every output written exactly once."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2406_14542_b200 import nusht
    cfg, theta, phi, alm, x = inputs.make_config(3)
    L, M, npts = cfg["lmax"], cfg["mmax"], cfg["npts"]
    plan = nusht.Plan(L, M, cu(theta), cu(phi), eps, dtype="f32")
    d_alm = cu(alm.astype(np.complex64))
    f = plan.synthesis(d_alm)
    rng = np.random.default_rng(98)
    idx = np.sort(rng.choice(npts, 200, replace=False))
    idx = np.unique(np.concatenate([idx, [0, npts - 1, np.argmin(theta), np.argmax(theta)]]))
    f_ref = oracle.synthesis(L, M, theta[idx], phi[idx], alm, "ld")
    bar = 1e-4 if eps >= 1e-5 else 3e-4
    assert rel(f[torch.from_numpy(idx).cuda()].cpu().numpy().astype(np.float64), f_ref) <= bar
    # same plan, register-window kernel with the direct scatter map[perm[j]]: same grid, same weights
    g = torch.randn(plan.grid_shape(), dtype=torch.float32, device="cuda")
    f_blocked = plan.stage_interp(g)
    monkeypatch.setenv("NUSHT_INTERP_F32", "window")
    f_window = plan.stage_interp(g)
    monkeypatch.delenv("NUSHT_INTERP_F32")
    assert float((f_blocked - f_window).abs().max()) <= 4e-6 * float(f_window.abs().max())
    # every output was written exactly once: no element keeps the sentinel
    out = torch.full((npts,), float("nan"), dtype=torch.float32, device="cuda")
    plan.synthesis(d_alm, out)
    assert not bool(torch.isnan(out).any())
    assert torch.equal(out, f)
    plan.destroy()
