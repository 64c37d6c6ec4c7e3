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
