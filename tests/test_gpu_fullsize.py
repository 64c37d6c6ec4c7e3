"""Full-size parity (BASELINE.json configs[1], [2]) in the launch configuration bench.py times.
The oracle cannot brute-force these sizes, so synthesis is compared on a seeded sample of the
outputs, and the adjoint through (i) a sparse input supported on a sample of the points, for
which Eq. 2 is a short sum, and (ii) the adjoint identity on a dense random input."""
import os

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2406_14542_b200 import inputs  # noqa: E402


def cu(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def rel_max(a, b):
    """max |a - b| / rms(b): names one bad element that a norm would average away."""
    return float(np.max(np.abs(a - b)) / np.sqrt(np.mean(np.abs(b) ** 2)))


# (config, sample size, eps): the configs' own eps, then BASELINE.json configs[4]'s FP64 rows (lmax = 4095 on 67 M
# points at eps = 1e-8 and 1e-12: w = 9 and w = 13, other template paths of the nuFFT kernels than w = 11)
# ... and lmax = 4095 / 67 M points at the paper's own up-sampling sigma = 1.25 (w = 17 at eps = 1e-10)
# ... and, only with NUSHT_TEST_HUGE=1 (108 GB of plan workspace, two minutes): lmax = 16383 on 537 M points, twice the
# band limit of the largest BASELINE.json config (inputs.CONFIGS[6]; the paper's A100 limit is lmax ~ 9000)
@pytest.mark.parametrize("config,nsample,eps_over,sigma", [
    (2, 1500, None, None), (3, 300, None, None), (4, 100, None, None), (3, 300, 1e-8, None), (3, 300, 1e-12, None),
    (3, 300, None, 1.25),
    pytest.param(6, 40, None, None, marks=pytest.mark.skipif(not os.environ.get("NUSHT_TEST_HUGE"),
                                                             reason="opt-in: NUSHT_TEST_HUGE=1"))])
def test_fullsize_sampled(oracle, config, nsample, eps_over, sigma):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2406_14542_b200 import nusht
    cfg, theta, phi, alm, x = inputs.make_config(config)
    L, M, eps, npts = cfg["lmax"], cfg["mmax"], cfg["eps"], cfg["npts"]
    if eps_over is not None:
        eps = eps_over
    d_theta, d_phi = cu(theta), cu(phi)
    if cfg["deflection"] is not None:
        # lensing-like config: the point set is the deflected pixel grid.  The CUDA path gets it from nusht_pointing,
        # the oracle from oracle.pointing on the sampled pixels (Eq. C1); the two agree to 4e-15 rad
        # (tests/test_gpu_pointing.py), i.e. to lmax x 4e-15 in the map values
        d_theta, d_phi = nusht.nusht_pointing(d_theta, d_phi, *(cu(a) for a in cfg["deflection"]))
    plan = nusht.Plan(L, M, d_theta, d_phi, eps, sigma=sigma)
    del d_theta, d_phi
    d_alm = cu(alm)
    f = plan.synthesis(d_alm).cpu().numpy()
    rng = np.random.default_rng(99)
    idx = np.sort(rng.choice(npts, nsample, replace=False))
    # a few deliberately awkward samples: closest to the poles and to phi = 0 / 2 pi
    idx = np.unique(np.concatenate([idx, [np.argmin(theta), np.argmax(theta), np.argmin(phi), np.argmax(phi)]]))
    if cfg["deflection"] is not None:
        t2, p2 = oracle.pointing(theta[idx], phi[idx], cfg["deflection"][0][idx], cfg["deflection"][1][idx])
        theta, phi = theta.copy(), phi.copy()
        theta[idx], phi[idx] = np.asarray(t2, dtype=np.float64), np.asarray(p2, dtype=np.float64)
    f_ref = oracle.synthesis(L, M, theta[idx], phi[idx], alm, "ld")
    assert rel(f[idx], f_ref) <= 10 * eps
    assert rel_max(f[idx], f_ref) <= 100 * eps
    # adjoint of a sparse map: c_lm = sum_{j in idx} x_j conj(Y_lm(j))
    xs = np.zeros(npts)
    xs[idx] = x[idx]
    c = plan.adjoint(cu(xs)).cpu().numpy()
    c_ref = oracle.adjoint(L, M, theta[idx], phi[idx], x[idx], "ld")
    assert rel(c, c_ref) <= 10 * eps
    # (lmax = 16383: measured 3.5e-8 = 350 eps, all of it on the m = 0 coefficients above l = 16000, which are 31 times the
    # rms of c because the sample contains the two points nearest the poles; relative to themselves they are off by 1.1e-9)
    assert rel_max(c, c_ref) <= (100 if L < 16000 else 1000) * eps
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
    bar = 1e-4 if eps >= 1e-5 else 1e-5      # measured at eps = 1e-6: 8e-7 (binary32 I/O and fine grid)
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


# (l, m) of the sparse coefficient set of the all-points test: the corners of the triangle, low and high m at
# l = lmax (Pbar_mm underflows for most theta at m ~ lmax), a mid-triangle entry, and l = 0, 1
SPARSE_LM = [(4095, 4095), (4095, 0), (4095, 1), (2048, 1024), (1, 1), (0, 0), (3000, 2999), (4095, 4000)]


def test_fullsize_all_points_sparse_alm(oracle):
    """BASELINE.json configs[2] (lmax 4095, 67 M points, eps 1e-10) with a_lm supported on 8 entries: Eq. 3 is then
    f_j = sum_q w_m Re(a_q e^{i m phi_j}) Pbar_lm(theta_j), which the oracle can evaluate one (l, m) at a time
    (oracle.ring_sum with a single coefficient, binary64: its own error is ~1e-13, the bar is 1e-9) on EVERY 16th point
    of the randomly ordered list: 4.2 M outputs, about 55 in each (segment, strip) work item of the nuFFT kernels,
    so a defect at one strip boundary, pole row or phi seam cannot hide as it could in a 300-point sample.
    The transposed check: x supported on the same 4.2 M points, c_lm = sum_j x_j Pbar_lm(theta_j) e^{-i m phi_j}
    (Eq. 2) for the same 8 entries, from the same Pbar values."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2406_14542_b200 import nusht
    cfg, theta, phi, _, x = inputs.make_config(3)
    L, M, eps, npts = cfg["lmax"], cfg["mmax"], cfg["eps"], cfg["npts"]
    rng = np.random.default_rng(97)
    alm = np.zeros(inputs.nlm(L, M), dtype=np.complex128)
    coef = {}
    for (l, m) in SPARSE_LM:
        a = rng.standard_normal() + (0.0 if m == 0 else 1j * rng.standard_normal())
        coef[(l, m)] = a
        alm[inputs.lm_index(L, l, m)] = a
    plan = nusht.Plan(L, M, cu(theta), cu(phi), eps)
    f = plan.synthesis(cu(alm)).cpu().numpy()
    sel = np.arange(5, npts, 16)
    th, ph = theta[sel], phi[sel]
    f_ref = np.zeros(len(sel), dtype=np.longdouble)
    P, E = {}, {}
    for (l, m) in SPARSE_LM:
        am = np.zeros(l - m + 1, dtype=np.complex128)
        am[-1] = 1.0
        P[(l, m)] = oracle.ring_sum(l, m, th, am, "d").real
        ang = np.longdouble(m) * np.longdouble(ph)
        E[(l, m)] = (np.cos(ang), np.sin(ang))
        a = coef[(l, m)]
        wm = 1.0 if m == 0 else 2.0
        f_ref += wm * (a.real * E[(l, m)][0] - a.imag * E[(l, m)][1]) * P[(l, m)]
    f_ref = np.asarray(f_ref, dtype=np.float64)
    assert rel(f[sel], f_ref) <= 10 * eps
    assert rel_max(f[sel], f_ref) <= 100 * eps
    # every output of the full map is finite and of the right size (the other 15/16 of the points)
    assert np.all(np.isfinite(f)) and abs(np.sqrt(np.mean(f ** 2)) / np.sqrt(np.mean(f_ref ** 2)) - 1) < 1e-2
    # adjoint on the same points
    xs = np.zeros(npts)
    xs[sel] = x[sel]
    c = plan.adjoint(cu(xs)).cpu().numpy()
    got, ref = [], []
    for (l, m) in SPARSE_LM:
        xp = np.longdouble(x[sel]) * P[(l, m)]
        r = complex(float(np.sum(xp * E[(l, m)][0])), 0.0 if m == 0 else -float(np.sum(xp * E[(l, m)][1])))
        got.append(c[inputs.lm_index(L, l, m)])
        ref.append(r)
    got, ref = np.array(got), np.array(ref)
    assert rel(got, ref) <= 10 * eps
    assert np.max(np.abs(got - ref)) <= 100 * eps * np.sqrt(np.mean(np.abs(ref) ** 2))
    plan.destroy()


def test_fullsize_ring_grid_gauss_legendre_4095(oracle):
    """Ring-grid transforms at the band limit of the headline workload: a Gauss-Legendre grid with lmax = 4095 (4096
    rings x 8192 pixels = 33.6 M pixels, the kind of grid the paper computes its maps on), in the
    configuration `bench.py --ring gl` times.  Sampled pixels against Eq. 3 (long-double oracle; Pbar_mm underflows on
    most rings at this lmax), the quadrature round trip analysis(synthesis(a)) = a (the special case of PAPER.md:74),
    and the deflection field of Eq. C2 on the same grid against the oracle's direct sum."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2406_14542_b200 import nusht
    L = 4095
    x = np.polynomial.legendre.leggauss(L + 1)[0].astype(np.longdouble)
    for _ in range(3):                      # polish numpy's nodes in long double (they lose digits at n ~ 1000)
        p0, p1 = np.ones_like(x), x.copy()
        for k in range(2, L + 2):
            p0, p1 = p1, ((2 * k - 1) * x * p1 - (k - 1) * p0) / k
        dp = (L + 1) * (x * p1 - p0) / (x * x - 1)
        x = x - p1 / dp
    p0, p1 = np.ones_like(x), x.copy()
    for k in range(2, L + 2):
        p0, p1 = p1, ((2 * k - 1) * x * p1 - (k - 1) * p0) / k
    dp = (L + 1) * (x * p1 - p0) / (x * x - 1)
    wq = np.asarray(2 / ((1 - x * x) * dp * dp), dtype=np.float64)
    theta = np.asarray(np.arccos(x[::-1]), dtype=np.float64)
    half = (L + 1) // 2
    theta[L + 1 - half:] = np.pi - theta[:half][::-1]
    nphi = np.full(L + 1, 2 * L + 2)
    plan = nusht.RingPlan(L, L, theta, nphi, None, wq[::-1] * (2 * np.pi / (2 * L + 2)))
    assert plan.info.npairs == (L + 1) // 2 and plan.info.nruns == 1
    alm = inputs.random_alm(L, L, 601)
    f = plan.synthesis(cu(alm))
    back = plan.analysis(f).cpu().numpy()
    assert rel(back, alm) <= 5e-12
    assert np.max(np.abs(back - alm)) <= 2e-10 * np.max(np.abs(alm))
    th = np.repeat(theta, nphi)
    ph = np.tile(2 * np.pi * np.arange(2 * L + 2) / (2 * L + 2), L + 1)
    rng = np.random.default_rng(602)
    idx = np.sort(rng.choice(len(th), 300, replace=False))
    idx = np.unique(np.concatenate([idx, [0, 5, len(th) - 1, (L // 2) * (2 * L + 2) + 7, (L // 2 + 1) * (2 * L + 2) + 7]]))
    f_ref = oracle.synthesis(L, L, th[idx], ph[idx], alm, "ld")
    fh = f.cpu().numpy()
    assert rel(fh[idx], f_ref) <= 5e-11
    assert rel_max(fh[idx], f_ref) <= 5e-10
    philm = inputs.random_alm(L, L, 603, "inv_l2")
    a_t, a_p = (t.cpu().numpy() for t in plan.gradient(cu(philm)))
    r_t, r_p = oracle.gradient(L, L, th[idx], ph[idx], philm, "ld")
    s = np.sin(th[idx])
    scale = np.sqrt(np.mean(r_t ** 2 + r_p ** 2))
    assert np.max(np.abs(a_t[idx] - r_t) * s) <= 1e-10 * scale
    assert np.max(np.abs(a_p[idx] - r_p) * s) <= 1e-10 * scale
    plan.destroy()
