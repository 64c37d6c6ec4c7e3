"""Stage pins on the GPU: each half of the factorisation Y = N F D S (Eq. 5,
PAPER.md:80-86) against a definition of its OWN, written out in numpy in this file (no product code, no oracle
code), so that a defect cannot hide behind adjointness or behind the other half.

  P7   S, D (a1-a2) + a plain FFT:  the 2-D Fourier series  sum_m w_m Re[e^{i m phi} sum_k c[m,k] e^{i k theta}]
       with c = FFT(Ftilde)/Ntheta must equal Eq. 3 (the oracle) at arbitrary points -- independent of the nuFFT.
  P10  N alone: interpolation / spreading against the direct sum over the w x w footprint with the
       exponential-of-semicircle kernel itself (ref. [38]); and F + N (a3-a7, a8-a9) against the
       brute-force nonuniform DFT (and its transpose) of a random band-limited spectrum -- independent of the
       Legendre stage.
"""
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


def cu(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def awkward_points(npts, seed):
    theta, phi = inputs.uniform_sphere_points(npts, seed)
    theta[:6] = [0.0, np.pi, 1e-9, np.pi - 1e-9, 0.01, np.pi - 0.01]
    phi[:6] = [0.0, 2 * np.pi - 1e-12, 6.28, 1e-15, 2 * np.pi - 1e-3, 1e-3]
    return theta, phi


def fourier_series(c, k, theta, phi):
    """sum_m w_m Re[ e^{i m phi_j} sum_k c[m,k] e^{i k theta_j} ], w_0 = 1, w_m = 2; c[m, :] on the frequencies k."""
    E = np.exp(1j * np.outer(theta, k))                  # [npts, nk]
    T = E @ c.T                                          # [npts, M+1]
    m = np.arange(c.shape[0])
    w = np.where(m == 0, 1.0, 2.0)
    return np.sum(w[None, :] * np.real(np.exp(1j * np.outer(phi, m)) * T), axis=1)


# ---- P7 ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("L,M,npts", [(15, 15, 2000), (63, 63, 4000), (255, 200, 3000), (100, 37, 2000)])
def test_p7_legendre_dfs_fft_equals_eq3(nusht, oracle, L, M, npts):
    alm = inputs.random_alm(L, M, 300 + L)
    plan = nusht.Plan(L, M, None, None, 1e-10)
    ft = plan.stage_legendre_synthesis(cu(alm)).cpu().numpy()
    n = plan.info.n_theta
    c = np.fft.fft(ft, axis=1) / n
    k = np.rint(np.fft.fftfreq(n, 1.0 / n)).astype(int)
    scale = np.max(np.abs(c))
    # the doubled map has band limit exactly lmax in theta (fn. 4 at 106); the Nyquist row is 0
    assert np.max(np.abs(c[:, np.abs(k) > L])) <= 1e-13 * scale
    # DFS symmetry c[m, -k] = (-1)^m c[m, k]
    sgn = np.where(np.arange(M + 1) % 2 == 0, 1.0, -1.0)[:, None]
    assert np.max(np.abs(c[:, (-np.arange(n)) % n] - sgn * c)) <= 1e-13 * scale
    theta, phi = awkward_points(npts, 301)
    f = fourier_series(c, k, theta, phi)
    f_ref = oracle.synthesis(L, M, theta, phi, alm, "ld")
    assert rel(f, f_ref) <= 1e-13 * max(1.0, L / 50.0)
    assert np.max(np.abs(f - f_ref)) <= 2e-12 * np.sqrt(np.mean(f_ref ** 2)) * max(1.0, L / 50.0)
    plan.destroy()


# ---- P10: the kernel footprint sums, by their definition --------------------------------------------------
def es_weights(X, w, beta):
    """origin a0 = ceil(X - w/2) and the w weights phi_ES(2 (a0 + i - X)/w), phi_ES(z) = exp(beta (sqrt(1 - z^2) - 1))."""
    a0 = np.ceil(X - 0.5 * w).astype(np.int64)
    z = 2.0 * (a0[:, None] + np.arange(w)[None, :] - X[:, None]) / w
    return a0, np.exp(beta * (np.sqrt(np.clip(1.0 - z * z, 0.0, None)) - 1.0)) * (np.abs(z) <= 1.0)


def footprints(info, theta, phi):
    """rows / columns of the stored half grid (theta in [0, pi]; beyond a pole: the DFS mirror g[-a][b] =
    g[a][b + n_phi/2], Fig. 1 at PAPER.md:88-90) and the separable weights of every point."""
    nth, nph, w, beta = info.n_theta_fine, info.n_phi_fine, info.kernel_width, info.kernel_beta
    X = theta * (nth / (2 * np.pi))
    ph = phi - 2 * np.pi * np.floor(phi / (2 * np.pi))
    Y = ph * (nph / (2 * np.pi))
    Y = np.where(Y >= nph, Y - nph, Y)
    a0, wt = es_weights(X, w, beta)
    b0, wp = es_weights(Y, w, beta)
    a = (a0[:, None] + np.arange(w)[None, :]) % nth                      # [npts, w]
    mirror = a > nth // 2
    rows = np.where(mirror, nth - a, a)
    b = b0[:, None] + np.arange(w)[None, :]
    cols_n = b % nph
    cols_m = (b + nph // 2) % nph
    return rows, mirror, cols_n, cols_m, wt, wp


EPS_ALL = [1e-1, 1e-2, 1e-3, 1e-4, 1e-5, 1e-6, 1e-7, 1e-8, 1e-9, 1e-10, 1e-11, 1e-12, 1e-13]


@pytest.mark.parametrize("sigma", [None, 1.25])
@pytest.mark.parametrize("eps", EPS_ALL)
def test_p10_interp_and_spread_against_the_footprint_sum(nusht, eps, sigma):
    """FP64, every kernel width 2..14.  The CUDA kernels evaluate the kernel as a piecewise polynomial fitted to
    phi_ES; the definition here uses phi_ES itself, so the two differ by the fit error, which must stay below eps
    (it is part of the error budget the width rule leaves).  Points include both poles, footprints across the
    phi = 0 seam and across the pole rows."""
    if sigma is not None and eps < 1e-10:
        pytest.skip("sigma = 1.25 is limited to eps >= 1e-10 (PAPER.md:164)")
    L, npts = 61, 6000                      # fine grid 248 x 248: strips of 16 / 24 columns do not divide it
    theta, phi = awkward_points(npts, 310)
    plan = nusht.Plan(L, L, cu(theta), cu(phi), eps, sigma=sigma)
    info = plan.info
    rows, mirror, cn, cm, wt, wp = footprints(info, theta, phi)
    w = info.kernel_width
    rng = np.random.default_rng(311)
    g = rng.standard_normal(plan.grid_shape())
    x = rng.standard_normal(npts)
    f_ref = np.zeros(npts)
    gs_ref = np.zeros(plan.grid_shape())
    for i in range(w):
        for j in range(w):
            cols = np.where(mirror[:, i], cm[:, j], cn[:, j])
            wgt = wt[:, i] * wp[:, j]
            f_ref += g[rows[:, i], cols] * wgt
            np.add.at(gs_ref, (rows[:, i], cols), x * wgt)
    f = plan.stage_interp(cu(g)).cpu().numpy()
    gs = plan.stage_spread(cu(x)).cpu().numpy()
    bar = 2.0 * eps + 1e-14
    assert rel(f, f_ref) <= bar
    assert rel(gs, gs_ref) <= bar
    assert np.max(np.abs(f - f_ref)) <= 20 * bar * np.sqrt(np.mean(f_ref ** 2))
    plan.destroy()


@pytest.mark.parametrize("eps", [1e-2, 1e-4, 1e-6])
def test_p10_fp32_interp_and_spread_against_the_footprint_sum(nusht, eps):
    L, npts = 61, 6000
    theta, phi = awkward_points(npts, 312)
    plan = nusht.Plan(L, L, cu(theta), cu(phi), eps, dtype="f32")
    rows, mirror, cn, cm, wt, wp = footprints(plan.info, theta, phi)
    w = plan.info.kernel_width
    rng = np.random.default_rng(313)
    g = rng.standard_normal(plan.grid_shape()).astype(np.float32)
    x = rng.standard_normal(npts).astype(np.float32)
    f_ref = np.zeros(npts)
    gs_ref = np.zeros(plan.grid_shape())
    for i in range(w):
        for j in range(w):
            cols = np.where(mirror[:, i], cm[:, j], cn[:, j])
            wgt = wt[:, i] * wp[:, j]
            f_ref += g[rows[:, i], cols].astype(np.float64) * wgt
            np.add.at(gs_ref, (rows[:, i], cols), x.astype(np.float64) * wgt)
    f = plan.stage_interp(cu(g)).cpu().numpy().astype(np.float64)
    gs = plan.stage_spread(cu(x)).cpu().numpy().astype(np.float64)
    bar = 2.0 * eps + 2e-6
    assert rel(f, f_ref) <= bar
    assert rel(gs, gs_ref) <= bar
    plan.destroy()


# ---- P10: F + N against the brute-force nonuniform DFT ------------------------------------------------------
def random_dfs_spectrum(L, M, n, seed):
    """c[m, k] on the FFT frequency layout of length n, |k| <= L, with c[m,-k] = (-1)^m c[m,k]."""
    rng = np.random.default_rng(seed)
    c = np.zeros((M + 1, n), dtype=np.complex128)
    v = rng.standard_normal((M + 1, L + 1)) + 1j * rng.standard_normal((M + 1, L + 1))
    sgn = np.where(np.arange(M + 1) % 2 == 0, 1.0, -1.0)
    c[:, : L + 1] = v
    c[:, 0] = np.where(sgn > 0, v[:, 0], 0.0)            # k = 0 of an odd column must vanish
    for k in range(1, L + 1):
        c[:, n - k] = sgn * v[:, k]
    return c


def fold(gt, nr):
    """a10: G[k] = Gt[k] + (-1)^m Gt[n - k] away from the poles."""
    n = gt.shape[1]
    sgn = np.where(np.arange(gt.shape[0]) % 2 == 0, 1.0, -1.0)[:, None]
    out = gt[:, :nr].copy()
    k = np.arange(1, nr - 1)
    out[:, 1: nr - 1] += sgn * gt[:, n - k]
    return out


@pytest.mark.parametrize("eps", EPS_ALL)
@pytest.mark.parametrize("L,M,sigma", [(63, 63, None), (89, 70, None), (63, 63, 1.25), (89, 70, 1.25)])
def test_p10_nufft_against_brute_force_nudft(nusht, eps, L, M, sigma):
    """Ntheta = 128 (fused theta chain) and 180 (cuFFT chain) at sigma = 2; the general chain at sigma = 1.25."""
    if sigma is not None and eps < 1e-10:
        pytest.skip("sigma = 1.25 is limited to eps >= 1e-10 (PAPER.md:164)")
    npts = 3000
    theta, phi = awkward_points(npts, 320)
    plan = nusht.Plan(L, M, cu(theta), cu(phi), eps, sigma=sigma)
    n, nr = plan.info.n_theta, plan.info.n_rings
    c = random_dfs_spectrum(L, M, n, 321)
    k = np.rint(np.fft.fftfreq(n, 1.0 / n)).astype(int)
    ft = np.fft.ifft(c, axis=1) * n                       # Ftilde[m][r] = sum_k c[m,k] e^{2 pi i k r/n}
    grid = plan.stage_fourier_synthesis(cu(ft))
    f = plan.stage_interp(grid).cpu().numpy()
    f_ref = fourier_series(c, k, theta, phi)
    # per dimension the width rule leaves (0.6-2) eps; two dimensions
    bar = 4.0 * eps + 2e-13
    assert rel(f, f_ref) <= bar, rel(f, f_ref)
    assert np.max(np.abs(f - f_ref)) <= 20 * bar * np.sqrt(np.mean(f_ref ** 2))
    # transpose: Gtilde[m][r] = (1/n) sum_{|k|<=L} e^{2 pi i k r/n} sum_j x_j e^{-i k theta_j - i m phi_j},
    # compared after the fold of a10 (the fused chains define Gtilde up to what the fold cancels)
    x = np.random.default_rng(322).standard_normal(npts)
    gt = plan.stage_fourier_adjoint(plan.stage_spread(cu(x))).cpu().numpy()
    kk = k[np.abs(k) <= L]
    Eth = np.exp(-1j * np.outer(kk, theta))              # [nk, npts]
    Eph = np.exp(-1j * np.outer(np.arange(M + 1), phi))  # [M+1, npts]
    cd = (Eph * x[None, :]) @ Eth.T                      # [M+1, nk]
    cfull = np.zeros((M + 1, n), dtype=np.complex128)
    cfull[:, kk % n] = cd
    gt_ref = np.fft.ifft(cfull, axis=1)
    G, G_ref = fold(gt, nr), fold(gt_ref, nr)
    G[0], G_ref[0] = G[0].real, G_ref[0].real            # m = 0: only the real part is used by a11
    # the pole rings of m > 0 are never used either: Pbar_lm(0) = Pbar_lm(pi) = 0 there (a11 multiplies them by 0)
    G[1:, 0] = G_ref[1:, 0] = 0.0
    G[1:, nr - 1] = G_ref[1:, nr - 1] = 0.0
    assert rel(G, G_ref) <= bar, rel(G, G_ref)
    plan.destroy()
