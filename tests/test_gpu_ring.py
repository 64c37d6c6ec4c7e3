"""Ring-grid transforms ("rSHT": PAPER.md:154, 218) and the deflection field of the lensing
potential (Eq. C2; 8(f) rank 4) on the GPU against the CPU oracle evaluated at the pixel centres:
Eq. 3 / Eq. 2 / Eq. C2 by their direct sums, no grid structure used on the oracle side."""
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


def pixel_centres(theta, nphi, phi0):
    th = np.repeat(theta, nphi)
    ph = np.concatenate([p0 + 2 * np.pi * np.arange(n) / n for n, p0 in zip(nphi, phi0)])
    return th, ph


def leggauss_refined(n):
    """Gauss-Legendre nodes and weights: numpy's, polished by Newton steps on P_n in long double (numpy's own values
    lose digits at n ~ 1000: the round trip below would see 1e-10 from the quadrature alone)."""
    x = np.polynomial.legendre.leggauss(n)[0].astype(np.longdouble)
    for _ in range(3):
        p0, p1 = np.ones_like(x), x.copy()
        for k in range(2, n + 1):
            p0, p1 = p1, ((2 * k - 1) * x * p1 - (k - 1) * p0) / k
        dp = n * (x * p1 - p0) / (x * x - 1)
        x = x - p1 / dp
    p0, p1 = np.ones_like(x), x.copy()
    for k in range(2, n + 1):
        p0, p1 = p1, ((2 * k - 1) * x * p1 - (k - 1) * p0) / k
    dp = n * (x * p1 - p0) / (x * x - 1)
    w = 2 / ((1 - x * x) * dp * dp)
    return x, w


def gauss_legendre_grid(L):
    xl, wl = leggauss_refined(L + 1)
    theta = np.asarray(np.arccos(xl[::-1]), dtype=np.float64)        # north to south
    wg = np.asarray(wl, dtype=np.float64)
    half = (L + 1) // 2                                              # mirror rings exactly symmetric
    theta[L + 1 - half:] = np.pi - theta[:half][::-1]
    nphi = np.full(L + 1, 2 * L + 2)
    return theta, nphi, np.zeros(L + 1), wg[::-1] * (2 * np.pi / (2 * L + 2))


def healpix_like_grid(nside):
    """Ring layout of the HEALPix pixelisation (Gorski et al. 2005), restated: 4 nside - 1 rings; polar caps with
    4 i pixels on ring i at cos(theta) = 1 - i^2/(3 nside^2), pixels at (j + 1/2) pi/(2 i); equatorial belt with
    4 nside pixels at cos(theta) = 4/3 - 2 i/(3 nside), shifted by half a pixel on every other ring."""
    theta, nphi, phi0 = [], [], []
    for i in range(1, 4 * nside):
        if i < nside:
            z, n, p0 = 1 - i * i / (3.0 * nside * nside), 4 * i, np.pi / (4 * i)
        elif i <= 3 * nside:
            z, n = 4.0 / 3 - 2.0 * i / (3 * nside), 4 * nside
            p0 = ((i - nside + 1) % 2) * np.pi / (4 * nside)
        else:
            k = 4 * nside - i
            z, n, p0 = -(1 - k * k / (3.0 * nside * nside)), 4 * k, np.pi / (4 * k)
        theta.append(np.arccos(z)); nphi.append(n); phi0.append(p0)
    theta = np.array(theta)
    half = len(theta) // 2                      # exact mirror symmetry of the colatitudes, as the pixelisation has
    theta[len(theta) - half:] = np.pi - theta[:half][::-1]
    npix = int(np.sum(nphi))
    return theta, np.array(nphi), np.array(phi0), np.full(len(theta), 4 * np.pi / npix)


def irregular_grid(seed):
    rng = np.random.default_rng(seed)
    theta = np.concatenate([[0.0, np.pi / 2, 3.0], np.arccos(rng.uniform(-1, 1, 21))])     # unsorted, a pole, the equator
    nphi = np.concatenate([[1, 64, 3], rng.integers(1, 90, 21)])
    nphi[5], nphi[6], nphi[7] = 2, 7, 128
    phi0 = rng.uniform(-1.0, 7.0, len(theta))
    weight = rng.uniform(0.1, 2.0, len(theta))
    return theta, nphi, phi0, weight


# ---- synthesis / analysis against Eq. 3 / Eq. 2 at the pixel centres ------------------------------------------
@pytest.mark.parametrize("grid,L,M", [("gl", 63, 63), ("gl", 50, 17), ("healpix", 47, 47), ("healpix", 32, 32),
                                      ("healpix", 95, 95), ("irregular", 40, 40), ("irregular", 40, 9)])
def test_ring_transforms_all_pixels(nusht, oracle, grid, L, M):
    theta, nphi, phi0, weight = {"gl": lambda: gauss_legendre_grid(L), "healpix": lambda: healpix_like_grid(16),
                                 "irregular": lambda: irregular_grid(500)}[grid]()
    plan = nusht.RingPlan(L, M, theta, nphi, phi0, weight)
    th, ph = pixel_centres(theta, nphi, phi0)
    assert plan.npix == len(th)
    alm = inputs.random_alm(L, M, 501)
    f = plan.synthesis(cu(alm)).cpu().numpy()
    f_ref = oracle.synthesis(L, M, th, ph, alm, "ld")
    assert rel(f, f_ref) <= 5e-13 * max(1.0, L / 50.0)
    assert np.max(np.abs(f - f_ref)) <= 1e-11 * np.sqrt(np.mean(f_ref ** 2))
    x = inputs.random_map(len(th), 502)
    c = plan.analysis(cu(x)).cpu().numpy()
    c_ref = oracle.adjoint(L, M, th, ph, np.repeat(weight, nphi) * x, "ld")
    assert rel(c, c_ref) <= 5e-13 * max(1.0, L / 50.0)
    assert np.all(c[: L + 1].imag == 0)
    if grid != "irregular":
        assert plan.info.npairs == (len(theta) + 1) // 2          # symmetric grids: one recurrence per ring pair
    plan.destroy()


def test_gauss_legendre_roundtrip_lmax_1023(nusht, oracle):
    """The 'special case' of PAPER.md:74: with Gauss-Legendre weights the analysis inverts the synthesis."""
    L = 1023
    theta, nphi, phi0, weight = gauss_legendre_grid(L)
    plan = nusht.RingPlan(L, L, theta, nphi, phi0, weight)
    alm = inputs.random_alm(L, L, 503)
    f = plan.synthesis(cu(alm))
    back = plan.analysis(f).cpu().numpy()
    assert np.max(np.abs(back - alm)) <= 1e-11 * np.max(np.abs(alm))
    assert rel(back, alm) <= 1e-12
    # a sample of the pixels against Eq. 3
    th, ph = pixel_centres(theta, nphi, phi0)
    idx = np.sort(np.random.default_rng(504).choice(len(th), 1500, replace=False))
    idx = np.unique(np.concatenate([idx, [0, len(th) - 1, 2 * L + 1, 2 * L + 2]]))
    f_ref = oracle.synthesis(L, L, th[idx], ph[idx], alm, "ld")
    assert rel(f.cpu().numpy()[idx], f_ref) <= 2e-11
    plan.destroy()


# ---- the Bluestein pool (rings of short runs) against the per-run cuFFT route and against the oracle --------------
@pytest.mark.parametrize("grid", ["healpix", "irregular", "gl"])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_ring_pool_matches_per_run_fft(nusht, monkeypatch, grid, dtype):
    """NUSHT_RING_POOL=0: every run of equal-length rings is a real cuFFT plan; =all: every ring goes through the
    chirp-z pool; default: short runs only.  Same transform three ways."""
    L = 95
    theta, nphi, phi0, weight = {"gl": lambda: gauss_legendre_grid(L), "healpix": lambda: healpix_like_grid(32),
                                 "irregular": lambda: irregular_grid(510)}[grid]()
    cd = np.complex128 if dtype == "f64" else np.complex64
    rd = np.float64 if dtype == "f64" else np.float32
    alm = inputs.random_alm(L, L, 511).astype(cd)
    x = inputs.random_map(int(np.sum(nphi)), 512).astype(rd)
    res = {}
    for mode in ["0", "all", None]:
        if mode is None:
            monkeypatch.delenv("NUSHT_RING_POOL", raising=False)
        else:
            monkeypatch.setenv("NUSHT_RING_POOL", mode)
        plan = nusht.RingPlan(L, L, theta, nphi, phi0, weight, dtype=dtype)
        res[mode] = (plan.synthesis(cu(alm)).cpu().numpy().astype(np.float64),
                     plan.analysis(cu(x)).cpu().numpy().astype(np.complex128), plan.info.nruns)
        plan.destroy()
    bar = 2e-13 if dtype == "f64" else 2e-6
    for mode in ["all", None]:
        assert rel(res[mode][0], res["0"][0]) <= bar, mode
        assert rel(res[mode][1], res["0"][1]) <= bar, mode
    if grid == "healpix":
        assert res["0"][2] == 2 * 31 + 1            # one plan per cap ring + the belt
        assert res[None][2] <= 8                    # the belt + one pool group per padded length 8 .. 256


def test_healpix_nside_256_sampled(nusht, oracle):
    """2 x 255 cap rings of distinct lengths (4 .. 1020, most of them awkward FFT sizes) through the pool, at
    lmax = 2 nside - 1: sampled pixels against Eq. 3, and <S a, x> = <a, S^T x> over the whole map."""
    nside, L = 256, 511
    theta, nphi, phi0, weight = healpix_like_grid(nside)
    plan = nusht.RingPlan(L, L, theta, nphi, phi0, None)
    assert plan.info.nruns <= 12
    alm = inputs.random_alm(L, L, 513)
    f = plan.synthesis(cu(alm)).cpu().numpy()
    th, ph = pixel_centres(theta, nphi, phi0)
    rng = np.random.default_rng(514)
    idx = np.unique(np.concatenate([rng.choice(len(th), 1500, replace=False), np.arange(0, 40),
                                    len(th) - 1 - np.arange(0, 40), rng.choice(4 * nside * nside // 2, 300)]))
    f_ref = oracle.synthesis(L, L, th[idx], ph[idx], alm, "ld")
    assert rel(f[idx], f_ref) <= 5e-12
    assert np.max(np.abs(f[idx] - f_ref)) <= 5e-11 * np.sqrt(np.mean(f_ref ** 2))
    x = inputs.random_map(len(th), 515)
    c = plan.analysis(cu(x)).cpu().numpy()
    w = np.where(np.arange(plan.nlm) <= L, 1.0, 2.0)                     # m = 0 block first: weights of the G3 product
    lhs = np.sum(np.asarray(f, dtype=np.longdouble) * x)
    rhs = np.sum(np.asarray(w * (alm.real * c.real + alm.imag * c.imag), dtype=np.longdouble))
    assert abs(lhs - rhs) <= 1e-12 * np.linalg.norm(f) * np.linalg.norm(x)
    plan.destroy()


def test_ring_fp32_and_edge_cases(nusht, oracle):
    L = 63
    theta, nphi, phi0, weight = gauss_legendre_grid(L)
    plan = nusht.RingPlan(L, L, theta, nphi, phi0, weight, dtype="f32")
    alm = inputs.random_alm(L, L, 505)
    f = plan.synthesis(cu(alm.astype(np.complex64)))
    assert f.dtype == torch.float32
    th, ph = pixel_centres(theta, nphi, phi0)
    assert rel(f.cpu().numpy().astype(np.float64), oracle.synthesis(L, L, th, ph, alm, "ld")) <= 2e-6
    back = plan.analysis(f).cpu().numpy().astype(np.complex128)
    assert rel(back, alm) <= 5e-6
    plan.destroy()
    # a single ring; lmax = 0; bad arguments
    plan = nusht.RingPlan(0, 0, [1.0], [5])
    f = plan.synthesis(cu(np.array([2.0 + 0j]))).cpu().numpy()
    assert np.allclose(f, 2.0 / np.sqrt(4 * np.pi), rtol=0, atol=1e-15)
    plan.destroy()
    with pytest.raises(nusht.NushtError):
        nusht.RingPlan(4, 4, [3.5], [8])
    with pytest.raises(nusht.NushtError):
        nusht.RingPlan(4, 4, [1.0], [0])


# ---- Eq. C2 --------------------------------------------------------------------------------------------------
def ring_grid_without_poles(nrings, npix):
    theta = np.pi * (np.arange(nrings) + 0.5) / nrings          # the equi-angular grid of BASELINE config 2
    return theta, np.full(nrings, npix), np.zeros(nrings)


@pytest.mark.parametrize("grid,L,M", [("equi", 63, 63), ("equi", 40, 12), ("healpix", 47, 47)])
def test_gradient_all_pixels(nusht, oracle, grid, L, M):
    if grid == "equi":
        theta, nphi, phi0 = ring_grid_without_poles(2 * (L + 1), 2 * (L + 1))
    else:
        theta, nphi, phi0, _ = healpix_like_grid(16)
    plan = nusht.RingPlan(L, M, theta, nphi, phi0)
    philm = inputs.random_alm(L, M, 506, "inv_l2")
    a_t, a_p = (t.cpu().numpy() for t in plan.gradient(cu(philm)))
    th, ph = pixel_centres(theta, nphi, phi0)
    r_t, r_p = oracle.gradient(L, M, th, ph, philm, "ld")
    scale = np.sqrt(np.mean(r_t ** 2 + r_p ** 2))
    # the GPU forms sin(theta) x gradient and divides by sin(theta): the absolute error grows as 1 / sin(theta)
    s = np.sin(th)
    assert np.max(np.abs(a_t - r_t) * s) <= 2e-13 * scale * max(1.0, L / 50.0)
    assert np.max(np.abs(a_p - r_p) * s) <= 2e-13 * scale * max(1.0, L / 50.0)
    assert rel(a_t, r_t) <= 1e-11 and rel(a_p, r_p) <= 1e-11
    plan.destroy()


def test_gradient_rejects_pole_rings(nusht):
    plan = nusht.RingPlan(8, 8, [0.0, 1.0, 2.0], [1, 8, 8])
    with pytest.raises(nusht.NushtError) as e:
        plan.gradient(cu(inputs.random_alm(8, 8, 1)))
    assert e.value.code == -5
    plan.destroy()


def test_lensing_chain_gradient_pointing_synthesis(nusht, oracle):
    """The paper's use case end to end on the GPU (App. C): lensing potential -> deflection field
    (Eq. C2) -> deflected positions (Eq. C1) -> nuSHT synthesis of the unlensed a_lm at those positions; the CPU
    oracle does the same chain by its direct sums on a sample of the pixels."""
    L = 255
    nr = 2 * (L + 1)
    theta, nphi, phi0 = ring_grid_without_poles(nr, nr)
    rplan = nusht.RingPlan(L, L, theta, nphi, phi0)
    # potential with a few-arcminute rms deflection: C_l^{phi phi} ~ 1/(l+1)^2, scaled
    philm = inputs.random_alm(L, L, 507, "inv_l2") * 2.0e-5
    philm[:2] = 0                                   # no monopole / dipole in the potential
    a_t, a_p = rplan.gradient(cu(philm))
    th, ph = pixel_centres(theta, nphi, phi0)
    t2, p2 = nusht.nusht_pointing(cu(th), cu(ph), a_t, a_p)
    rms = float(torch.sqrt(torch.mean(a_t ** 2 + a_p ** 2)))
    assert 2e-4 < rms < 5e-3                        # arcminutes, not degrees
    plan = nusht.Plan(L, L, t2, p2, 1e-10)
    alm = inputs.random_alm(L, L, 508, "inv_l2")
    f = plan.synthesis(cu(alm)).cpu().numpy()
    idx = np.sort(np.random.default_rng(509).choice(len(th), 3000, replace=False))
    g_t, g_p = oracle.gradient(L, L, th[idx], ph[idx], philm, "ld")
    o_t, o_p = oracle.pointing(th[idx], ph[idx], g_t, g_p)
    o_t, o_p = np.asarray(o_t, dtype=np.float64), np.asarray(o_p, dtype=np.float64)
    assert np.max(np.abs(t2.cpu().numpy()[idx] - o_t)) <= 1e-13
    f_ref = oracle.synthesis(L, L, o_t, o_p, alm, "ld")
    assert rel(f[idx], f_ref) <= 1e-9
    plan.destroy()
    rplan.destroy()


def test_lensing_chain_on_a_healpix_layout_with_set_points(nusht, oracle):
    """The same chain as bench.py --ring healpix-lens runs it: the nuSHT plan is built once on the undeflected pixel
    centres and re-pointed with nusht_set_points for every potential (two realisations here), on a HEALPix-style
    layout whose cap rings go through the chirp-z pool."""
    nside, L = 64, 127
    theta, nphi, phi0, _ = healpix_like_grid(nside)
    rplan = nusht.RingPlan(L, L, theta, nphi, phi0)
    th, ph = pixel_centres(theta, nphi, phi0)
    d_th, d_ph = cu(th), cu(ph)
    plan = nusht.Plan(L, L, d_th, d_ph, 1e-10)
    alm = inputs.random_alm(L, L, 520, "inv_l2")
    idx = np.sort(np.random.default_rng(521).choice(len(th), 1500, replace=False))
    idx = np.unique(np.concatenate([idx, np.arange(12), len(th) - 1 - np.arange(12)]))      # cap pixels too
    for k in range(2):
        philm = inputs.random_alm(L, L, 522 + k, "inv_l2") * 4.0e-5
        philm[:2] = 0
        a_t, a_p = rplan.gradient(cu(philm))
        t2, p2 = nusht.nusht_pointing(d_th, d_ph, a_t, a_p)
        plan.set_points(t2, p2)
        f = plan.synthesis(cu(alm)).cpu().numpy()
        g_t, g_p = oracle.gradient(L, L, th[idx], ph[idx], philm, "ld")
        o_t, o_p = oracle.pointing(th[idx], ph[idx], g_t, g_p)
        o_t, o_p = np.asarray(o_t, dtype=np.float64), np.asarray(o_p, dtype=np.float64)
        assert np.max(np.abs(t2.cpu().numpy()[idx] - o_t)) <= 1e-12, k
        f_ref = oracle.synthesis(L, L, o_t, o_p, alm, "ld")
        assert rel(f[idx], f_ref) <= 1e-9, k
    plan.destroy()
    rplan.destroy()
