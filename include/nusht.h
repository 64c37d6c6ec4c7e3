/*
 * nusht.h -- C ABI of the B200-native nonuniform spin-0 spherical harmonic transform (nuSHT)
 * defined in arXiv 2406.14542 ("cunuSHT").  Citations are PAPER.md:<line> of the paper text.
 *
 * The library computes, to a requested accuracy eps (Eq. 9-10),
 *   synthesis / type 2 (Eq. 3):  f_j  = sum_{l<=lmax} sum_m c_lm Y_lm(theta_j, phi_j)
 *   adjoint   / type 1 (Eq. 2):  c_lm = sum_j f_j conj(Y_lm(theta_j, phi_j))
 * by the double-Fourier-sphere factorisation Y = N F D S (Eq. 5-6): ring Legendre
 * transform onto an equi-angular theta grid (S), doubling theta to [0, 2 pi) (D), uniform FFT (F),
 * nonuniform FFT to the points (N); the adjoint runs the transposed chain.  "Plan once, execute
 * repeatedly"; nothing touches host memory between stages.
 *
 * Conventions (readings G1-G3, G11, G12):
 *   Y_lm = Pbar_lm(theta) e^{i m phi}, orthonormal on the sphere, Condon-Shortley phase (Eq. 1,
 *   PAPER.md:47-49; fn. 4).  Real field, only m >= 0 stored:
 *     f_j = sum_l Re(a_l0) Pbar_l0 + 2 sum_{m=1}^{mmax} Re[ e^{i m phi_j} sum_l a_lm Pbar_lm(theta_j) ].
 *   Im(a_l0) is ignored by synthesis and returned as exactly 0 by the adjoint.
 *   The adjoint is the transpose (no quadrature weights), with respect to
 *     <a, c> = sum_l a_l0 c_l0 + 2 sum_{m>=1} Re(a_lm conj(c_lm))   and   <f, x> = sum_j f_j x_j.
 *
 * Layouts:
 *   alm : nlm = (mmax+1)(lmax+1) - mmax(mmax+1)/2 complex numbers of the plan's dtype, interleaved
 *         (re, im), m-major triangular: idx(l, m) = m (2 lmax + 1 - m)/2 + l, 0 <= m <= mmax, m <= l <= lmax.
 *   map : npts reals of the plan's dtype, in the caller's point order.
 *   theta, phi : npts binary64 each, for both dtypes.  theta in [0, pi] (poles allowed), phi any
 *         finite value (wrapped mod 2 pi).  Duplicate points are allowed.
 *
 * Ownership: every data pointer is caller-owned.  Unless a function says HOST, pointers are DEVICE
 * pointers on the current CUDA device.  nusht_plan copies what it needs from theta/phi (they may
 * be freed afterwards) and owns all workspace.  nusht_synthesis / nusht_adjoint allocate nothing,
 * touch no host memory, enqueue on `stream` (a cudaStream_t passed as void*; NULL = default
 * stream) and return without synchronising.  nusht_adjoint OVERWRITES alm.  A plan must not be
 * used from two streams at once (shared workspace).
 *
 * Errors: every call returns a status; nothing throws or exits.  There is no CPU fallback: without
 * a CUDA device nusht_plan returns NUSHT_ERR_CUDA.
 */
#ifndef NUSHT_H
#define NUSHT_H

#include <stdint.h>

#if defined(__GNUC__)
#define NUSHT_API __attribute__((visibility("default")))
#else
#define NUSHT_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nusht_plan_s nusht_plan_t; /* opaque, library-owned */

enum { NUSHT_F64 = 0, NUSHT_F32 = 1 };

enum {
    NUSHT_OK = 0,
    NUSHT_ERR_INVALID_ARG = -1, /* bad lmax/mmax/npts/eps/dtype or NULL pointer */
    NUSHT_ERR_ALLOC = -2,       /* device or host allocation failed */
    NUSHT_ERR_CUDA = -3,        /* CUDA runtime / launch error (also: no device) */
    NUSHT_ERR_CUFFT = -4,       /* cuFFT plan or exec error */
    NUSHT_ERR_UNSUPPORTED = -5, /* valid request this build does not implement */
    NUSHT_ERR_BAD_POINTS = -6,  /* NaN/Inf coordinates or theta outside [0, pi] */
    NUSHT_ERR_TOO_LARGE = -7    /* request beyond the fixed capacity of nusht_stage_legendre_adjoint_static */
};

/* Stage slots reported by nusht_stage_times.
 * When the plan uses a fused theta chain (Ntheta a power of two <= 16384: one kernel does a3 + a4 + the
 * theta pass of a5, and one its transpose in a9) the whole chain is reported in the *_FFT_FINE_THETA slot
 * and the *_FFT_THETA / *_DECONV_* slots read ~0.  The environment variable NUSHT_THETA_CHAIN =
 * cufft | single | cluster, read by nusht_plan, selects the chain variant where it exists (testing). */
enum {
    NUSHT_SYN_ALM_PREP = 0,  /* a1 prologue: coefficient scaling + odd-class fold (O(lmax^2)) */
    NUSHT_SYN_LEGENDRE = 1,  /* a1 + a2: Legendre synthesis with fused DFS doubling */
    NUSHT_SYN_FFT_THETA = 2, /* a3: theta FFT of the doubled rings (cuFFT) */
    NUSHT_SYN_DECONV_PAD = 3,/* a4: kernel deconvolution + zero-pad to the fine grid */
    NUSHT_SYN_FFT_FINE_THETA = 4, /* a5, theta pass (cuFFT) */
    NUSHT_SYN_FFT_FINE_PHI = 5,   /* a5, phi C2R pass (cuFFT) */
    NUSHT_SYN_INTERP = 6,    /* a7: type-2 interpolation */
    NUSHT_ADJ_SPREAD = 0,    /* a8: type-1 spreading (includes zeroing the fine grid) */
    NUSHT_ADJ_FFT_FINE_PHI = 1,   /* a9: phi R2C (cuFFT) */
    NUSHT_ADJ_FFT_FINE_THETA = 2, /* a9: theta forward FFT on the fine grid (cuFFT) */
    NUSHT_ADJ_DECONV_TRUNC = 3,   /* a9: truncate to |k| <= lmax + deconvolve */
    NUSHT_ADJ_FFT_THETA = 4, /* a9: theta inverse FFT back to the doubled rings (cuFFT) */
    NUSHT_ADJ_LEGENDRE = 5,  /* a10 + a11: fold + adjoint Legendre */
    NUSHT_ADJ_ALM_POST = 6,  /* a11 epilogue: odd-class unfold + scaling */
    NUSHT_NUM_STAGES = 7
};

typedef struct {
    int lmax, mmax, dtype;
    int64_t npts, nlm;
    double eps;
    int n_rings;        /* N_r: Clenshaw-Curtis rings theta_k = pi k/(N_r-1), k = 0..N_r-1 */
    int n_theta;        /* doubled length 2 (N_r - 1) (App. B; reading G4) */
    int n_theta_fine;   /* up-sampled grid, theta direction (covers [0, 2 pi)) */
    int n_phi_fine;     /* up-sampled grid, phi direction */
    int kernel_width;   /* w: taps per dimension of the exponential-of-semicircle kernel */
    int kernel_degree;  /* degree of the piecewise polynomial that evaluates it */
    double kernel_beta; /* phi_ES(z) = exp(beta (sqrt(1 - z^2) - 1)) */
    double sigma;       /* up-sampling factor */
    int64_t workspace_bytes; /* device memory owned by the plan */
    double plan_ms;     /* wall time of nusht_plan (sort + tables + cuFFT plans) */
    double sort_ms;     /* a6 alone: point keys + histogram, scan, scatter (CUDA events inside nusht_plan) */
    int64_t legendre_fma_synthesis; /* FP64 FMAs ONE launch of the Legendre synthesis kernel executes: the (l, m, ring */
    int64_t legendre_fma_adjoint;   /* pair) steps left after the plan-time fast-forward x 3 (measurement: the roofline's
                                       executed fraction); the adjoint's cross-lane adds are not counted */
    double set_points_ms; /* wall time of the last nusht_set_points (0: never called) */
} nusht_info_t;

/* Build a plan: choose grid sizes / kernel width from (lmax, mmax, eps), build recurrence and
 * deconvolution tables, counting-sort the points into strips (planning is done
 * before, and excluded from, the transforms).  Synchronous; may synchronise the device.
 *   0 <= lmax <= 32000 (larger: NUSHT_ERR_UNSUPPORTED), 0 <= mmax <= lmax, 0 <= npts < 2^31, dtype NUSHT_F64 | NUSHT_F32,
 *   eps in [1e-13, 1e-1] (F64) or [1e-6, 1e-1] (F32); theta/phi DEVICE pointers (may be NULL iff npts == 0). */
NUSHT_API int nusht_plan(nusht_plan_t** out, int lmax, int mmax, int64_t npts, const double* theta,
               const double* phi, double eps, int dtype);

/* Plan options.  sigma: up-sampling factor of the nuFFT grid, 2 (default; 0 means default) or 1.25, the paper's own
 * choice "to reduce the memory usage at a small price of increased computation time": the fine grid
 * shrinks by (1.25/2)^2 while the kernel widens (w = 17 instead of 11 at eps = 1e-10).  At sigma = 1.25 eps is limited
 * to [1e-10, 1e-1] in FP64 (the floor the paper states, fn. 6 at PAPER.md:164) and [1e-5, 1e-1] in FP32.
 * Other values of sigma: NUSHT_ERR_INVALID_ARG.  nusht_plan(...) == nusht_plan_ex(..., NULL). */
typedef struct {
    double sigma;
    int reserved[6];    /* must be zero */
} nusht_opts_t;
NUSHT_API int nusht_plan_ex(nusht_plan_t** out, int lmax, int mmax, int64_t npts, const double* theta,
                            const double* phi, double eps, int dtype, const nusht_opts_t* opts);

/* Replace the plan's point set, keeping everything that depends on (lmax, mmax, eps, dtype, sigma) only: recurrence
 * and deconvolution tables, FFT plans, the fine grid.  Only the plan-time point sort (a6) runs again; the paper makes
 * the same split ("The plans allow for repeated and fast transforms, without reinitialization") and its
 * lensing use case needs it, one point set per deflection field (Appendix C).  theta, phi as in nusht_plan: DEVICE
 * FP64 arrays of the NEW length npts (0 <= npts < 2^31), read during the call only.  The call synchronises the device
 * (no transform of this plan may be in flight on the old points); with an unchanged npts the point tables are
 * overwritten in place, otherwise the old tables and the host-buffer staging maps are freed (the latter re-created on
 * the next nusht_*_host call or nusht_host_reserve) and new ones allocated; the sort's scratch (40 B per point) is
 * allocated and freed inside the call either way.  The plan's device must be current.  NaN/Inf coordinates or theta outside [0, pi]: NUSHT_ERR_BAD_POINTS, and the plan is
 * left valid WITHOUT points (npts = 0).  nusht_plan_info reports the new npts, workspace and set_points_ms. */
NUSHT_API int nusht_set_points(nusht_plan_t* plan, int64_t npts, const double* theta, const double* phi);

/* Synthesis, Eq. 3 / Eq. 5: alm (DEVICE, nlm complex) -> map (DEVICE, npts real).  npts == 0: no-op.
 * nusht_synthesis and nusht_adjoint allocate nothing and synchronise nothing: they enqueue kernels, cuFFT launches and
 * memsets on `stream` (the adjoint also forks to and joins from a plan-owned side stream with events).  After one eager
 * call of each (which sets kernel attributes) they can be recorded by a stream capture and replayed as a CUDA graph
 * (tests/test_gpu_parity.py::test_transforms_under_cuda_graph_capture). */
NUSHT_API int nusht_synthesis(nusht_plan_t* plan, const void* alm, void* map, void* stream);

/* Adjoint, Eq. 2 / Eq. 6: map (DEVICE, npts real) -> alm (DEVICE, nlm complex, overwritten).
 * npts == 0: alm is set to zero. */
NUSHT_API int nusht_adjoint(nusht_plan_t* plan, const void* map, void* alm, void* stream);

/* Free the plan and everything it owns.  NULL is accepted. */
NUSHT_API int nusht_destroy(nusht_plan_t* plan);

/* Same transforms with HOST buffers (pinned for overlap; pageable works but serialises): the call
 * uploads the input on a plan-owned copy stream, runs the transform on `stream`, downloads the result on
 * a second plan-owned copy stream, and returns without synchronising.  Uploads, kernels and downloads of
 * consecutive calls overlap: each direction has its own device staging buffers (allocated on first use), two sets
 * used in turn, so a call never waits for the copies of the call before it and a loop of host-buffer calls keeps the
 * kernels back to back (PCIe permitting).  The outputs are valid after nusht_host_sync(plan) (or a device-wide
 * synchronisation); synchronising `stream` alone is NOT enough.  The host buffers of a call must stay untouched
 * until then: calls in flight together need host buffers of their own. */
NUSHT_API int nusht_synthesis_host(nusht_plan_t* plan, const void* alm_host, void* map_host, void* stream);
NUSHT_API int nusht_adjoint_host(nusht_plan_t* plan, const void* map_host, void* alm_host, void* stream);
/* Block the calling thread until every host-buffer transform issued so far on this plan has delivered
 * its output. */
NUSHT_API int nusht_host_sync(nusht_plan_t* plan);
/* Allocate the device staging buffers and copy streams of the host-buffer calls now (4 x alm + 4 x map of device
 * memory: input and output of each direction, twice), so that the first nusht_*_host call allocates nothing either.
 * Idempotent. */
NUSHT_API int nusht_host_reserve(nusht_plan_t* plan);

/* Stage entry points (tests and per-stage measurement).
 * Legendre synthesis + DFS doubling alone: alm -> Ftilde, DEVICE complex128
 * [(mmax+1)][n_theta], theta-contiguous:
 *   Ftilde[m][r] = F_m(theta_r) for r < N_r,  (-1)^m F_m(theta_{n_theta - r}) for r >= N_r  (Fig. 1).
 * Its transpose (a10-a11): Gtilde (same layout) -> alm. */
NUSHT_API int nusht_stage_legendre_synthesis(nusht_plan_t* plan, const void* alm, void* ftilde, void* stream);
NUSHT_API int nusht_stage_legendre_adjoint(nusht_plan_t* plan, const void* gtilde, void* alm, void* stream);
/* The same transpose (a10-a11; Eq. 5: S^T D^T) for callers that may not allocate between set-up and
 * tear-down (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): the kernels of
 * nusht_stage_legendre_adjoint, accumulating into a file-scope `static __device__` array of the library instead of the
 * plan's workspace.  The call itself allocates nothing -- no cudaMalloc / cudaFree, no cuFFT, no host allocation -- and
 * enqueues a memset of the array (the kernels accumulate with global reductions, so it must start at zero; it keeps
 * the previous call's contents otherwise), the two Legendre launches and the alm conversion, on `stream` and on the
 * plan's side stream exactly as the ordinary call does.
 *   gtilde  DEVICE complex128 [(mmax+1)][n_theta], caller-owned, read only
 *   alm     DEVICE, plan's dtype, nlm complex, caller-owned, overwritten
 * Capacity: NUSHT_STATIC_SCRATCH_BYTES (8,404,992 B = 262,656 accumulators of 32 B: one per pair of even/odd degrees,
 * sum_m ((lmax - m)/2 + 1) of them), i.e. every plan up to lmax = mmax = 1023; every GPU that loads the library holds
 * the array until the process exits.  A larger plan gives NUSHT_ERR_TOO_LARGE (nothing is enqueued); the plan's
 * device must be the current device, else NUSHT_ERR_INVALID_ARG.
 * ALL calls on one device share the one array: two calls that can overlap on the GPU (different streams without an
 * ordering between them, also from different plans or host threads) race on it and both results are garbage; calls
 * on one stream, or ordered by events, are fine.  The array's device address is looked up once per device
 * (cudaGetSymbolAddress, which may load the module): nusht_static_scratch does that at set-up, so that no call under
 * graph capture is the first one; it returns the capacity in bytes through *bytes (may be NULL). */
#define NUSHT_STATIC_SCRATCH_BYTES 8404992
NUSHT_API int nusht_static_scratch(int64_t* bytes);
NUSHT_API int nusht_stage_legendre_adjoint_static(nusht_plan_t* plan, const void* gtilde, void* alm, void* stream);
/* Fourier stage alone (a3 + a4 + a5, and a9): Ftilde (layout above) -> the plan's half fine grid, DEVICE real
 * [n_theta_fine/2 + 1][n_phi_fine] of the plan's dtype, i.e. the coarse theta FFT, deconvolution by the kernel's
 * Fourier transform, zero-padding and the fine inverse FFT; and its transpose grid -> Gtilde.
 * Ftilde must carry the DFS symmetry Ftilde[m][n_theta - r] = (-1)^m Ftilde[m][r] that a2 produces (the fused chains
 * transform even/odd column pairs together and separate them by it); likewise the Gtilde returned by the transpose
 * is defined up to components that cancel in the fold of a10, G[k] = Gtilde[k] + (-1)^m Gtilde[n_theta - k].  Both
 * calls copy through the plan's own buffers (tests and per-stage measurement only). */
NUSHT_API int nusht_stage_fourier_synthesis(nusht_plan_t* plan, const void* ftilde, void* grid, void* stream);
NUSHT_API int nusht_stage_fourier_adjoint(nusht_plan_t* plan, const void* grid, void* gtilde, void* stream);
/* nuFFT stages alone (a7 / a8) on the plan's half fine grid: DEVICE real [n_theta_fine/2 + 1][n_phi_fine]
 * of the plan's dtype; rows outside [0, pi] are reached through the DFS mirror symmetry.
 * interp reads `grid`, writes `map`; spread zeroes `grid` then accumulates `map` into it. */
NUSHT_API int nusht_stage_interp(nusht_plan_t* plan, const void* grid, void* map, void* stream);
NUSHT_API int nusht_stage_spread(nusht_plan_t* plan, const void* map, void* grid, void* stream);

/* Per-stage CUDA-event timing.  enable != 0 makes every following synthesis/adjoint record events
 * around each stage (no extra synchronisation).  nusht_stage_times synchronises the events of the
 * last call of kind `which` (0 synthesis, 1 adjoint) and writes up to n (<= NUSHT_NUM_STAGES) times in ms. */
NUSHT_API int nusht_set_stage_timing(nusht_plan_t* plan, int enable);
NUSHT_API int nusht_stage_times(nusht_plan_t* plan, int which, float* ms, int n);

/* Pointing for CMB weak lensing (Appendix C, Eq. C1): the positions reached from
 * (theta_i, phi_i) by the deflection (alpha_theta_i, alpha_phi_i), components along e_theta and e_phi in radians,
 *   n' = cos(a) n + (sin(a)/a) (alpha_theta e_theta + alpha_phi e_phi),  a = |(alpha_theta, alpha_phi)|,
 * returned as theta' in [0, pi] and phi' in [0, 2 pi): the point set to hand to nusht_plan.  All six arrays are
 * DEVICE FP64 of length npts, caller-owned; the outputs may alias the inputs element for element (theta_out ==
 * theta is fine).  No plan is involved; the kernel is enqueued on `stream` and the call returns without
 * synchronising.  npts == 0 is a no-op; npts < 0 or a NULL array gives NUSHT_ERR_INVALID_ARG.  The deflection
 * field itself (Eq. C2) is an input here; nusht_ring_gradient computes it from the lensing potential on a ring grid. */
NUSHT_API int nusht_pointing(int64_t npts, const double* theta, const double* phi, const double* alpha_theta,
                             const double* alpha_phi, double* theta_out, double* phi_out, void* stream);

/* ---- transforms on ring grids ("rSHT") and the deflection field of the
 * lensing potential, Eq. C2 (8(f) rank 4) --------------------------------------------------------
 * A ring grid is nrings iso-latitude rings; ring r has colatitude theta[r] in [0, pi], nphi[r] >= 1 equidistant
 * pixels at phi0[r] + 2 pi j / nphi[r], j = 0 .. nphi[r]-1.  The map is the rings one after the other in the order
 * given (1 <= nphi[r] <= 2^21), npix = sum nphi reals of the plan's dtype (Gauss-Legendre, Clenshaw-Curtis, Fejer and HEALPix-style layouts
 * all fit).  theta, nphi, phi0 (NULL: 0) and weight (NULL: 1) are HOST arrays of length nrings, copied by the call.
 *   nusht_ring_synthesis  f(r, j) = sum_lm a_lm Y_lm(theta_r, phi_rj)                              (Eq. 3 on the grid)
 *   nusht_ring_analysis   c_lm = sum_r weight[r] sum_j f(r, j) conj Y_lm(theta_r, phi_rj)          (Eq. 2; weight = 1
 *                         is the plain adjoint; with quadrature weights, e.g. Gauss-Legendre w_r 2 pi / nphi, it inverts
 *                         the synthesis up to lmax, the "special case" of PAPER.md:74).  alm is overwritten.
 *   nusht_ring_gradient   alpha_theta + i alpha_phi = (d/dtheta + (i / sin theta) d/dphi) Phi, Phi = sum Phi_lm Y_lm
 *                         (Eq. C2): two maps of npix reals, the input of nusht_pointing.  A grid with a ring exactly
 *                         at a pole gives NUSHT_ERR_UNSUPPORTED (the components are undefined there).
 * alm / philm: the layout of nusht_synthesis (lmax, mmax of the ring plan).  Rings that mirror each other through the
 * equator (theta_a + theta_b = pi to 2 ulp) share one Legendre recurrence; any other ring costs a pair's work.
 * Maps must start on a 16-byte boundary (any cudaMalloc / torch allocation does).
 * All data pointers are DEVICE pointers; calls enqueue on `stream` and do not synchronise; a ring plan must not be used
 * from two streams at once.  nusht_ring_pairing exposes the pairing rule (host only, no device needed): returns the
 * number of pairs (>= 0) or a negative status; pair_s[j] = -1 marks a ring without mirror. */
typedef struct nusht_ring_plan_s nusht_ring_plan_t;
typedef struct {
    int lmax, mmax, dtype, nrings;
    int npairs;          /* ring pairs the Legendre stage works on (nrings/2 for a symmetric grid) */
    int nruns;           /* batched FFT plans per transform: runs of >= 16 consecutive equal-length rings (one real
                          * cuFFT plan each) + one chirp-z group per padded power-of-two length for all other rings */
    int64_t npix, nlm, workspace_bytes;
    double plan_ms;
} nusht_ring_info_t;
NUSHT_API int nusht_ring_plan(nusht_ring_plan_t** out, int lmax, int mmax, int nrings, const double* theta,
                              const int64_t* nphi, const double* phi0, const double* weight, int dtype);
NUSHT_API int nusht_ring_synthesis(nusht_ring_plan_t* plan, const void* alm, void* map, void* stream);
NUSHT_API int nusht_ring_analysis(nusht_ring_plan_t* plan, const void* map, void* alm, void* stream);
NUSHT_API int nusht_ring_gradient(nusht_ring_plan_t* plan, const void* philm, void* alpha_theta, void* alpha_phi,
                                  void* stream);
NUSHT_API int nusht_ring_info(const nusht_ring_plan_t* plan, nusht_ring_info_t* info);
NUSHT_API int nusht_ring_destroy(nusht_ring_plan_t* plan);
NUSHT_API int nusht_ring_pairing(int nrings, const double* theta, int* pair_n, int* pair_s);

NUSHT_API int nusht_plan_info(const nusht_plan_t* plan, nusht_info_t* info);
/* Number of kernels of THIS library launched by the process so far (cuFFT's kernels and memsets are not counted);
 * bench.py reports the difference over its timed region as `gpu_launches`. */
NUSHT_API int64_t nusht_launch_count(void);
/* Measurement aid (not part of any transform): FP64 throughput of the current device in TFLOP/s, measured with a
 * dependent-free instruction stream on every SM, CUDA events, best of 10 launches.  kind 0: DFMA chains (the
 * instruction of the Legendre kernels); kind 1: DMMA, mma.sync.m8n8k4.f64 (interpolation / spreading).  Synchronous. */
NUSHT_API int nusht_probe_fp64(int kind, double* tflops);
NUSHT_API const char* nusht_strerror(int code);
/* Library version string, e.g. "nusht-b200 0.1 (sm_100a)". */
NUSHT_API const char* nusht_version(void);

#ifdef __cplusplus
}
#endif
#endif /* NUSHT_H */
