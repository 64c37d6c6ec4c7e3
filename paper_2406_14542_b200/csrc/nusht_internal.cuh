// nusht_internal.cuh -- plan object and stage launchers shared by the translation units of
// libnusht.so.  Nothing here is visible across the C ABI (include/nusht.h).
#pragma once

#include <thread>
#include <vector>
#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>

#include "../../include/nusht.h"

#define NUSHT_CUDA_TRY(expr)                                   \
    do {                                                       \
        cudaError_t _e = (expr);                               \
        if (_e != cudaSuccess) {                               \
            nusht_note_cuda_error(_e, #expr, __FILE__, __LINE__); \
            return (_e == cudaErrorMemoryAllocation) ? NUSHT_ERR_ALLOC : NUSHT_ERR_CUDA; \
        }                                                      \
    } while (0)

#define NUSHT_CUFFT_TRY(expr)                                  \
    do {                                                       \
        cufftResult _r = (expr);                               \
        if (_r != CUFFT_SUCCESS) {                             \
            nusht_note_cufft_error((int)_r, #expr, __FILE__, __LINE__); \
            return (_r == CUFFT_ALLOC_FAILED) ? NUSHT_ERR_ALLOC : NUSHT_ERR_CUFFT; \
        }                                                      \
    } while (0)

#define NUSHT_TRY(expr)              \
    do {                             \
        int _s = (expr);             \
        if (_s != NUSHT_OK) return _s; \
    } while (0)

void nusht_note_cuda_error(cudaError_t e, const char* what, const char* file, int line);
// called once after every launch of one of OUR kernels: counts it (nusht_launch_count) and returns cudaGetLastError()
cudaError_t nusht_launched();
void nusht_note_cufft_error(int r, const char* what, const char* file, int line);

// ---- nuFFT geometry ------------------------------------------------------------------------
constexpr int NUSHT_MAX_W = 18;          // kernel width limit (sigma = 2: eps = 1e-13 -> w = 14; sigma = 1.25: eps = 1e-10 -> w = 17)
constexpr int NUSHT_MAX_DEG = 19;        // polynomial degree limit (degree = w)
constexpr int NUSHT_SEG_ROWS = 128;      // theta rows of patch origins per work item (strip segment)

struct NufftGeom {
    int nth, nph;        // fine grid (theta covers [0, 2 pi), phi covers [0, 2 pi))
    int nrow_half;       // nth/2 + 1 stored rows (theta in [0, pi])
    int w, fl;           // kernel width, floor(w/2)
    int deg;             // polynomial degree
    int mb;              // strip width in footprint-origin columns (strip columns - w + 1)
    int nstrip;          // ceil(nph / mb)
    int nseg;            // ceil((nth/2 + 2) / NUSHT_SEG_ROWS)
    double inv_hth, inv_hph;  // nth/(2 pi), nph/(2 pi)
};

// ---- Legendre geometry ---------------------------------------------------------------------
struct LegendreGeom {
    int lmax, mmax;
    int nr;              // rings on [0, pi]
    int nth2;            // doubled length 2 (nr - 1)
    int npairs;          // ring pairs (north j, south nr-1-j): ceil(nr/2)
    int has_equator;     // nr odd: last pair is the equator ring alone
    int ring_mode;       // 1: caller ring list (ring.cu): nr = nth2 = number of rings, pairs from d_pair_n / d_pair_s
};

struct nusht_plan_s {
    int lmax = 0, mmax = 0, dtype = 0;
    int64_t npts = 0, nlm = 0;
    double eps = 0, sigma = 2.0, beta = 0;
    int device = 0;
    LegendreGeom lg{};
    NufftGeom ng{};
    int64_t workspace_bytes = 0;
    double plan_ms = 0;
    double sort_ms = 0;             // a6 alone (keys + histogram, scan, scatter), CUDA events
    int64_t leg_fma_syn = 0, leg_fma_adj = 0;   // FP64 FMAs one Legendre launch executes (after the plan-time fast-forward)

    // --- Legendre tables (device) ---
    int64_t* d_eoff = nullptr;      // [mmax+2] offsets of column m in the per-(m,n) tables
    int64_t n_e_total = 0;          // sum_m ne(m)
    double2* d_ab = nullptr;        // (-alpha_n, alpha_n + beta_n) of the x^2-stepping recurrence (sin^2 form), followed at
                                    // + n_e_total by (alpha_n, beta_n), the cos^2 form used by the blocks next to the equator
    double* d_sig = nullptr;        // sigma_n: even-class scaling
    double* d_sodd = nullptr;       // sigma_n / c_{m+2n+1}: odd-class scaling
    double* d_rho = nullptr;        // c_{m+2n+2}/c_{m+2n+3}: odd-class fold ratio
    double* d_x2 = nullptr;         // operand of t_n per ring pair, synthesis decomposition: sin^2(theta_j) for blocks
                                    // before j_quarter, cos^2(theta_j) after (legendre.cu header)
    double* d_x2a = nullptr;        // the same for the adjoint's decomposition (more pairs per block)
    int j_quarter = 0;              // first ring pair with theta >= pi/4 (pairs run from the poles to the equator)
    double* d_x = nullptr;          // cos(theta_j)
    double2* d_logsin = nullptr;    // log2 sin(theta_j) as (hi, lo)
    double2* d_logkap = nullptr;    // log2 |Pbar_mm| prefactor per m as (hi, lo)
    int* d_ff_n = nullptr;          // fast-forward table: first in-range step per (m, block of ring pairs)
    double2* d_ff_p = nullptr;      //   recurrence state (p0, p1) per pair at that step
    int* d_ff_e = nullptr;          //   exponent counter per pair at that step
    int* d_ffa_n = nullptr;         // the same for the adjoint's decomposition (more ring pairs per thread)
    double2* d_ffa_p = nullptr;
    int* d_ffa_e = nullptr;
    int* d_pair_n = nullptr;        // ring-list mode: ring index of the north member of pair j
    int* d_pair_s = nullptr;        //   and of its mirror ring (theta_s = pi - theta_n), -1 if the grid has none
    const double* h_ring_theta = nullptr;   // ring-list mode: HOST colatitudes, valid during legendre_build_tables only
    int lmax_io = 0;                // band limit of the caller's alm layout (= lmax except in ring plans built one degree higher)
    cudaStream_t s_leg_aux = nullptr;       // side stream of the adjoint Legendre stage (second of its two launches)
    cudaEvent_t ev_leg_fork = nullptr, ev_leg_join = nullptr;
    int2* d_items_syn = nullptr;    // work list of the Legendre synthesis: (block of ring pairs, m) per CTA, longest first
    int n_items_syn = 0;
    // --- Legendre work buffers ---
    double4* d_aeo = nullptr;       // scaled coefficients per (m,n): (ae.re, ae.im, ao.re, ao.im)
    double2* d_ft = nullptr;        // Ftilde / Gtilde: [mmax+1][nth2] complex128
    // --- Fourier stage ---
    double* d_pth = nullptr;        // deconvolution factors p_theta(k), k = -lmax..lmax
    double* d_pph = nullptr;        // p_phi(m), m = 0..mmax
    void* d_h = nullptr;            // theta-pass buffer H[m][a]: [mmax+1][nth] complex (dtype)
    double2* d_twz = nullptr;       // W^m = e^{2 pi i m / n_phi}, m = 0..mmax (real-FFT pre/post-processing)
    void* d_grid = nullptr;         // fine real grid [nth/2+1][nph] (dtype)
    cufftHandle fft_theta_coarse = 0;  // Z2Z, length nth2, batch mmax+1
    cufftHandle fft_theta_fine = 0;    // C2C (dtype), length nth, batch mmax+1
    cufftHandle fft_phi = 0;           // C2C (dtype), length nph/2, batch nth/2+1, in place on the grid rows
    bool have_fft = false;
    int theta_chain = 0;            // 0: cuFFT chain, 1: fused chain, one CTA per column, 2: fused chain, cluster pair per column
    bool theta_fused = false;       // a3 + a4 + a5-theta (and their transposes) as one kernel per direction (fourier.cu)
    bool phi_fused = false;         // a9-phi as one shared-memory FFT kernel (fourier.cu: k_phi_adj)
    bool phi_fused_syn = false;     //   ... and a5-phi too (k_phi_syn; only with NUSHT_PHI=fused, see fourier_build)
    double2* d_phitab = nullptr;    //   its twiddle tables (length n_phi / 2)
    bool phi_attr_set[2] = {false, false};
    bool fourier_general = false;   // sigma != 2: full-length fine theta FFT and an out-of-place real phi FFT (fourier.cu)
    void* d_z = nullptr;            //   half spectra of the grid rows, [nth/2+1][nph/2+1] complex (dtype)
    cufftHandle fft_phi_r2c = 0;    //   R2C (dtype), length nph, batch nth/2+1 (fft_phi is then the C2R plan)
    void* d_fftwork = nullptr;      //   one cuFFT work area shared by the four plans of that chain
    double2* d_tw2n = nullptr;      // tables of the fused theta chains (twiddles, position-ordered deconvolution factors)
    int n_sm = 0;                   // SM count of the plan's device (persistent grids)
    bool chain_attr_set[2] = {false, false};   // MaxDynamicSharedMemorySize set for this plan's device (syn, adj)
    // --- points ---
    double* d_px = nullptr;         // sorted theta in fine-grid units
    double* d_py = nullptr;         // sorted phi in fine-grid units
    int* d_perm = nullptr;          // sorted position -> caller index
    int* d_item_off = nullptr;      // [nseg*nstrip + 1] start of each (segment, strip) work item
    int* d_item_order = nullptr;    // work items sorted by decreasing point count
    int n_items = 0;
    // L2-blocked un-permutation of the FP32 interpolation result (nufft.cu): bucket-major slots
    int n_buckets = 1;              // 1: results are scattered through d_perm directly
    int* d_slot = nullptr;          // sorted position -> slot (bucket-major, stable inside a bucket)
    int* d_dest = nullptr;          // slot -> caller index
    void* d_stage = nullptr;        // [npts] results in slot order (dtype)
    int64_t points_bytes = 0;       // device memory of the point tables (the part of workspace_bytes nusht_set_points replaces)
    void* kernel_host = nullptr;    // nufft.cu: host model of the kernel polynomial
    // --- host-buffer staging (allocated on first use of *_host) ---
    // every staging buffer twice: call k of a direction uses set k & 1, so that the upload of the next call and the
    // download of the previous one overlap the kernels of the current one without waiting for each other's buffers
    void *d_in_alm[2] = {}, *d_out_alm[2] = {}, *d_in_map[2] = {}, *d_out_map[2] = {};
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
    cudaEvent_t ev_in[2][2] = {}, ev_cdone[2][2] = {}, ev_out[2][2] = {};   // [0] synthesis, [1] adjoint; [set]
    unsigned host_seq[2] = {0, 0};                                          // host-buffer calls so far, per direction
    int64_t host_npts = 0;                                                  // npts the staging maps were sized for
    double set_points_ms = 0;                                               // wall time of the last nusht_set_points
    // --- stage timing ---
    int timing = 0;
    cudaEvent_t ev[2][NUSHT_NUM_STAGES + 1] = {};
    bool ev_valid[2] = {false, false};
};

// ---- legendre.cu ----
int legendre_build_tables(nusht_plan_s* p);
// pairs rings theta_a + theta_b = pi (to 2 ulp of pi); pair_n / pair_s (size >= nrings) receive the ring indices of
// each pair (pair_s = -1 for a ring without mirror), pairs ordered by increasing distance from the nearer pole.
// Returns the number of pairs.  Host only.
int legendre_pair_rings(int nrings, const double* theta, int* pair_n, int* pair_s);
int legendre_alm_prep(nusht_plan_s* p, const void* alm, cudaStream_t s);
int legendre_synthesis(nusht_plan_s* p, double2* ft, cudaStream_t s);
int legendre_adjoint(nusht_plan_s* p, const double2* gt, cudaStream_t s);
int legendre_alm_post(nusht_plan_s* p, void* alm, cudaStream_t s);
int legendre_static_scratch(int64_t* bytes);                                              // no-allocation variant
int legendre_adjoint_static(nusht_plan_s* p, const double2* gt, void* alm, cudaStream_t s);  // (legendre.cu, end)
void legendre_free(nusht_plan_s* p);

// ---- fourier.cu ----
int fourier_build(nusht_plan_s* p);
int fourier_synthesis(nusht_plan_s* p, cudaStream_t s, cudaEvent_t* ev);   // ft -> grid
int fourier_adjoint(nusht_plan_s* p, cudaStream_t s, cudaEvent_t* ev);     // grid -> ft
void fourier_free(nusht_plan_s* p);

// ---- nufft.cu ----
int nufft_choose_kernel(nusht_plan_s* p);   // w, beta, degree, polynomial + deconvolution tables
int nufft_sort_points(nusht_plan_s* p, const double* theta, const double* phi);
int nufft_interp(nusht_plan_s* p, const void* grid, void* map, cudaStream_t s);
int nufft_spread(nusht_plan_s* p, const void* map, void* grid, cudaStream_t s);
void nufft_free_points(nusht_plan_s* p);     // the point tables only (nusht_set_points)
void nufft_free(nusht_plan_s* p);
// host-side kernel model used by fourier_build: Fourier transform of the piecewise-polynomial kernel
double nufft_kernel_ft(const nusht_plan_s* p, double k, int n);

// plan-time host loops over independent entries (deconvolution tables): the index range cut into one slice per
// hardware thread; body(lo, hi) must not touch shared state
template <typename F>
inline void nusht_parallel_for(int n, F body) {
    unsigned nt = std::thread::hardware_concurrency();
    if (nt > 32) nt = 32;
    if (nt < 2 || n < 64) {
        body(0, n);
        return;
    }
    const int chunk = (n + (int)nt - 1) / (int)nt;
    std::vector<std::thread> pool;
    for (int lo = chunk; lo < n; lo += chunk) pool.emplace_back(body, lo, lo + chunk < n ? lo + chunk : n);
    body(0, chunk < n ? chunk : n);
    for (auto& t : pool) t.join();
}
