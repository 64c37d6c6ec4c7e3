// api.cu -- the C ABI of libnusht.so (include/nusht.h): plan construction, the two transforms,
// stage entry points, timing.  Orchestration only; the arithmetic lives in legendre.cu,
// fourier.cu and nufft.cu.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <atomic>
#include <chrono>
#include <new>

#include <nvtx3/nvToolsExt.h>   // header-only; a no-op unless a profiler injects the NVTX library

#include "nusht_internal.cuh"

static thread_local char g_last_error[512] = "";

// NVTX range over the host-side enqueue of one stage (tracing); Nsight tools project it onto
// the kernels launched inside
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

void nusht_note_cuda_error(cudaError_t e, const char* what, const char* file, int line) {
    snprintf(g_last_error, sizeof(g_last_error), "CUDA error %d (%s) at %s:%d: %s", (int)e, cudaGetErrorString(e),
             file, line, what);
    if (getenv("NUSHT_VERBOSE")) fprintf(stderr, "[nusht] %s\n", g_last_error);
    cudaGetLastError();   // clear the sticky-free error state
}
static std::atomic<long long> g_launches{0};
cudaError_t nusht_launched() {
    g_launches.fetch_add(1, std::memory_order_relaxed);
    return cudaGetLastError();
}
extern "C" int64_t nusht_launch_count(void) { return (int64_t)g_launches.load(std::memory_order_relaxed); }

void nusht_note_cufft_error(int r, const char* what, const char* file, int line) {
    snprintf(g_last_error, sizeof(g_last_error), "cuFFT error %d at %s:%d: %s", r, file, line, what);
    if (getenv("NUSHT_VERBOSE")) fprintf(stderr, "[nusht] %s\n", g_last_error);
}

// smallest even n >= nmin whose only prime factors are 2, 3, 5, 7 (App. B "good numbers")
static int good_even_size(int nmin) {
    int n = nmin + (nmin & 1);
    for (;; n += 2) {
        int k = n;
        for (int pr : {2, 3, 5, 7})
            while (k % pr == 0) k /= pr;
        if (k == 1) return n;
    }
}

extern "C" const char* nusht_version(void) { return "nusht-b200 0.1 (sm_100a)"; }

extern "C" const char* nusht_strerror(int code) {
    switch (code) {
        case NUSHT_OK: return "ok";
        case NUSHT_ERR_INVALID_ARG: return "invalid argument";
        case NUSHT_ERR_ALLOC: return "allocation failed";
        case NUSHT_ERR_CUDA: return g_last_error[0] ? g_last_error : "CUDA error";
        case NUSHT_ERR_CUFFT: return g_last_error[0] ? g_last_error : "cuFFT error";
        case NUSHT_ERR_UNSUPPORTED: return "unsupported request";
        case NUSHT_ERR_BAD_POINTS: return "bad point coordinates (NaN/Inf or theta outside [0, pi])";
        case NUSHT_ERR_TOO_LARGE:
            return "plan too large for the static scratch array of nusht_stage_legendre_adjoint_static "
                   "(NUSHT_STATIC_SCRATCH_BYTES: up to lmax = mmax = 1023)";
    }
    return "unknown status";
}

// the staging buffers, streams and events of the host-buffer calls (sized by npts: nusht_set_points drops them too)
static void host_release(nusht_plan_s* p) {
    if (p->s_h2d) {
        const int64_t esz = p->dtype == NUSHT_F64 ? 8 : 4;
        p->workspace_bytes -= 4 * (p->nlm * 2 * esz) + 4 * (p->host_npts * esz);
    }
    for (int b = 0; b < 2; ++b) {
        cudaFree(p->d_in_alm[b]); cudaFree(p->d_out_alm[b]); cudaFree(p->d_in_map[b]); cudaFree(p->d_out_map[b]);
        p->d_in_alm[b] = p->d_out_alm[b] = p->d_in_map[b] = p->d_out_map[b] = nullptr;
    }
    if (p->s_h2d) cudaStreamDestroy(p->s_h2d);
    if (p->s_d2h) cudaStreamDestroy(p->s_d2h);
    p->s_h2d = p->s_d2h = nullptr;
    for (int k = 0; k < 2; ++k)
        for (int b = 0; b < 2; ++b) {
            if (p->ev_in[k][b]) cudaEventDestroy(p->ev_in[k][b]);
            if (p->ev_cdone[k][b]) cudaEventDestroy(p->ev_cdone[k][b]);
            if (p->ev_out[k][b]) cudaEventDestroy(p->ev_out[k][b]);
            p->ev_in[k][b] = p->ev_cdone[k][b] = p->ev_out[k][b] = nullptr;
        }
    p->host_seq[0] = p->host_seq[1] = 0;
}

static void plan_release(nusht_plan_s* p) {
    if (!p) return;
    legendre_free(p);
    fourier_free(p);
    nufft_free(p);
    host_release(p);
    for (int k = 0; k < 2; ++k)
        for (int i = 0; i <= NUSHT_NUM_STAGES; ++i)
            if (p->ev[k][i]) cudaEventDestroy(p->ev[k][i]);
    delete p;
}

extern "C" int nusht_destroy(nusht_plan_t* plan) {
    plan_release(plan);
    return NUSHT_OK;
}

extern "C" int nusht_plan(nusht_plan_t** out, int lmax, int mmax, int64_t npts, const double* theta,
                          const double* phi, double eps, int dtype) {
    return nusht_plan_ex(out, lmax, mmax, npts, theta, phi, eps, dtype, nullptr);
}

extern "C" int nusht_plan_ex(nusht_plan_t** out, int lmax, int mmax, int64_t npts, const double* theta,
                             const double* phi, double eps, int dtype, const nusht_opts_t* opts) {
    if (!out) return NUSHT_ERR_INVALID_ARG;
    *out = nullptr;
    if (lmax < 0 || mmax < 0 || mmax > lmax || npts < 0 || npts >= ((int64_t)1 << 31)) return NUSHT_ERR_INVALID_ARG;
    if (dtype != NUSHT_F64 && dtype != NUSHT_F32) return NUSHT_ERR_INVALID_ARG;
    double sigma = 2.0;
    if (opts && opts->sigma != 0.0) sigma = opts->sigma;
    if (opts)
        for (int i = 0; i < 6; ++i)
            if (opts->reserved[i] != 0) return NUSHT_ERR_INVALID_ARG;
    if (sigma != 2.0 && sigma != 1.25) return NUSHT_ERR_INVALID_ARG;
    if (!(eps <= 1e-1)) return NUSHT_ERR_INVALID_ARG;
    // accuracy floors: FP64 1e-13 at sigma = 2, 1e-10 at sigma = 1.25 (the paper's fn. 6); FP32 1e-6 / 1e-5
    if (dtype == NUSHT_F64 && !(eps >= (sigma == 2.0 ? 1e-13 : 1e-10))) return NUSHT_ERR_INVALID_ARG;
    if (dtype == NUSHT_F32 && !(eps >= (sigma == 2.0 ? 1e-6 : 1e-5))) return NUSHT_ERR_INVALID_ARG;
    if (npts > 0 && (!theta || !phi)) return NUSHT_ERR_INVALID_ARG;
    if (lmax > 32000) return NUSHT_ERR_UNSUPPORTED;

    const auto t0 = std::chrono::steady_clock::now();
    int dev = 0;
    NUSHT_CUDA_TRY(cudaGetDevice(&dev));

    nusht_plan_s* p = new (std::nothrow) nusht_plan_s();
    if (!p) return NUSHT_ERR_ALLOC;
    p->lmax = lmax;
    p->lmax_io = lmax;
    p->mmax = mmax;
    p->npts = npts;
    p->eps = eps;
    p->dtype = dtype;
    p->sigma = sigma;
    p->device = dev;
    p->nlm = (int64_t)(mmax + 1) * (lmax + 1) - (int64_t)mmax * (mmax + 1) / 2;

    // NUSHT_VERBOSE: wall time of each planning phase on stderr
    const bool verbose = getenv("NUSHT_VERBOSE") != nullptr;
    auto lap = [&, last = t0](const char* what) mutable {
        if (!verbose) return;
        cudaDeviceSynchronize();
        const auto now = std::chrono::steady_clock::now();
        fprintf(stderr, "[nusht] plan: %-28s %8.2f ms\n", what, std::chrono::duration<double, std::milli>(now - last).count());
        last = now;
    };
    int st = nufft_choose_kernel(p);
    lap("kernel width + polynomial fit");
    if (st == NUSHT_OK) {
        // Clenshaw-Curtis rings: N_r >= lmax + 2 with the doubled length 2 (N_r - 1) a good FFT size (reading G4/G5)
        const int nth2 = good_even_size(2 * (lmax + 1));
        p->lg.lmax = lmax;
        p->lg.mmax = mmax;
        p->lg.nth2 = nth2;
        p->lg.nr = nth2 / 2 + 1;
        p->lg.npairs = (p->lg.nr + 1) / 2;
        p->lg.has_equator = p->lg.nr & 1;
        p->lg.ring_mode = 0;
        // fine grid: up-sampling sigma (2, or the paper's 1.25: PAPER.md:152) of the 2 lmax + 2 (2 mmax + 2) Fourier
        // modes (reading G7)
        const int w = p->ng.w;
        int nth = (int)ceil(sigma * (2 * lmax + 2)), nph = (int)ceil(sigma * (2 * mmax + 2));
        p->fourier_general = sigma != 2.0;
        if (nth < 2 * w + 2) nth = 2 * w + 2;
        if (nph < 2 * w + 2) nph = 2 * w + 2;
        p->ng.nth = good_even_size(nth);
        p->ng.nph = good_even_size(nph);
        p->ng.nrow_half = p->ng.nth / 2 + 1;
        st = legendre_build_tables(p);
        lap("Legendre tables");
    }
    if (st == NUSHT_OK) st = fourier_build(p);
    lap("Fourier tables + FFT plans");
    if (st == NUSHT_OK) st = nufft_sort_points(p, theta, phi);
    lap("point sort");
    if (st == NUSHT_OK) {
        for (int k = 0; k < 2 && st == NUSHT_OK; ++k)
            for (int i = 0; i <= NUSHT_NUM_STAGES; ++i)
                if (cudaEventCreate(&p->ev[k][i]) != cudaSuccess) {
                    st = NUSHT_ERR_CUDA;
                    break;
                }
    }
    if (st == NUSHT_OK && cudaDeviceSynchronize() != cudaSuccess) st = NUSHT_ERR_CUDA;
    if (st != NUSHT_OK) {
        plan_release(p);
        return st;
    }
    p->plan_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    *out = p;
    return NUSHT_OK;
}

extern "C" int nusht_set_points(nusht_plan_t* p, int64_t npts, const double* theta, const double* phi) {
    if (!p || npts < 0 || npts >= ((int64_t)1 << 31) || (npts > 0 && (!theta || !phi))) return NUSHT_ERR_INVALID_ARG;
    int dev = -1;
    NUSHT_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != p->device) return NUSHT_ERR_INVALID_ARG;
    const auto t0 = std::chrono::steady_clock::now();
    NUSHT_CUDA_TRY(cudaDeviceSynchronize());      // no transform of this plan may still read the old tables
    if (npts != p->npts) {                        // same count: the tables and staging maps are kept and overwritten
        nufft_free_points(p);
        host_release(p);                          // the staging maps are sized by npts
    }
    p->npts = npts;
    const int st = nufft_sort_points(p, theta, phi);
    if (st != NUSHT_OK || cudaDeviceSynchronize() != cudaSuccess) {
        nufft_free_points(p);                     // leave a valid plan without points
        p->npts = 0;
        p->set_points_ms = 0;
        return st != NUSHT_OK ? st : NUSHT_ERR_CUDA;
    }
    p->set_points_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    return NUSHT_OK;
}

extern "C" int nusht_plan_info(const nusht_plan_t* p, nusht_info_t* info) {
    if (!p || !info) return NUSHT_ERR_INVALID_ARG;
    memset(info, 0, sizeof(*info));
    info->lmax = p->lmax;
    info->mmax = p->mmax;
    info->dtype = p->dtype;
    info->npts = p->npts;
    info->nlm = p->nlm;
    info->eps = p->eps;
    info->n_rings = p->lg.nr;
    info->n_theta = p->lg.nth2;
    info->n_theta_fine = p->ng.nth;
    info->n_phi_fine = p->ng.nph;
    info->kernel_width = p->ng.w;
    info->kernel_degree = p->ng.deg;
    info->kernel_beta = p->beta;
    info->sigma = p->sigma;
    info->workspace_bytes = p->workspace_bytes;
    info->plan_ms = p->plan_ms;
    info->sort_ms = p->sort_ms;
    info->legendre_fma_synthesis = p->leg_fma_syn;
    info->legendre_fma_adjoint = p->leg_fma_adj;
    info->set_points_ms = p->set_points_ms;
    return NUSHT_OK;
}

// ---------------------------------------------------------------------------------------------
// transforms
// ---------------------------------------------------------------------------------------------
#define STAGE_MARK(kind, i)                                                    \
    do {                                                                       \
        if (p->timing) NUSHT_CUDA_TRY(cudaEventRecord(p->ev[(kind)][(i)], s)); \
    } while (0)

static size_t real_size(const nusht_plan_s* p) { return p->dtype == NUSHT_F64 ? 8 : 4; }

extern "C" int nusht_synthesis(nusht_plan_t* p, const void* alm, void* map, void* stream) {
    if (!p || !alm || (!map && p->npts > 0)) return NUSHT_ERR_INVALID_ARG;
    if (p->npts == 0) return NUSHT_OK;
    cudaStream_t s = (cudaStream_t)stream;
    cudaEvent_t fev[5];
    NvtxRange r_all("nusht_synthesis");
    STAGE_MARK(0, 0);
    {
        NvtxRange r("nusht:a1 alm_prep");
        NUSHT_TRY(legendre_alm_prep(p, alm, s));
    }
    STAGE_MARK(0, 1);
    {
        NvtxRange r("nusht:a1+a2 legendre_synthesis");
        NUSHT_TRY(legendre_synthesis(p, p->d_ft, s));
    }
    // stages 2..5 are bracketed inside fourier_synthesis: ev[2] .. ev[6]
    for (int i = 0; i < 5; ++i) fev[i] = p->ev[0][2 + i];
    {
        NvtxRange r("nusht:a3-a5 fourier_synthesis");
        NUSHT_TRY(fourier_synthesis(p, s, p->timing ? fev : nullptr));
    }
    {
        NvtxRange r("nusht:a7 interp");
        NUSHT_TRY(nufft_interp(p, p->d_grid, map, s));
    }
    STAGE_MARK(0, 7);
    if (p->timing) p->ev_valid[0] = true;
    return NUSHT_OK;
}

extern "C" int nusht_adjoint(nusht_plan_t* p, const void* map, void* alm, void* stream) {
    if (!p || !alm || (!map && p->npts > 0)) return NUSHT_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    if (p->npts == 0) {
        NUSHT_CUDA_TRY(cudaMemsetAsync(alm, 0, (size_t)p->nlm * 2 * real_size(p), s));
        return NUSHT_OK;
    }
    cudaEvent_t fev[5];
    NvtxRange r_all("nusht_adjoint");
    STAGE_MARK(1, 0);
    {
        NvtxRange r("nusht:a8 spread");
        NUSHT_TRY(nufft_spread(p, map, p->d_grid, s));
    }
    // stages 1..4 are bracketed inside fourier_adjoint: ev[1] .. ev[5]
    for (int i = 0; i < 5; ++i) fev[i] = p->ev[1][1 + i];
    {
        NvtxRange r("nusht:a9 fourier_adjoint");
        NUSHT_TRY(fourier_adjoint(p, s, p->timing ? fev : nullptr));
    }
    {
        NvtxRange r("nusht:a10+a11 legendre_adjoint");
        NUSHT_TRY(legendre_adjoint(p, p->d_ft, s));
    }
    STAGE_MARK(1, 6);
    {
        NvtxRange r("nusht:a11 alm_post");
        NUSHT_TRY(legendre_alm_post(p, alm, s));
    }
    STAGE_MARK(1, 7);
    if (p->timing) p->ev_valid[1] = true;
    return NUSHT_OK;
}

// Host-buffer transforms.  Copies run on two plan-owned streams (host->device, device->host) and are
// ordered against the compute on `stream` with events, so that with pinned host memory the upload of
// the next input and the download of the previous result overlap the kernels of the current call
// (PCIe is full duplex).  Each direction has its own input and output staging buffers, two sets of them used in
// turn: a call waits for the call before the previous one of its direction to have released its set, never for the
// previous one, so a loop of host-buffer calls without a nusht_host_sync in between runs the kernels back to back.
static int host_setup(nusht_plan_s* p) {
    if (p->s_h2d) return NUSHT_OK;
    const size_t abytes = (size_t)p->nlm * 2 * real_size(p), mbytes = (size_t)p->npts * real_size(p);
    NUSHT_CUDA_TRY(cudaStreamCreateWithFlags(&p->s_h2d, cudaStreamNonBlocking));
    NUSHT_CUDA_TRY(cudaStreamCreateWithFlags(&p->s_d2h, cudaStreamNonBlocking));
    for (int k = 0; k < 2; ++k)
        for (int b = 0; b < 2; ++b) {
            NUSHT_CUDA_TRY(cudaEventCreateWithFlags(&p->ev_in[k][b], cudaEventDisableTiming));
            NUSHT_CUDA_TRY(cudaEventCreateWithFlags(&p->ev_cdone[k][b], cudaEventDisableTiming));
            NUSHT_CUDA_TRY(cudaEventCreateWithFlags(&p->ev_out[k][b], cudaEventDisableTiming));
        }
    for (int b = 0; b < 2; ++b) {
        NUSHT_CUDA_TRY(cudaMalloc(&p->d_in_alm[b], abytes ? abytes : 16));
        NUSHT_CUDA_TRY(cudaMalloc(&p->d_out_alm[b], abytes ? abytes : 16));
        NUSHT_CUDA_TRY(cudaMalloc(&p->d_in_map[b], mbytes ? mbytes : 16));
        NUSHT_CUDA_TRY(cudaMalloc(&p->d_out_map[b], mbytes ? mbytes : 16));
    }
    p->workspace_bytes += (int64_t)(4 * abytes + 4 * mbytes);
    p->host_npts = p->npts;
    return NUSHT_OK;
}

extern "C" int nusht_host_reserve(nusht_plan_t* p) {
    if (!p) return NUSHT_ERR_INVALID_ARG;
    return host_setup(p);
}

extern "C" int nusht_synthesis_host(nusht_plan_t* p, const void* alm_host, void* map_host, void* stream) {
    if (!p || !alm_host || (!map_host && p->npts > 0)) return NUSHT_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t abytes = (size_t)p->nlm * 2 * real_size(p), mbytes = (size_t)p->npts * real_size(p);
    NUSHT_TRY(host_setup(p));
    const int b = (int)(p->host_seq[0]++ & 1u);
    // upload: this set's input buffer is free once the synthesis that last used it (two calls ago) has consumed it
    NUSHT_CUDA_TRY(cudaStreamWaitEvent(p->s_h2d, p->ev_cdone[0][b], 0));
    NUSHT_CUDA_TRY(cudaMemcpyAsync(p->d_in_alm[b], alm_host, abytes, cudaMemcpyHostToDevice, p->s_h2d));
    NUSHT_CUDA_TRY(cudaEventRecord(p->ev_in[0][b], p->s_h2d));
    // compute: needs the input, and this set's output buffer back from its previous download
    NUSHT_CUDA_TRY(cudaStreamWaitEvent(s, p->ev_in[0][b], 0));
    NUSHT_CUDA_TRY(cudaStreamWaitEvent(s, p->ev_out[0][b], 0));
    NUSHT_TRY(nusht_synthesis(p, p->d_in_alm[b], p->d_out_map[b], stream));
    NUSHT_CUDA_TRY(cudaEventRecord(p->ev_cdone[0][b], s));
    // download
    NUSHT_CUDA_TRY(cudaStreamWaitEvent(p->s_d2h, p->ev_cdone[0][b], 0));
    if (mbytes) NUSHT_CUDA_TRY(cudaMemcpyAsync(map_host, p->d_out_map[b], mbytes, cudaMemcpyDeviceToHost, p->s_d2h));
    NUSHT_CUDA_TRY(cudaEventRecord(p->ev_out[0][b], p->s_d2h));
    return NUSHT_OK;
}

extern "C" int nusht_adjoint_host(nusht_plan_t* p, const void* map_host, void* alm_host, void* stream) {
    if (!p || !alm_host || (!map_host && p->npts > 0)) return NUSHT_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t abytes = (size_t)p->nlm * 2 * real_size(p), mbytes = (size_t)p->npts * real_size(p);
    NUSHT_TRY(host_setup(p));
    const int b = (int)(p->host_seq[1]++ & 1u);
    NUSHT_CUDA_TRY(cudaStreamWaitEvent(p->s_h2d, p->ev_cdone[1][b], 0));
    if (mbytes) NUSHT_CUDA_TRY(cudaMemcpyAsync(p->d_in_map[b], map_host, mbytes, cudaMemcpyHostToDevice, p->s_h2d));
    NUSHT_CUDA_TRY(cudaEventRecord(p->ev_in[1][b], p->s_h2d));
    NUSHT_CUDA_TRY(cudaStreamWaitEvent(s, p->ev_in[1][b], 0));
    NUSHT_CUDA_TRY(cudaStreamWaitEvent(s, p->ev_out[1][b], 0));
    NUSHT_TRY(nusht_adjoint(p, p->d_in_map[b], p->d_out_alm[b], stream));
    NUSHT_CUDA_TRY(cudaEventRecord(p->ev_cdone[1][b], s));
    NUSHT_CUDA_TRY(cudaStreamWaitEvent(p->s_d2h, p->ev_cdone[1][b], 0));
    NUSHT_CUDA_TRY(cudaMemcpyAsync(alm_host, p->d_out_alm[b], abytes, cudaMemcpyDeviceToHost, p->s_d2h));
    NUSHT_CUDA_TRY(cudaEventRecord(p->ev_out[1][b], p->s_d2h));
    return NUSHT_OK;
}

extern "C" int nusht_host_sync(nusht_plan_t* p) {
    if (!p) return NUSHT_ERR_INVALID_ARG;
    if (!p->s_d2h) return NUSHT_OK;
    NUSHT_CUDA_TRY(cudaStreamSynchronize(p->s_d2h));   // downloads are ordered after their compute and upload
    return NUSHT_OK;
}

// ---------------------------------------------------------------------------------------------
// stage entry points
// ---------------------------------------------------------------------------------------------
extern "C" int nusht_stage_legendre_synthesis(nusht_plan_t* p, const void* alm, void* ftilde, void* stream) {
    if (!p || !alm || !ftilde) return NUSHT_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    NUSHT_TRY(legendre_alm_prep(p, alm, s));
    return legendre_synthesis(p, (double2*)ftilde, s);
}

extern "C" int nusht_stage_legendre_adjoint(nusht_plan_t* p, const void* gtilde, void* alm, void* stream) {
    if (!p || !alm || !gtilde) return NUSHT_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    NUSHT_TRY(legendre_adjoint(p, (const double2*)gtilde, s));
    return legendre_alm_post(p, alm, s);
}

extern "C" int nusht_static_scratch(int64_t* bytes) { return legendre_static_scratch(bytes); }

extern "C" int nusht_stage_legendre_adjoint_static(nusht_plan_t* p, const void* gtilde, void* alm, void* stream) {
    if (!p || !alm || !gtilde) return NUSHT_ERR_INVALID_ARG;
    return legendre_adjoint_static(p, (const double2*)gtilde, alm, (cudaStream_t)stream);
}

extern "C" int nusht_stage_fourier_synthesis(nusht_plan_t* p, const void* ftilde, void* grid, void* stream) {
    if (!p || !ftilde || !grid) return NUSHT_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t fbytes = sizeof(double2) * (size_t)(p->mmax + 1) * (size_t)p->lg.nth2;
    const size_t gbytes = (size_t)p->ng.nrow_half * (size_t)p->ng.nph * real_size(p);
    NUSHT_CUDA_TRY(cudaMemcpyAsync(p->d_ft, ftilde, fbytes, cudaMemcpyDeviceToDevice, s));
    NUSHT_TRY(fourier_synthesis(p, s, nullptr));
    NUSHT_CUDA_TRY(cudaMemcpyAsync(grid, p->d_grid, gbytes, cudaMemcpyDeviceToDevice, s));
    return NUSHT_OK;
}

extern "C" int nusht_stage_fourier_adjoint(nusht_plan_t* p, const void* grid, void* gtilde, void* stream) {
    if (!p || !gtilde || !grid) return NUSHT_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    const size_t fbytes = sizeof(double2) * (size_t)(p->mmax + 1) * (size_t)p->lg.nth2;
    const size_t gbytes = (size_t)p->ng.nrow_half * (size_t)p->ng.nph * real_size(p);
    NUSHT_CUDA_TRY(cudaMemcpyAsync(p->d_grid, grid, gbytes, cudaMemcpyDeviceToDevice, s));
    NUSHT_TRY(fourier_adjoint(p, s, nullptr));
    NUSHT_CUDA_TRY(cudaMemcpyAsync(gtilde, p->d_ft, fbytes, cudaMemcpyDeviceToDevice, s));
    return NUSHT_OK;
}

extern "C" int nusht_stage_interp(nusht_plan_t* p, const void* grid, void* map, void* stream) {
    if (!p || !grid || (!map && p->npts > 0)) return NUSHT_ERR_INVALID_ARG;
    return nufft_interp(p, grid, map, (cudaStream_t)stream);
}

extern "C" int nusht_stage_spread(nusht_plan_t* p, const void* map, void* grid, void* stream) {
    if (!p || !grid || (!map && p->npts > 0)) return NUSHT_ERR_INVALID_ARG;
    return nufft_spread(p, map, grid, (cudaStream_t)stream);
}

extern "C" int nusht_set_stage_timing(nusht_plan_t* p, int enable) {
    if (!p) return NUSHT_ERR_INVALID_ARG;
    p->timing = enable ? 1 : 0;
    if (!enable) p->ev_valid[0] = p->ev_valid[1] = false;
    return NUSHT_OK;
}

extern "C" int nusht_stage_times(nusht_plan_t* p, int which, float* ms, int n) {
    if (!p || !ms || which < 0 || which > 1 || n < 0 || n > NUSHT_NUM_STAGES) return NUSHT_ERR_INVALID_ARG;
    if (!p->ev_valid[which]) return NUSHT_ERR_INVALID_ARG;
    NUSHT_CUDA_TRY(cudaEventSynchronize(p->ev[which][NUSHT_NUM_STAGES]));
    for (int i = 0; i < n; ++i) NUSHT_CUDA_TRY(cudaEventElapsedTime(&ms[i], p->ev[which][i], p->ev[which][i + 1]));
    return NUSHT_OK;
}
