// ring.cu -- spherical harmonic transforms on caller-supplied RING grids (iso-latitude rings of equidistant pixels:
// Gauss-Legendre, Clenshaw-Curtis / Fejer, HEALPix-style layouts), the "rSHT" the paper's package also offers
// ("calculated on a Gauss-Legendre grid", "works on standard pixelization schemes such as
// HEALPix, and can also perform rSHTs"), and on top of it the deflection field of the
// lensing potential, Eq. C2 (second half).
//
//   synthesis  f(r, j) = sum_lm a_lm Y_lm(theta_r, phi0_r + 2 pi j / n_r)                         (Eq. 3 on the grid)
//   analysis   c_lm    = sum_r w_r sum_j f(r, j) conj Y_lm(theta_r, phi0_r + 2 pi j / n_r)        (Eq. 2 with weights;
//              w_r = 1: the plain adjoint; quadrature weights: the inverse on grids that have one)
//   gradient   alpha_theta + i alpha_phi = (d/dtheta + (i / sin theta) d/dphi) Phi                  (Eq. C2)
//
// Pipeline: the Legendre kernels of legendre.cu in ring-list mode (rings paired north/south where the grid is
// symmetric, any colatitudes otherwise) between alm and F[m][ring], then per ring the phi transform: the m of a ring
// are folded onto its n_r Fourier bins (aliasing: rings near the poles have fewer pixels than 2 mmax + 1), followed
// by one real FFT per ring.  cuFFT does the uniform FFTs; everything else is our own kernels.  Long runs of
// consecutive rings of one length (a Gauss-Legendre grid, the equatorial belt of a HEALPix-style layout) are one
// batched real cuFFT plan each.  Rings in short runs (the polar caps of a HEALPix-style layout: 4 i pixels on ring i,
// every ring its own length, 2 x 2047 lengths at nside = 2048) go to a POOL instead, transformed by Bluestein's
// chirp-z algorithm so that a handful of batched power-of-two cuFFT plans serve all of them: with
// c_j = exp(i pi j^2 / n),  exp(2 pi i j k / n) = c_j c_k conj(c_{j-k}),  hence
//   f_j = sum_k Z_k exp(2 pi i j k / n) = c_j * [ (Z c) (*) conj(c) ]_j,
// a linear convolution done as a circular one of length P = 2^p >= 2 n - 1: FFT_P, product with the plan-time
// spectrum of the chirp, inverse FFT_P.  Pool rings are grouped by P; per direction the pool costs two batched Z2Z
// per group plus three elementwise kernels, instead of one cuFFT call of an awkward length per ring (measured at
// nside = 2048: 90 ms per transform with 4095 per-ring calls and 28 s of plan time).
//
// Eq. C2 needs no spin-1 recurrence: with c_l^2 = (l^2 - m^2)/(4 l^2 - 1),
//   sin(theta) dPbar_lm/dtheta = l c_{l+1} Pbar_{l+1,m} - (l + 1) c_l Pbar_{l-1,m},
// so sin(theta) dPhi/dtheta is a SCALAR synthesis, band limit lmax + 1, of the coefficients
//   a'_{l'm} = (l' - 1) c_{l'} Phi_{l'-1,m} - (l' + 2) c_{l'+1} Phi_{l'+1,m},
// dPhi/dphi is the scalar synthesis of i m Phi_lm, and both are divided by sin(theta_r) ring by ring.  The ring plan
// therefore builds its Legendre tables one degree higher than the caller's lmax.
#include <limits.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <chrono>
#include <map>
#include <new>
#include <utility>
#include <vector>

#include "nusht_internal.cuh"

namespace {

struct RingRun {
    int first, count, nphi;
    int64_t pixoff, zoff;
    cufftHandle c2r, r2c;
    bool staged;       // the run's pixels do not start on a 16-byte (FP32: 8-byte) boundary: cuFFT goes through d_stage
};

struct RingMeta {
    const int* nphi;          // pixels per ring
    const int64_t* zoff;      // offset of the ring's half spectrum (n/2 + 1 complex) in z
    const double* phi0;       // azimuth of pixel 0
    const double* scale;      // per-ring factor (analysis: quadrature weight; gradient: 1 / sin theta) or nullptr
    int nrings, M;
    int64_t stride;           // row stride of F[m][ring]
    int small_below;          // synthesis: rings shorter than this are left to k_ring_spec_syn_small (0: none)
    const int* small;         // their indices
};

template <typename C> struct RealOf;
template <> struct RealOf<double2> { using type = double; };
template <> struct RealOf<float2> { using type = float; };

// e^{i m phi0} with the product formed exactly: m phi0 = hi + lo
__device__ __forceinline__ double2 phase(int m, double phi0) {
    const double dm = (double)m, hi = dm * phi0, lo = fma(dm, phi0, -hi);
    double s, c;
    sincos(hi, &s, &c);
    return make_double2(fma(-lo, s, c), fma(lo, c, s));
}

// synthesis, ring r: Fourier bins of the real ring signal.  Mode m contributes A_m = (w_m / 2) F_m e^{i m phi0} to bin
// m mod n and conj(A_m) to bin -m mod n (w_0 = 1, w_m = 2: real field, m >= 0 stored); the half spectrum k = 0 .. n/2
// goes to z (bins 0 and n/2 come out real by construction).  32 rings x 32 bins per CTA, transposed through shared
// memory so that F is read along the ring index and z written along k.
template <typename C>
__global__ void __launch_bounds__(256)
k_ring_spec_syn(RingMeta R, const double2* __restrict__ F, C* __restrict__ z) {
    __shared__ double2 tile[32][33];
    const int r0 = blockIdx.x * 32, k0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    {
        const int r = r0 + tx;
        int n = r < R.nrings ? R.nphi[r] : 0;
        if (n < R.small_below) n = 0;                 // short rings: k_ring_spec_syn_small
        const double phi0 = r < R.nrings ? R.phi0[r] : 0.0;
        const double sc = (r < R.nrings && R.scale) ? R.scale[r] : 1.0;
#pragma unroll 1
        for (int kk = ty; kk < 32; kk += 8) {
            const int k = k0 + kk;
            double2 acc = make_double2(0.0, 0.0);
            if (n > 0 && k <= n / 2) {
                // a ring of n pixels folds (M + 1) / n modes onto each bin: rings next to the poles loop long, so the
                // loads of four terms are issued together (one dependent L2 round trip per term otherwise: the
                // 4-pixel ring of a HEALPix-style grid at lmax = 4095 alone took 0.7 ms)
                auto fold = [&](int m0, double sgn) {
                    int m = m0;
                    for (; m + 3 * n <= R.M; m += 4 * n) {
                        double2 g[4];
#pragma unroll
                        for (int u = 0; u < 4; ++u) g[u] = F[(int64_t)(m + u * n) * R.stride + r];
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            const double2 e = phase(m + u * n, phi0);
                            const double w = (m + u * n) == 0 ? 0.5 : 1.0;
                            acc.x += w * (g[u].x * e.x - g[u].y * e.y);
                            acc.y += sgn * w * (g[u].x * e.y + g[u].y * e.x);
                        }
                    }
                    for (; m <= R.M; m += n) {
                        const double2 g = F[(int64_t)m * R.stride + r], e = phase(m, phi0);
                        const double w = m == 0 ? 0.5 : 1.0;
                        acc.x += w * (g.x * e.x - g.y * e.y);
                        acc.y += sgn * w * (g.x * e.y + g.y * e.x);
                    }
                };
                fold(k, 1.0);
                fold((n - k) % n, -1.0);
                acc.x *= sc;
                acc.y *= sc;
            }
            tile[kk][tx] = acc;
        }
    }
    __syncthreads();
#pragma unroll 1
    for (int rr = ty; rr < 32; rr += 8) {
        const int r = r0 + rr, k = k0 + tx;
        if (r >= R.nrings) continue;
        const int n = R.nphi[r];
        if (k > n / 2 || n < R.small_below) continue;
        const double2 v = tile[tx][rr];
        C out;
        out.x = (typename RealOf<C>::type)v.x;
        out.y = (typename RealOf<C>::type)v.y;
        z[R.zoff[r] + k] = out;
    }
}

// synthesis, rings of fewer than RING_SMALL pixels (the first rings of a polar cap): such a ring folds (M + 1) / n modes
// onto each of its few bins, a loop of thousands of dependent global loads for a handful of threads in the kernel above
// (0.7 ms for the 4-pixel ring of a HEALPix-style grid at lmax = 4095).  Here one CTA takes one ring: all threads bring
// A_m = w_m F_m e^{i m phi0} for a block of 4096 modes into shared memory, then thread k sums the entries of bin k.
// Same terms in the same order as the kernel above.
constexpr int RING_SMALL = 64;
constexpr int RING_SMALL_MODES = 4096;
template <typename C>
__global__ void __launch_bounds__(256)
k_ring_spec_syn_small(RingMeta R, const double2* __restrict__ F, C* __restrict__ z) {
    extern __shared__ double2 s_a[];
    const int r = R.small[blockIdx.x], t = threadIdx.x;
    const int n = R.nphi[r];
    const double phi0 = R.phi0[r], sc = R.scale ? R.scale[r] : 1.0;
    double2 acc = make_double2(0.0, 0.0), accm = make_double2(0.0, 0.0);   // terms m = k, and m = -k (mod n)
    for (int m0 = 0; m0 <= R.M; m0 += RING_SMALL_MODES) {
        const int cnt = min(RING_SMALL_MODES, R.M + 1 - m0);
        for (int i = t; i < cnt; i += 256) {
            const int m = m0 + i;
            const double2 g = F[(int64_t)m * R.stride + r], e = phase(m, phi0);
            const double w = m == 0 ? 0.5 : 1.0;
            s_a[i] = make_double2(w * (g.x * e.x - g.y * e.y), w * (g.x * e.y + g.y * e.x));
        }
        __syncthreads();
        if (t <= n / 2) {
            int i = ((t - m0) % n + n) % n;                 // first mode of this block with m = t (mod n)
            for (; i < cnt; i += n) {
                acc.x += s_a[i].x;
                acc.y += s_a[i].y;
            }
            i = (((n - t) % n - m0) % n + n) % n;           // ... with m = -t (mod n)
            for (; i < cnt; i += n) {
                accm.x += s_a[i].x;
                accm.y -= s_a[i].y;
            }
        }
        __syncthreads();
    }
    if (t <= n / 2) {
        C out;
        out.x = (typename RealOf<C>::type)((acc.x + accm.x) * sc);
        out.y = (typename RealOf<C>::type)((acc.y + accm.y) * sc);
        z[R.zoff[r] + t] = out;
    }
}

// analysis, ring r: G_m = scale_r e^{-i m phi0} Y[m],  Y[m] = sum_j f_j e^{-2 pi i m j/n} = bin (m mod n) of the real
// FFT of the ring (bins above n/2 by Hermitian symmetry).
template <typename C>
__global__ void __launch_bounds__(256)
k_ring_spec_adj(RingMeta R, const C* __restrict__ z, double2* __restrict__ G) {
    __shared__ double2 tile[32][33];
    const int r0 = blockIdx.x * 32, m0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll 1
    for (int rr = ty; rr < 32; rr += 8) {
        const int r = r0 + rr, m = m0 + tx;
        double2 g = make_double2(0.0, 0.0);
        if (r < R.nrings && m <= R.M) {
            const int n = R.nphi[r];
            const int b = m % n;
            const C y = (b <= n / 2) ? z[R.zoff[r] + b] : z[R.zoff[r] + (n - b)];
            const double yr = (double)y.x, yi = (b <= n / 2) ? (double)y.y : -(double)y.y;
            const double2 e = phase(m, R.phi0[r]);
            const double sc = R.scale ? R.scale[r] : 1.0;
            g.x = sc * (yr * e.x + yi * e.y);
            g.y = sc * (yi * e.x - yr * e.y);
        }
        tile[rr][tx] = g;
    }
    __syncthreads();
#pragma unroll 1
    for (int mm = ty; mm < 32; mm += 8) {
        const int m = m0 + mm, r = r0 + tx;
        if (m <= R.M && r < R.nrings) G[(int64_t)m * R.stride + r] = tile[tx][mm];
    }
}

// Eq. C2 coefficients (header): ga = a' (band limit L + 1), gb = i m Phi, both in the alm layout of band limit L + 1
template <typename T>
__global__ void __launch_bounds__(256)
k_grad_coeffs(int L, int M, const T* __restrict__ philm, T* __restrict__ ga, T* __restrict__ gb) {
    const int m = blockIdx.y;
    const int lp = m + blockIdx.x * 256 + threadIdx.x;      // l' = m .. L + 1
    if (lp > L + 1) return;
    const int64_t in = (int64_t)m * (2 * L + 1 - m) / 2, out = (int64_t)m * (2 * (L + 1) + 1 - m) / 2;
    auto c = [m](int l) -> double {
        return sqrt((double)((long long)(l - m) * (long long)(l + m)) / (4.0 * (double)l * (double)l - 1.0));
    };
    double are = 0.0, aim = 0.0, bre = 0.0, bim = 0.0;
    if (lp - 1 >= m) {                                       // from Phi_{l'-1,m}:  (l' - 1) c_{l'}
        const double f = (double)(lp - 1) * c(lp);
        are += f * (double)philm[2 * (in + lp - 1)];
        aim += f * (double)philm[2 * (in + lp - 1) + 1];
    }
    if (lp + 1 <= L) {                                       // from Phi_{l'+1,m}:  -(l' + 2) c_{l'+1}
        const double f = -(double)(lp + 2) * c(lp + 1);
        are += f * (double)philm[2 * (in + lp + 1)];
        aim += f * (double)philm[2 * (in + lp + 1) + 1];
    }
    if (lp <= L) {
        bre = -(double)m * (double)philm[2 * (in + lp) + 1];
        bim = (double)m * (double)philm[2 * (in + lp)];
    }
    if (m == 0) aim = 0.0;                                   // Im Phi_l0 is ignored (real field)
    ga[2 * (out + lp)] = (T)are;
    ga[2 * (out + lp) + 1] = (T)aim;
    gb[2 * (out + lp)] = (T)bre;
    gb[2 * (out + lp) + 1] = (T)bim;
}

// ---- Bluestein pool -------------------------------------------------------------------------------------------
struct BlueMeta {
    const int* ring;          // pool slot q -> ring index
    const int* P;             // padded length of the slot's work row
    const int64_t* woff;      // offset of the work row (double2 elements)
    const int64_t* boff;      // offset of the chirp spectrum FFT_P(conj c) of the ring's length
    const int64_t* coff;      // offset of the chirp table c_j, j = 0 .. n-1
    const int64_t* pixoff;    // offset of the ring's pixels in the map
    const int* nphi;          // per ring (not per slot)
    const int64_t* zoff;      // per ring
};

__device__ __forceinline__ double2 zmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// c_j = exp(i pi j^2 / n), the argument reduced exactly: j^2 mod 2 n in integers
__global__ void __launch_bounds__(256)
k_blue_chirp(int n, double2* __restrict__ c) {
    const int j = blockIdx.x * 256 + threadIdx.x;
    if (j >= n) return;
    const long long q = ((long long)j * j) % (2LL * n);
    double sn, cs;
    sincospi((double)q / (double)n, &sn, &cs);
    c[j] = make_double2(cs, sn);
}

// b~_p = conj(c_p) for p < n, conj(c_{P-p}) for P - p < n, else 0  (the chirp, wrapped for the circular convolution)
__global__ void __launch_bounds__(256)
k_blue_kernel_row(int n, int P, const double2* __restrict__ c, double2* __restrict__ row) {
    const int p = blockIdx.x * 256 + threadIdx.x;
    if (p >= P) return;
    double2 v = make_double2(0.0, 0.0);
    if (p < n) v = c[p];
    else if (P - p < n) v = c[P - p];
    v.y = -v.y;
    row[p] = v;
}

// synthesis, before the forward FFT: a_k = Z_k c_k (Z: the ring's Hermitian spectrum from its stored half), zero-padded
template <typename C>
__global__ void __launch_bounds__(256)
k_blue_pre_syn(BlueMeta B, const C* __restrict__ z, const double2* __restrict__ chirp, double2* __restrict__ work) {
    const int q = blockIdx.x, k = blockIdx.y * 256 + threadIdx.x;
    const int P = B.P[q];
    if (k >= P) return;
    const int r = B.ring[q], n = B.nphi[r];
    double2 a = make_double2(0.0, 0.0);
    if (k < n) {
        const bool upper = k > n / 2;
        const C zz = z[B.zoff[r] + (upper ? n - k : k)];
        a = zmul(make_double2((double)zz.x, upper ? -(double)zz.y : (double)zz.y), chirp[B.coff[q] + k]);
    }
    work[B.woff[q] + k] = a;
}

// between the two FFTs: times the chirp spectrum (analysis: its conjugate, the spectrum of the conjugate chirp)
template <bool CONJ>
__global__ void __launch_bounds__(256)
k_blue_mul(BlueMeta B, const double2* __restrict__ spec, double2* __restrict__ work) {
    const int q = blockIdx.x, p = blockIdx.y * 256 + threadIdx.x;
    if (p >= B.P[q]) return;
    double2 b = spec[B.boff[q] + p];
    if (CONJ) b.y = -b.y;
    const int64_t i = B.woff[q] + p;
    work[i] = zmul(work[i], b);
}

// synthesis, after the inverse FFT: f_j = Re(c_j conv_j) / P
template <typename T>
__global__ void __launch_bounds__(256)
k_blue_post_syn(BlueMeta B, const double2* __restrict__ work, const double2* __restrict__ chirp, T* __restrict__ map) {
    const int q = blockIdx.x, j = blockIdx.y * 256 + threadIdx.x;
    const int r = B.ring[q], n = B.nphi[r];
    if (j >= n) return;
    const double2 w = work[B.woff[q] + j], c = chirp[B.coff[q] + j];
    map[B.pixoff[q] + j] = (T)((w.x * c.x - w.y * c.y) / (double)B.P[q]);
}

// analysis, before the forward FFT: a_j = f_j conj(c_j), zero-padded
template <typename T>
__global__ void __launch_bounds__(256)
k_blue_pre_ana(BlueMeta B, const T* __restrict__ map, const double2* __restrict__ chirp, double2* __restrict__ work) {
    const int q = blockIdx.x, j = blockIdx.y * 256 + threadIdx.x;
    const int P = B.P[q];
    if (j >= P) return;
    const int r = B.ring[q], n = B.nphi[r];
    double2 a = make_double2(0.0, 0.0);
    if (j < n) {
        const double f = (double)map[B.pixoff[q] + j];
        const double2 c = chirp[B.coff[q] + j];
        a = make_double2(f * c.x, -f * c.y);
    }
    work[B.woff[q] + j] = a;
}

// analysis, after the inverse FFT: Y_k = conj(c_k) conv_k / P, k = 0 .. n/2
template <typename C>
__global__ void __launch_bounds__(256)
k_blue_post_ana(BlueMeta B, const double2* __restrict__ work, const double2* __restrict__ chirp, C* __restrict__ z) {
    const int q = blockIdx.x, k = blockIdx.y * 256 + threadIdx.x;
    const int r = B.ring[q], n = B.nphi[r];
    if (k > n / 2) return;
    const double2 w = work[B.woff[q] + k], c = chirp[B.coff[q] + k];
    const double inv = 1.0 / (double)B.P[q];
    C out;
    out.x = (typename RealOf<C>::type)((w.x * c.x + w.y * c.y) * inv);
    out.y = (typename RealOf<C>::type)((w.y * c.x - w.x * c.y) * inv);
    z[B.zoff[r] + k] = out;
}

struct BlueGroup {
    int P, count, first;      // padded length, rings, first pool slot
    int64_t woff;             // offset of the group's [count][P] block in the work array
    cufftHandle z2z;
};

}  // namespace

struct nusht_ring_plan_s {
    nusht_plan_s core;                 // Legendre tables (band limit lmax + 1), d_aeo, d_ft = F[m][ring]
    int lmax = 0, mmax = 0, dtype = 0, nrings = 0, max_nphi = 0;
    int64_t npix = 0, nz = 0;
    bool has_pole_ring = false;
    int* d_nphi = nullptr;
    int64_t* d_zoff = nullptr;
    double *d_phi0 = nullptr, *d_weight = nullptr, *d_isin = nullptr;
    void* d_z = nullptr;               // half spectra of all rings, complex (dtype)
    void* d_fftwork = nullptr;         // one cuFFT work area shared by all plans (executions are stream-ordered)
    void* d_stage = nullptr;           // aligned staging for runs whose pixels start off cuFFT's alignment (odd ring lengths)
    void *d_ga = nullptr, *d_gb = nullptr;   // Eq. C2 coefficients
    std::vector<RingRun> runs;         // long runs: batched real cuFFT
    std::map<std::pair<int, int>, std::pair<cufftHandle, cufftHandle>> fft;   // (nphi, batch) -> (C2R, R2C)
    // Bluestein pool (rings of short runs), slots ordered by group
    std::vector<BlueGroup> groups;
    int nsmall = 0;                    // rings of fewer than RING_SMALL pixels (k_ring_spec_syn_small)
    int* d_small = nullptr;
    int npool = 0, pool_maxP = 0;
    int *d_bring = nullptr, *d_bP = nullptr;
    int64_t *d_bwoff = nullptr, *d_bboff = nullptr, *d_bcoff = nullptr, *d_bpix = nullptr;
    double2 *d_bwork = nullptr, *d_bspec = nullptr, *d_bchirp = nullptr;
    int64_t workspace_bytes = 0;
    double plan_ms = 0;
};

static void ring_release(nusht_ring_plan_s* rp) {
    if (!rp) return;
    legendre_free(&rp->core);
    for (auto& kv : rp->fft) {
        if (kv.second.first) cufftDestroy(kv.second.first);
        if (kv.second.second) cufftDestroy(kv.second.second);
    }
    cudaFree(rp->d_nphi); cudaFree(rp->d_zoff); cudaFree(rp->d_phi0); cudaFree(rp->d_weight); cudaFree(rp->d_isin);
    cudaFree(rp->d_z); cudaFree(rp->d_fftwork); cudaFree(rp->d_ga); cudaFree(rp->d_gb); cudaFree(rp->d_stage);
    for (auto& g : rp->groups)
        if (g.z2z) cufftDestroy(g.z2z);
    cudaFree(rp->d_small);
    cudaFree(rp->d_bring); cudaFree(rp->d_bP); cudaFree(rp->d_bwoff); cudaFree(rp->d_bboff); cudaFree(rp->d_bcoff);
    cudaFree(rp->d_bpix); cudaFree(rp->d_bwork); cudaFree(rp->d_bspec); cudaFree(rp->d_bchirp);
    delete rp;
}

template <typename T>
static int r_alloc(T** ptr, size_t bytes, nusht_ring_plan_s* rp) {
    if (bytes == 0) bytes = 16;
    NUSHT_CUDA_TRY(cudaMalloc((void**)ptr, bytes));
    rp->workspace_bytes += (int64_t)bytes;
    return NUSHT_OK;
}

extern "C" int nusht_ring_pairing(int nrings, const double* theta, int* pair_n, int* pair_s) {
    if (nrings < 0 || (nrings > 0 && (!theta || !pair_n || !pair_s))) return NUSHT_ERR_INVALID_ARG;
    for (int i = 0; i < nrings; ++i)
        if (!(theta[i] >= 0.0) || !(theta[i] <= 3.14159265358979323846)) return NUSHT_ERR_BAD_POINTS;
    return legendre_pair_rings(nrings, theta, pair_n, pair_s);
}

static int ring_build(nusht_ring_plan_s* rp, const double* theta, const int64_t* nphi, const double* phi0,
                      const double* weight) {
    const int nr = rp->nrings, M = rp->mmax;
    const bool f64 = rp->dtype == NUSHT_F64;
    nusht_plan_s* c = &rp->core;
    c->lmax = rp->lmax + 1;
    c->lmax_io = rp->lmax;
    c->mmax = M;
    c->dtype = rp->dtype;
    c->npts = 0;
    c->nlm = (int64_t)(M + 1) * (rp->lmax + 1) - (int64_t)M * (M + 1) / 2;
    NUSHT_CUDA_TRY(cudaGetDevice(&c->device));
    c->lg.lmax = c->lmax;
    c->lg.mmax = M;
    c->lg.nr = nr;
    c->lg.nth2 = nr;            // row stride of F[m][ring]
    c->lg.ring_mode = 1;
    c->h_ring_theta = theta;
    NUSHT_TRY(legendre_build_tables(c));
    c->h_ring_theta = nullptr;
    rp->workspace_bytes += c->workspace_bytes;

    // per-ring metadata and runs of consecutive rings of one length
    std::vector<int> h_n(nr);
    std::vector<int64_t> h_zoff(nr);
    std::vector<double> h_phi0(nr), h_w(nr), h_isin(nr);
    std::vector<RingRun> all_runs;
    int64_t pix = 0, zo = 0;
    const long double PI_L = 3.14159265358979323846264338327950288L;
    for (int r = 0; r < nr; ++r) {
        h_n[r] = (int)nphi[r];
        h_zoff[r] = zo;
        h_phi0[r] = phi0 ? phi0[r] : 0.0;
        h_w[r] = weight ? weight[r] : 1.0;
        const long double s = sinl((long double)theta[r]);
        const bool pole = !(theta[r] > 0.0) || !((long double)theta[r] < PI_L) || !(s > 0.0L);
        if (pole) rp->has_pole_ring = true;
        h_isin[r] = pole ? 0.0 : (double)(1.0L / s);
        if (!all_runs.empty() && all_runs.back().nphi == h_n[r]) {
            all_runs.back().count += 1;
        } else {
            RingRun run;
            run.first = r; run.count = 1; run.nphi = h_n[r]; run.pixoff = pix; run.zoff = zo; run.c2r = run.r2c = 0;
            run.staged = (pix % 2) != 0;      // cuFFT wants real data aligned like complex data (map base: 16 bytes)
            all_runs.push_back(run);
        }
        pix += h_n[r];
        zo += h_n[r] / 2 + 1;
        if (h_n[r] > rp->max_nphi) rp->max_nphi = h_n[r];
    }
    rp->npix = pix;
    rp->nz = zo;
    // long runs keep a batched real cuFFT plan each; the rings of short runs go to the Bluestein pool (header).
    // NUSHT_RING_POOL=0 pools nothing, =all pools every ring (tests compare the two routes).
    struct PoolSlot { int ring, n, P; int64_t pixoff; };
    std::vector<PoolSlot> slots;
    {
        int min_run = 16;
        if (const char* ev = getenv("NUSHT_RING_POOL")) {
            if (strcmp(ev, "0") == 0) min_run = 0;
            else if (strcmp(ev, "all") == 0) min_run = INT_MAX;
        }
        for (const auto& run : all_runs) {
            if (run.count >= min_run) {
                rp->runs.push_back(run);
                continue;
            }
            for (int i = 0; i < run.count; ++i) {
                PoolSlot sl;
                sl.ring = run.first + i;
                sl.n = run.nphi;
                sl.pixoff = run.pixoff + (int64_t)i * run.nphi;
                sl.P = 4;
                while (sl.P < 2 * sl.n - 1) sl.P *= 2;
                slots.push_back(sl);
            }
        }
        std::stable_sort(slots.begin(), slots.end(), [](const PoolSlot& a, const PoolSlot& b) {
            return a.P != b.P ? a.P < b.P : a.n < b.n;
        });
    }
    NUSHT_TRY(r_alloc(&rp->d_nphi, sizeof(int) * (size_t)nr, rp));
    NUSHT_TRY(r_alloc(&rp->d_zoff, sizeof(int64_t) * (size_t)nr, rp));
    NUSHT_TRY(r_alloc(&rp->d_phi0, sizeof(double) * (size_t)nr, rp));
    NUSHT_TRY(r_alloc(&rp->d_weight, sizeof(double) * (size_t)nr, rp));
    NUSHT_TRY(r_alloc(&rp->d_isin, sizeof(double) * (size_t)nr, rp));
    NUSHT_CUDA_TRY(cudaMemcpy(rp->d_nphi, h_n.data(), sizeof(int) * (size_t)nr, cudaMemcpyHostToDevice));
    NUSHT_CUDA_TRY(cudaMemcpy(rp->d_zoff, h_zoff.data(), sizeof(int64_t) * (size_t)nr, cudaMemcpyHostToDevice));
    NUSHT_CUDA_TRY(cudaMemcpy(rp->d_phi0, h_phi0.data(), sizeof(double) * (size_t)nr, cudaMemcpyHostToDevice));
    NUSHT_CUDA_TRY(cudaMemcpy(rp->d_weight, h_w.data(), sizeof(double) * (size_t)nr, cudaMemcpyHostToDevice));
    NUSHT_CUDA_TRY(cudaMemcpy(rp->d_isin, h_isin.data(), sizeof(double) * (size_t)nr, cudaMemcpyHostToDevice));
    NUSHT_TRY(r_alloc(&rp->d_z, (size_t)zo * (f64 ? 16 : 8), rp));
    {
        std::vector<int> h_small;
        for (int r = 0; r < nr; ++r)
            if (h_n[r] < RING_SMALL) h_small.push_back(r);
        rp->nsmall = (int)h_small.size();
        if (rp->nsmall) {
            NUSHT_TRY(r_alloc(&rp->d_small, sizeof(int) * h_small.size(), rp));
            NUSHT_CUDA_TRY(cudaMemcpy(rp->d_small, h_small.data(), sizeof(int) * h_small.size(), cudaMemcpyHostToDevice));
            NUSHT_CUDA_TRY(cudaFuncSetAttribute(k_ring_spec_syn_small<double2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                RING_SMALL_MODES * (int)sizeof(double2)));
            NUSHT_CUDA_TRY(cudaFuncSetAttribute(k_ring_spec_syn_small<float2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                RING_SMALL_MODES * (int)sizeof(double2)));
        }
    }
    {   // Eq. C2 coefficient buffers (band limit lmax + 1)
        const int64_t nlm1 = (int64_t)(M + 1) * (rp->lmax + 2) - (int64_t)M * (M + 1) / 2;
        NUSHT_TRY(r_alloc(&rp->d_ga, (size_t)nlm1 * (f64 ? 16 : 8), rp));
        NUSHT_TRY(r_alloc(&rp->d_gb, (size_t)nlm1 * (f64 ? 16 : 8), rp));
    }

    // cuFFT plans, one per distinct (length, batch), all on one shared work area
    size_t wmax = 0;
    for (auto& run : rp->runs) {
        const auto key = std::make_pair(run.nphi, run.count);
        auto it = rp->fft.find(key);
        if (it == rp->fft.end()) {
            cufftHandle hc = 0, hr = 0;
            size_t ws = 0;
            int n[1] = {run.nphi};
            NUSHT_CUFFT_TRY(cufftCreate(&hc));
            rp->fft[key] = std::make_pair(hc, (cufftHandle)0);
            NUSHT_CUFFT_TRY(cufftSetAutoAllocation(hc, 0));
            NUSHT_CUFFT_TRY(cufftMakePlanMany(hc, 1, n, nullptr, 1, 0, nullptr, 1, 0, f64 ? CUFFT_Z2D : CUFFT_C2R, run.count, &ws));
            if (ws > wmax) wmax = ws;
            NUSHT_CUFFT_TRY(cufftCreate(&hr));
            rp->fft[key].second = hr;
            NUSHT_CUFFT_TRY(cufftSetAutoAllocation(hr, 0));
            NUSHT_CUFFT_TRY(cufftMakePlanMany(hr, 1, n, nullptr, 1, 0, nullptr, 1, 0, f64 ? CUFFT_D2Z : CUFFT_R2C, run.count, &ws));
            if (ws > wmax) wmax = ws;
            it = rp->fft.find(key);
        }
        run.c2r = it->second.first;
        run.r2c = it->second.second;
    }
    // Bluestein pool: slots in group order, one batched Z2Z plan per padded length
    rp->npool = (int)slots.size();
    std::vector<int> h_bring, h_bP;
    std::vector<int64_t> h_bwoff, h_bboff, h_bcoff, h_bpix;
    struct Distinct { int n, P; int64_t coff, boff; };
    std::vector<Distinct> distinct;           // distinct ring lengths in slot order (grouped by P)
    int64_t wtot = 0, ctot = 0, btot = 0;
    for (int q = 0; q < rp->npool; ++q) {
        const PoolSlot& sl = slots[q];
        if (rp->groups.empty() || rp->groups.back().P != sl.P) {
            BlueGroup g;
            g.P = sl.P; g.count = 0; g.first = q; g.woff = wtot; g.z2z = 0;
            rp->groups.push_back(g);
        }
        rp->groups.back().count += 1;
        if (distinct.empty() || distinct.back().n != sl.n) {
            distinct.push_back({sl.n, sl.P, ctot, btot});
            ctot += sl.n;
            btot += sl.P;
        }
        h_bring.push_back(sl.ring);
        h_bP.push_back(sl.P);
        h_bwoff.push_back(wtot);
        h_bboff.push_back(distinct.back().boff);
        h_bcoff.push_back(distinct.back().coff);
        h_bpix.push_back(sl.pixoff);
        wtot += sl.P;
        if (sl.P > rp->pool_maxP) rp->pool_maxP = sl.P;
    }
    for (auto& g : rp->groups) {
        size_t ws = 0;
        int n[1] = {g.P};
        NUSHT_CUFFT_TRY(cufftCreate(&g.z2z));
        NUSHT_CUFFT_TRY(cufftSetAutoAllocation(g.z2z, 0));
        NUSHT_CUFFT_TRY(cufftMakePlanMany(g.z2z, 1, n, nullptr, 1, 0, nullptr, 1, 0, CUFFT_Z2Z, g.count, &ws));
        if (ws > wmax) wmax = ws;
    }
    NUSHT_TRY(r_alloc(&rp->d_fftwork, wmax, rp));
    if (rp->npool) {
        const size_t nq = (size_t)rp->npool;
        NUSHT_TRY(r_alloc(&rp->d_bring, sizeof(int) * nq, rp));
        NUSHT_TRY(r_alloc(&rp->d_bP, sizeof(int) * nq, rp));
        NUSHT_TRY(r_alloc(&rp->d_bwoff, sizeof(int64_t) * nq, rp));
        NUSHT_TRY(r_alloc(&rp->d_bboff, sizeof(int64_t) * nq, rp));
        NUSHT_TRY(r_alloc(&rp->d_bcoff, sizeof(int64_t) * nq, rp));
        NUSHT_TRY(r_alloc(&rp->d_bpix, sizeof(int64_t) * nq, rp));
        NUSHT_CUDA_TRY(cudaMemcpy(rp->d_bring, h_bring.data(), sizeof(int) * nq, cudaMemcpyHostToDevice));
        NUSHT_CUDA_TRY(cudaMemcpy(rp->d_bP, h_bP.data(), sizeof(int) * nq, cudaMemcpyHostToDevice));
        NUSHT_CUDA_TRY(cudaMemcpy(rp->d_bwoff, h_bwoff.data(), sizeof(int64_t) * nq, cudaMemcpyHostToDevice));
        NUSHT_CUDA_TRY(cudaMemcpy(rp->d_bboff, h_bboff.data(), sizeof(int64_t) * nq, cudaMemcpyHostToDevice));
        NUSHT_CUDA_TRY(cudaMemcpy(rp->d_bcoff, h_bcoff.data(), sizeof(int64_t) * nq, cudaMemcpyHostToDevice));
        NUSHT_CUDA_TRY(cudaMemcpy(rp->d_bpix, h_bpix.data(), sizeof(int64_t) * nq, cudaMemcpyHostToDevice));
        NUSHT_TRY(r_alloc(&rp->d_bwork, sizeof(double2) * (size_t)wtot, rp));
        NUSHT_TRY(r_alloc(&rp->d_bspec, sizeof(double2) * (size_t)btot, rp));
        NUSHT_TRY(r_alloc(&rp->d_bchirp, sizeof(double2) * (size_t)ctot, rp));
        // chirp tables, then their spectra: the distinct lengths of a group fill the first rows of the group's work
        // block, the group's own plan transforms the block, the rows are kept
        for (const auto& d : distinct) {
            k_blue_chirp<<<(d.n + 255) / 256, 256>>>(d.n, rp->d_bchirp + d.coff);
            NUSHT_CUDA_TRY(nusht_launched());
        }
        size_t di = 0;
        for (auto& g : rp->groups) {
            NUSHT_CUFFT_TRY(cufftSetWorkArea(g.z2z, rp->d_fftwork));
            double2* block = rp->d_bwork + g.woff;
            NUSHT_CUDA_TRY(cudaMemset(block, 0, sizeof(double2) * (size_t)g.count * (size_t)g.P));
            const size_t d0 = di;
            for (; di < distinct.size() && distinct[di].P == g.P; ++di) {
                k_blue_kernel_row<<<(g.P + 255) / 256, 256>>>(distinct[di].n, g.P, rp->d_bchirp + distinct[di].coff,
                                                               block + (di - d0) * (size_t)g.P);
                NUSHT_CUDA_TRY(nusht_launched());
            }
            NUSHT_CUFFT_TRY(cufftSetStream(g.z2z, 0));
            NUSHT_CUFFT_TRY(cufftExecZ2Z(g.z2z, (cufftDoubleComplex*)block, (cufftDoubleComplex*)block, CUFFT_FORWARD));
            NUSHT_CUDA_TRY(cudaMemcpy(rp->d_bspec + distinct[d0].boff, block, sizeof(double2) * (di - d0) * (size_t)g.P,
                                      cudaMemcpyDeviceToDevice));
        }
    }
    {
        size_t smax = 0;
        for (const auto& run : rp->runs)
            if (run.staged) smax = std::max(smax, (size_t)run.count * (size_t)run.nphi * (f64 ? 8 : 4));
        if (smax) NUSHT_TRY(r_alloc(&rp->d_stage, smax, rp));
    }
    for (auto& kv : rp->fft) {
        NUSHT_CUFFT_TRY(cufftSetWorkArea(kv.second.first, rp->d_fftwork));
        NUSHT_CUFFT_TRY(cufftSetWorkArea(kv.second.second, rp->d_fftwork));
    }
    NUSHT_CUDA_TRY(cudaDeviceSynchronize());
    return NUSHT_OK;
}

extern "C" int nusht_ring_plan(nusht_ring_plan_t** out, int lmax, int mmax, int nrings, const double* theta,
                               const int64_t* nphi, const double* phi0, const double* weight, int dtype) {
    if (!out) return NUSHT_ERR_INVALID_ARG;
    *out = nullptr;
    if (lmax < 0 || mmax < 0 || mmax > lmax || nrings < 1 || !theta || !nphi) return NUSHT_ERR_INVALID_ARG;
    if (dtype != NUSHT_F64 && dtype != NUSHT_F32) return NUSHT_ERR_INVALID_ARG;
    if (lmax > 32000) return NUSHT_ERR_UNSUPPORTED;
    int64_t npix = 0;
    for (int r = 0; r < nrings; ++r) {
        if (!(theta[r] >= 0.0) || !(theta[r] <= 3.14159265358979323846)) return NUSHT_ERR_BAD_POINTS;
        if (phi0 && !isfinite(phi0[r])) return NUSHT_ERR_BAD_POINTS;
        if (weight && !isfinite(weight[r])) return NUSHT_ERR_INVALID_ARG;
        if (nphi[r] < 1 || nphi[r] > (1 << 21)) return NUSHT_ERR_INVALID_ARG;   // (grid.y of k_ring_spec_syn: n/64 blocks)
        npix += nphi[r];
    }
    const auto t0 = std::chrono::steady_clock::now();
    nusht_ring_plan_s* rp = new (std::nothrow) nusht_ring_plan_s();
    if (!rp) return NUSHT_ERR_ALLOC;
    rp->lmax = lmax;
    rp->mmax = mmax;
    rp->dtype = dtype;
    rp->nrings = nrings;
    const int st = ring_build(rp, theta, nphi, phi0, weight);
    if (st != NUSHT_OK) {
        ring_release(rp);
        return st;
    }
    rp->plan_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
    *out = rp;
    return NUSHT_OK;
}

extern "C" int nusht_ring_destroy(nusht_ring_plan_t* rp) {
    ring_release(rp);
    return NUSHT_OK;
}

extern "C" int nusht_ring_info(const nusht_ring_plan_t* rp, nusht_ring_info_t* info) {
    if (!rp || !info) return NUSHT_ERR_INVALID_ARG;
    memset(info, 0, sizeof(*info));
    info->lmax = rp->lmax;
    info->mmax = rp->mmax;
    info->dtype = rp->dtype;
    info->nrings = rp->nrings;
    info->npairs = rp->core.lg.npairs;
    info->nruns = (int)(rp->runs.size() + rp->groups.size());     // batched FFT plans: long runs + pool groups
    info->npix = rp->npix;
    info->nlm = rp->core.nlm;
    info->workspace_bytes = rp->workspace_bytes;
    info->plan_ms = rp->plan_ms;
    return NUSHT_OK;
}

static BlueMeta blue_meta(const nusht_ring_plan_s* rp) {
    BlueMeta B;
    B.ring = rp->d_bring; B.P = rp->d_bP; B.woff = rp->d_bwoff; B.boff = rp->d_bboff; B.coff = rp->d_bcoff;
    B.pixoff = rp->d_bpix; B.nphi = rp->d_nphi; B.zoff = rp->d_zoff;
    return B;
}

// the two batched FFTs of the pool with the chirp-spectrum product between them (work array in place)
static int blue_convolve(nusht_ring_plan_s* rp, bool analysis, cudaStream_t s) {
    const BlueMeta B = blue_meta(rp);
    const dim3 grid(rp->npool, (rp->pool_maxP + 255) / 256);
    for (auto& g : rp->groups) {
        cufftDoubleComplex* block = (cufftDoubleComplex*)(rp->d_bwork + g.woff);
        NUSHT_CUFFT_TRY(cufftSetStream(g.z2z, s));
        NUSHT_CUFFT_TRY(cufftExecZ2Z(g.z2z, block, block, CUFFT_FORWARD));
    }
    if (analysis) k_blue_mul<true><<<grid, 256, 0, s>>>(B, rp->d_bspec, rp->d_bwork);
    else k_blue_mul<false><<<grid, 256, 0, s>>>(B, rp->d_bspec, rp->d_bwork);
    NUSHT_CUDA_TRY(nusht_launched());
    for (auto& g : rp->groups) {
        cufftDoubleComplex* block = (cufftDoubleComplex*)(rp->d_bwork + g.woff);
        NUSHT_CUFFT_TRY(cufftExecZ2Z(g.z2z, block, block, CUFFT_INVERSE));
    }
    return NUSHT_OK;
}

static RingMeta ring_meta(const nusht_ring_plan_s* rp, const double* scale) {
    RingMeta R;
    R.nphi = rp->d_nphi;
    R.zoff = rp->d_zoff;
    R.phi0 = rp->d_phi0;
    R.scale = scale;
    R.nrings = rp->nrings;
    R.M = rp->mmax;
    R.stride = rp->nrings;
    R.small_below = 0;
    R.small = rp->d_small;
    return R;
}

// F[m][ring] -> pixels
static int ring_phi_synthesis(nusht_ring_plan_s* rp, const double* scale, void* map, cudaStream_t s) {
    const bool f64 = rp->dtype == NUSHT_F64;
    RingMeta R = ring_meta(rp, scale);
    if (rp->nsmall) R.small_below = RING_SMALL;
    const dim3 grid((rp->nrings + 31) / 32, (rp->max_nphi / 2 + 1 + 31) / 32);
    if (f64) k_ring_spec_syn<double2><<<grid, 256, 0, s>>>(R, rp->core.d_ft, (double2*)rp->d_z);
    else k_ring_spec_syn<float2><<<grid, 256, 0, s>>>(R, rp->core.d_ft, (float2*)rp->d_z);
    NUSHT_CUDA_TRY(nusht_launched());
    if (rp->nsmall) {
        const size_t smem = RING_SMALL_MODES * sizeof(double2);
        if (f64) k_ring_spec_syn_small<double2><<<rp->nsmall, 256, smem, s>>>(R, rp->core.d_ft, (double2*)rp->d_z);
        else k_ring_spec_syn_small<float2><<<rp->nsmall, 256, smem, s>>>(R, rp->core.d_ft, (float2*)rp->d_z);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    const size_t esz = f64 ? 8 : 4;
    for (const auto& run : rp->runs) {
        NUSHT_CUFFT_TRY(cufftSetStream(run.c2r, s));
        void* dst = run.staged ? rp->d_stage : (void*)((char*)map + (size_t)run.pixoff * esz);
        if (f64)
            NUSHT_CUFFT_TRY(cufftExecZ2D(run.c2r, (cufftDoubleComplex*)rp->d_z + run.zoff, (double*)dst));
        else
            NUSHT_CUFFT_TRY(cufftExecC2R(run.c2r, (cufftComplex*)rp->d_z + run.zoff, (float*)dst));
        if (run.staged)
            NUSHT_CUDA_TRY(cudaMemcpyAsync((char*)map + (size_t)run.pixoff * esz, rp->d_stage,
                                           (size_t)run.count * run.nphi * esz, cudaMemcpyDeviceToDevice, s));
    }
    if (rp->npool) {
        const BlueMeta B = blue_meta(rp);
        const dim3 bgrid(rp->npool, (rp->pool_maxP + 255) / 256);
        if (f64) k_blue_pre_syn<double2><<<bgrid, 256, 0, s>>>(B, (const double2*)rp->d_z, rp->d_bchirp, rp->d_bwork);
        else k_blue_pre_syn<float2><<<bgrid, 256, 0, s>>>(B, (const float2*)rp->d_z, rp->d_bchirp, rp->d_bwork);
        NUSHT_CUDA_TRY(nusht_launched());
        NUSHT_TRY(blue_convolve(rp, false, s));
        if (f64) k_blue_post_syn<double><<<bgrid, 256, 0, s>>>(B, rp->d_bwork, rp->d_bchirp, (double*)map);
        else k_blue_post_syn<float><<<bgrid, 256, 0, s>>>(B, rp->d_bwork, rp->d_bchirp, (float*)map);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    return NUSHT_OK;
}

// pixels -> G[m][ring] (times scale_r)
static int ring_phi_analysis(nusht_ring_plan_s* rp, const double* scale, const void* map, cudaStream_t s) {
    const bool f64 = rp->dtype == NUSHT_F64;
    const size_t esz = f64 ? 8 : 4;
    for (const auto& run : rp->runs) {
        NUSHT_CUFFT_TRY(cufftSetStream(run.r2c, s));
        const void* src = (const char*)map + (size_t)run.pixoff * esz;
        if (run.staged) {
            NUSHT_CUDA_TRY(cudaMemcpyAsync(rp->d_stage, src, (size_t)run.count * run.nphi * esz, cudaMemcpyDeviceToDevice, s));
            src = rp->d_stage;
        }
        if (f64)
            NUSHT_CUFFT_TRY(cufftExecD2Z(run.r2c, (double*)src, (cufftDoubleComplex*)rp->d_z + run.zoff));
        else
            NUSHT_CUFFT_TRY(cufftExecR2C(run.r2c, (float*)src, (cufftComplex*)rp->d_z + run.zoff));
    }
    if (rp->npool) {
        const BlueMeta B = blue_meta(rp);
        const dim3 bgrid(rp->npool, (rp->pool_maxP + 255) / 256);
        if (f64) k_blue_pre_ana<double><<<bgrid, 256, 0, s>>>(B, (const double*)map, rp->d_bchirp, rp->d_bwork);
        else k_blue_pre_ana<float><<<bgrid, 256, 0, s>>>(B, (const float*)map, rp->d_bchirp, rp->d_bwork);
        NUSHT_CUDA_TRY(nusht_launched());
        NUSHT_TRY(blue_convolve(rp, true, s));
        if (f64) k_blue_post_ana<double2><<<bgrid, 256, 0, s>>>(B, rp->d_bwork, rp->d_bchirp, (double2*)rp->d_z);
        else k_blue_post_ana<float2><<<bgrid, 256, 0, s>>>(B, rp->d_bwork, rp->d_bchirp, (float2*)rp->d_z);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    const RingMeta R = ring_meta(rp, scale);
    const dim3 grid((rp->nrings + 31) / 32, (rp->mmax + 32) / 32);
    if (f64) k_ring_spec_adj<double2><<<grid, 256, 0, s>>>(R, (const double2*)rp->d_z, rp->core.d_ft);
    else k_ring_spec_adj<float2><<<grid, 256, 0, s>>>(R, (const float2*)rp->d_z, rp->core.d_ft);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}

extern "C" int nusht_ring_synthesis(nusht_ring_plan_t* rp, const void* alm, void* map, void* stream) {
    if (!rp || !alm || !map || ((uintptr_t)map & 15)) return NUSHT_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    rp->core.lmax_io = rp->lmax;
    NUSHT_TRY(legendre_alm_prep(&rp->core, alm, s));
    NUSHT_TRY(legendre_synthesis(&rp->core, rp->core.d_ft, s));
    return ring_phi_synthesis(rp, nullptr, map, s);
}

extern "C" int nusht_ring_analysis(nusht_ring_plan_t* rp, const void* map, void* alm, void* stream) {
    if (!rp || !alm || !map || ((uintptr_t)map & 15)) return NUSHT_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    rp->core.lmax_io = rp->lmax;
    NUSHT_TRY(ring_phi_analysis(rp, rp->d_weight, map, s));
    NUSHT_TRY(legendre_adjoint(&rp->core, rp->core.d_ft, s));
    return legendre_alm_post(&rp->core, alm, s);
}

extern "C" int nusht_ring_gradient(nusht_ring_plan_t* rp, const void* philm, void* alpha_theta, void* alpha_phi,
                                   void* stream) {
    if (!rp || !philm || !alpha_theta || !alpha_phi) return NUSHT_ERR_INVALID_ARG;
    if (((uintptr_t)alpha_theta & 15) || ((uintptr_t)alpha_phi & 15)) return NUSHT_ERR_INVALID_ARG;
    if (rp->has_pole_ring) return NUSHT_ERR_UNSUPPORTED;       // e_theta, e_phi are undefined at the poles
    cudaStream_t s = (cudaStream_t)stream;
    const bool f64 = rp->dtype == NUSHT_F64;
    const int L = rp->lmax, M = rp->mmax;
    const dim3 grid((L + 2 + 255) / 256, M + 1);
    if (f64) k_grad_coeffs<double><<<grid, 256, 0, s>>>(L, M, (const double*)philm, (double*)rp->d_ga, (double*)rp->d_gb);
    else k_grad_coeffs<float><<<grid, 256, 0, s>>>(L, M, (const float*)philm, (float*)rp->d_ga, (float*)rp->d_gb);
    NUSHT_CUDA_TRY(nusht_launched());
    rp->core.lmax_io = L + 1;
    int st = legendre_alm_prep(&rp->core, rp->d_ga, s);
    if (st == NUSHT_OK) st = legendre_synthesis(&rp->core, rp->core.d_ft, s);
    if (st == NUSHT_OK) st = ring_phi_synthesis(rp, rp->d_isin, alpha_theta, s);
    if (st == NUSHT_OK) st = legendre_alm_prep(&rp->core, rp->d_gb, s);
    if (st == NUSHT_OK) st = legendre_synthesis(&rp->core, rp->core.d_ft, s);
    if (st == NUSHT_OK) st = ring_phi_synthesis(rp, rp->d_isin, alpha_phi, s);
    rp->core.lmax_io = L;
    return st;
}
