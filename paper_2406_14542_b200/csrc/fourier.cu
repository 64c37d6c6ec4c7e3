// fourier.cu -- uniform-FFT part of the nuSHT (operator F and the grid side of N; arXiv
// 2406.14542 Eq. 5-6).
//
// Only the theta FFT of F survives: the phi FFTs of S and F cancel, so the Legendre
// stage hands over Ftilde[m][r] in m-space and
//   a3  c[m,k]  = (1/Ntheta) sum_r Ftilde[m][r] e^{-2 pi i k r/Ntheta},  |k| <= lmax       (cuFFT)
//   a4  B[m][k mod n_theta] = c[m,k] p_theta(k) p_phi(m), zero elsewhere   (deconvolve + zero-pad)
//   a5  H[m][a] = sum_k B[m][k] e^{+2 pi i k a/n_theta}                                  (cuFFT)
//       g[a][b] = sum_m w_m Re(H[m][a] e^{+2 pi i m b/n_phi}),  rows a = 0..n_theta/2   (cuFFT C2R)
// and the adjoint (a9) runs the transposed chain: R2C, zero-extend in theta, forward FFT, truncate
// and deconvolve with the SAME factors, inverse FFT of length Ntheta.
// p(k) = 1/psihat(k): psihat is the Fourier transform of the piecewise-polynomial kernel that the
// interpolation actually evaluates (nufft.cu), so p is exact for that kernel.
// cuFFT is used for the FFTs only; everything else here is our own kernels.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include <cooperative_groups.h>

#include "fft_reg.cuh"
#include "fft_smem.cuh"
#include "nusht_internal.cuh"

namespace {

template <typename T> struct Cplx;
template <> struct Cplx<double> { using type = double2; };
template <> struct Cplx<float> { using type = float2; };

// The fine theta transform of length n_theta has at most n_theta/2 - 1 non-zero inputs (|k| <= lmax,
// n_theta >= 4 lmax + 4), so it is done as TWO transforms of length nh = n_theta/2, each of which cuFFT
// does in one pass through shared memory at the sizes of interest (a 16384-point FP64 transform is two
// passes over HBM):  y[2a'] = sum_k B[k] e^{2 pi i k a'/nh},  y[2a'+1] = sum_k (B[k] e^{2 pi i k/n_theta}) e^{2 pi i k a'/nh}.
// Buffer layout H[m][parity][nh]; rows a = 2a' + parity are re-interleaved by the transposes below.

// a4: deconvolve + wrap into the two length-nh spectra; one thread per slot k' of column m
template <typename T>
__global__ void k_deconv_pad(int L, int M, int nth2, int nh, const double2* __restrict__ ft,
                             const double* __restrict__ pth, const double* __restrict__ pph,
                             typename Cplx<T>::type* __restrict__ h) {
    const int kp = blockIdx.x * blockDim.x + threadIdx.x;
    const int m = blockIdx.y;
    if (kp >= nh) return;
    int k;
    bool in = true;
    if (kp <= L) k = kp;
    else if (kp >= nh - L) k = kp - nh;
    else { k = 0; in = false; }
    typename Cplx<T>::type e, o;
    e.x = e.y = o.x = o.y = 0;
    if (in) {
        const double2 c = ft[(int64_t)m * nth2 + (k >= 0 ? k : k + nth2)];
        const double f = pth[k + L] * pph[m];
        const double cr = c.x * f, ci = c.y * f;
        double sn, cs;
        sincospi((double)k / (double)nh, &sn, &cs);      // e^{2 pi i k / n_theta}
        e.x = (T)cr;
        e.y = (T)ci;
        o.x = (T)(cr * cs - ci * sn);
        o.y = (T)(cr * sn + ci * cs);
    }
    h[((int64_t)m * 2 + 0) * nh + kp] = e;
    h[((int64_t)m * 2 + 1) * nh + kp] = o;
}

// a9: combine the two forward transforms (transpose of the above), truncate to |k| <= lmax and
// deconvolve; one thread per slot r of the doubled-ring spectrum
template <typename T>
__global__ void k_deconv_trunc(int L, int M, int nth2, int nh, const typename Cplx<T>::type* __restrict__ h,
                               const double* __restrict__ pth, const double* __restrict__ pph,
                               double2* __restrict__ ft) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    const int m = blockIdx.y;
    if (r >= nth2) return;
    int k;
    bool in = true;
    if (r <= L) k = r;
    else if (r >= nth2 - L) k = r - nth2;
    else { k = 0; in = false; }
    double2 out = make_double2(0.0, 0.0);
    if (in) {
        const int kp = k >= 0 ? k : k + nh;
        const typename Cplx<T>::type e = h[((int64_t)m * 2 + 0) * nh + kp];
        const typename Cplx<T>::type o = h[((int64_t)m * 2 + 1) * nh + kp];
        double sn, cs;
        sincospi((double)k / (double)nh, &sn, &cs);      // conj twiddle e^{-2 pi i k / n_theta}
        const double f = pth[k + L] * pph[m];
        out.x = ((double)e.x + (double)o.x * cs + (double)o.y * sn) * f;
        out.y = ((double)e.y + (double)o.y * cs - (double)o.x * sn) * f;
    }
    ft[(int64_t)m * nth2 + r] = out;
}

// ---------------------------------------------------------------------------------------------
// General chain (up-sampling sigma != 2, the paper's 1.25: PAPER.md:152).  The two-half-length trick above needs
// n_theta/2 >= 2 lmax + 1 and the half-length real-FFT trick below needs mmax < n_phi/4; neither holds at
// sigma = 1.25, so here the fine theta transform is ONE full-length complex FFT per column and the phi transform a
// real (C2R / R2C) cuFFT out of place between a half-spectrum buffer Z[a][m], m = 0 .. n_phi/2, and the grid rows:
//   synthesis  c[m,k] --(p_theta p_phi, zero-pad)--> H[m][k mod n_theta] --iFFT--> H[m][a] --transpose-->
//              Z[a][m] (a <= n_theta/2; zero for m > mmax) --C2R--> g[a][b]   (the Hermitian extension of the C2R
//              supplies the weights w_m of the real field)
//   adjoint    g --R2C--> Z[a][m] --transpose, zero-extend a > n_theta/2--> H[m][a] --FFT--> truncate, deconvolve.
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void k_deconv_pad_gen(int L, int M, int nth2, int nth, const double2* __restrict__ ft,
                                 const double* __restrict__ pth, const double* __restrict__ pph,
                                 typename Cplx<T>::type* __restrict__ h) {
    const int kp = blockIdx.x * blockDim.x + threadIdx.x;
    const int m = blockIdx.y;
    if (kp >= nth) return;
    int k;
    bool in = true;
    if (kp <= L) k = kp;
    else if (kp >= nth - L) k = kp - nth;
    else { k = 0; in = false; }
    typename Cplx<T>::type v;
    v.x = v.y = 0;
    if (in) {
        const double2 c = ft[(int64_t)m * nth2 + (k >= 0 ? k : k + nth2)];
        const double f = pth[k + L] * pph[m];
        v.x = (T)(c.x * f);
        v.y = (T)(c.y * f);
    }
    h[(int64_t)m * nth + kp] = v;
}

template <typename T>
__global__ void k_deconv_trunc_gen(int L, int M, int nth2, int nth, const typename Cplx<T>::type* __restrict__ h,
                                   const double* __restrict__ pth, const double* __restrict__ pph,
                                   double2* __restrict__ ft) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    const int m = blockIdx.y;
    if (r >= nth2) return;
    int k;
    bool in = true;
    if (r <= L) k = r;
    else if (r >= nth2 - L) k = r - nth2;
    else { k = 0; in = false; }
    double2 out = make_double2(0.0, 0.0);
    if (in) {
        const typename Cplx<T>::type v = h[(int64_t)m * nth + (k >= 0 ? k : k + nth)];
        const double f = pth[k + L] * pph[m];
        out.x = (double)v.x * f;
        out.y = (double)v.y * f;
    }
    ft[(int64_t)m * nth2 + r] = out;
}

// H[m][a] -> Z[a][m], rows a < nrow_half; columns mmax < m <= n_phi/2 are zeroed, Im Z[a][0] := 0 (a real row)
template <typename C>
__global__ void __launch_bounds__(256)
k_h_to_zc(int M, int nth, int nrow_half, int nzc, const C* __restrict__ h, C* __restrict__ z) {
    __shared__ C tile[32][33];
    const int a0 = blockIdx.x * 32, m0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int m = m0 + r, a = a0 + tx;
        if (m <= M && a < nrow_half) tile[r][tx] = h[(int64_t)m * nth + a];
    }
    __syncthreads();
    C zero;
    zero.x = 0;
    zero.y = 0;
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int a = a0 + r, m = m0 + tx;
        if (a >= nrow_half || m >= nzc) continue;
        C v = (m <= M) ? tile[tx][r] : zero;
        if (m == 0) v.y = 0;
        z[(int64_t)a * nzc + m] = v;
    }
}

// Z[a][m] -> H[m][a] for a < nrow_half, H[m][a] = 0 for the rest of the theta period (transpose of "keep rows 0 .. n_theta/2")
template <typename C>
__global__ void __launch_bounds__(256)
k_zc_to_h(int M, int nth, int nrow_half, int nzc, const C* __restrict__ z, C* __restrict__ h) {
    __shared__ C tile[32][33];
    const int a0 = blockIdx.x * 32, m0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int a = a0 + r, m = m0 + tx;
        if (a < nrow_half && m <= M) tile[r][tx] = z[(int64_t)a * nzc + m];
    }
    __syncthreads();
    C zero;
    zero.x = 0;
    zero.y = 0;
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int m = m0 + r, a = a0 + tx;
        if (m > M || a >= nth) continue;
        h[(int64_t)m * nth + a] = (a < nrow_half) ? tile[tx][r] : zero;
    }
}

// a5 / a9, phi pass.  The real transform of length N = n_phi on row a is done as ONE complex transform of
// length N/2 on the row itself (the real row viewed as N/2 complex numbers x[2j] + i x[2j+1]), with the
// usual pre-/post-processing of a real FFT fused into the transposes between the theta-pass layout
// H[m][parity][a'] (a = 2a' + parity) and the grid rows:
//   synthesis:  Z[k] = (X[k] + conj X[N/2-k]) + i W^k (X[k] - conj X[N/2-k]),  W = e^{2 pi i/N},  X[k] = H_a[k] for
//               k <= mmax < N/4 and 0 otherwise, so Z[m] = X[m] (1 + i W^m), Z[N/2-m] = conj(X[m]) (1 - i W^{N/2-m});
//               the inverse transform of Z is x[2j] + i x[2j+1] with x[n] = sum_m w_m Re(X[m] W^{mn}).
//   adjoint:    Zf = forward transform of the row;  Y[m] = (Zf[m] + conj Zf[N/2-m])/2 - (i/2) W^{-m} (Zf[m] - conj Zf[N/2-m])
//               = sum_n x[n] W^{-mn}  for m <= mmax.
// 32 x 32 tiles through shared memory; only rows a <= n_theta/2 (theta in [0, pi]) and columns m <= mmax.
template <typename C>
__global__ void __launch_bounds__(256)
k_h_to_z(int M, int nh, int nrow_half, int nz, const double2* __restrict__ tw, const C* __restrict__ h,
         C* __restrict__ z) {
    __shared__ C tile[32][33];
    const int nblk = (nh + 31) / 32;
    const int par = blockIdx.x / nblk, ap0 = (blockIdx.x % nblk) * 32, m0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int m = m0 + r, ap = ap0 + tx;
        if (m <= M && ap < nh && 2 * ap + par < nrow_half) tile[r][tx] = h[((int64_t)m * 2 + par) * nh + ap];
    }
    __syncthreads();
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int a = 2 * (ap0 + r) + par, m = m0 + tx;
        if (ap0 + r >= nh || a >= nrow_half) continue;
        C* row = z + (int64_t)a * nz;
        if (m <= M) {
            const C x = tile[tx][r];
            const double2 w = tw[m];      // W^m = (cos, sin)
            const double xr = x.x, xi = x.y;
            C v;
            if (m == 0) {                 // X[0] is real for a real row; its imaginary part is ignored
                v.x = x.x;
                v.y = x.x;
                row[0] = v;
            } else {
                v.x = xr * (1.0 - w.y) - xi * w.x;
                v.y = xr * w.x + xi * (1.0 - w.y);
                row[m] = v;
                v.x = xr * (1.0 + w.y) + xi * w.x;
                v.y = xr * w.x - xi * (1.0 + w.y);
                row[nz - m] = v;
            }
        }
        if (blockIdx.y == 0) {            // columns mmax+1 .. N/2-mmax-1 carry no mode
            C zero;
            zero.x = 0;
            zero.y = 0;
            for (int k = M + 1 + tx; k <= nz - M - 1; k += 32) row[k] = zero;
        }
    }
}

// adjoint: post-processing of the forward transform + transpose + zero-extension of the theta axis to the
// full period (the transpose of "keep rows 0 .. n_theta/2")
template <typename C>
__global__ void __launch_bounds__(256)
k_z_to_h(int M, int nh, int nrow_half, int nz, bool write_ext, const double2* __restrict__ tw,
         const C* __restrict__ z, C* __restrict__ h) {
    __shared__ C ta[32][33], tb[32][33];
    const int nblk = (nh + 31) / 32;
    const int par = blockIdx.x / nblk, ap0 = (blockIdx.x % nblk) * 32, m0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int a = 2 * (ap0 + r) + par, m = m0 + tx;
        if (m <= M && a < nrow_half) {
            const C* row = z + (int64_t)a * nz;
            ta[r][tx] = row[m];
            tb[r][tx] = row[m == 0 ? 0 : nz - m];
        }
    }
    __syncthreads();
    C zero;
    zero.x = 0;
    zero.y = 0;
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int m = m0 + r, ap = ap0 + tx;
        if (m > M || ap >= nh) continue;
        C out = zero;
        if (2 * ap + par >= nrow_half && !write_ext) continue;   // the fused theta chain never reads the extension
        if (2 * ap + par < nrow_half) {
            const C A = ta[tx][r], Bc = tb[tx][r];
            const double2 w = tw[m];
            const double bx = Bc.x, by = -(double)Bc.y;          // B = conj Zf[N/2 - m]
            const double dx = (double)A.x - bx, dy = (double)A.y - by;
            out.x = 0.5 * (((double)A.x + bx) + (w.x * dy - w.y * dx));
            out.y = 0.5 * (((double)A.y + by) - (w.x * dx + w.y * dy));
        }
        h[((int64_t)m * 2 + par) * nh + ap] = out;
    }
}

// ---------------------------------------------------------------------------------------------
// Fused theta chains (a3 + a4 + a5-theta, and the theta part of a9), used when the coarse and the
// half fine length coincide (N = Ntheta = n_theta/2, a power of two <= 8192: sigma = 2 at the
// BASELINE sizes).  One CTA per m keeps the column in shared memory (fft_smem.cuh):
//   synthesis  Ftilde[m][.] --FFT--> c[m,k] --(p_theta p_phi, |k| <= lmax)--> registers
//              --(parity 0: as is; parity 1: e^{2 pi i k/n_theta})--> inverse FFT --> H[m][parity][a'],
//              storing only the rows a = 2a' + parity <= n_theta/2 that the phi pass reads;
//   adjoint    the transposed chain: H[m][parity][a'] (zero beyond n_theta/2) --FFT--> combine the
//              parities, truncate, deconvolve --> inverse FFT --> Gtilde[m][.].
// HBM traffic per column: N complex in, ~N complex out (the cuFFT chain it replaces moves 9 N).
// ---------------------------------------------------------------------------------------------
#ifndef NUSHT_CHAIN_DIV
#define NUSHT_CHAIN_DIV 16
#endif
constexpr int chain_threads(int n) { return n >= 32 * NUSHT_CHAIN_DIV ? n / NUSHT_CHAIN_DIV : 32; }

template <int N>
struct ChainCfg {
    static constexpr int T = chain_threads(N);          // threads per CTA: one radix-16 butterfly per thread and stage
    static constexpr int E = N / T;                     // spectrum entries held per thread
    static constexpr size_t SMEM = sizeof(double2) * (size_t)fftsm::padded_len(N);
};

// plan-time tables of the fused chains (one allocation, see fourier_build)
struct ChainTables {
    const double2* tw2;     // exp(-2 pi i i/N), i < N/2: the fused radix-2 stage
    const double2* stw;     // per-stage twiddles (fftsm::stage_table_offset)
    const double* fpos;     // p_theta(k(p)) for |k(p)| <= lmax, else 0, at digit-reversed position p
    const double2* twpar;   // exp(+2 pi i k(p)/(2N)): the parity-1 shift, at position p
};

template <int N, int SIGN>
struct DevExec {
    double2* s;
    const double2* stw;
    int tid;
    template <int R, int NS>
    __device__ __forceinline__ void dif() {
        fftsm::stage_dif<N, R, NS, SIGN>(s, tid, ChainCfg<N>::T, stw + fftsm::stage_table_offset(N, NS));
        __syncthreads();
    }
    template <int R, int NS>
    __device__ __forceinline__ void dit() {
        fftsm::stage_dit<N, R, NS, SIGN>(s, tid, ChainCfg<N>::T, stw + fftsm::stage_table_offset(N, NS));
        __syncthreads();
    }
};

// L2 prefetch of the next column while the current one is transformed (one CTA per SM: nothing else overlaps HBM)
__device__ __forceinline__ void prefetch_l2(const void* ptr, int bytes, int tid, int T) {
    for (int o = tid * 4096; o < bytes; o += T * 4096) {
        const int n = min(4096, bytes - o);
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"((const char*)ptr + o), "r"(n) : "memory");
    }
}

// Column pairs.  Ftilde_m has the DFS symmetry Ftilde_m[N - r] = (-1)^m Ftilde_m[r], which every step of the chain
// preserves: c[m,-k] = (-1)^m c[m,k], and the fine rows obey g_m[-a] = (-1)^m g_m[a].  An even
// column m and its odd neighbour m + 1 therefore go through the chain TOGETHER, as x = p_phi(m) Ftilde_m +
// p_phi(m+1) Ftilde_{m+1} (one forward and two inverse transforms per PAIR instead of three per column), and are
// separated at the end by their parity under a -> -a:  y_m = (u[a'] + u[mirror a']) / 2,  y_{m+1} = (u[a'] -
// u[mirror a']) / 2, with mirror a' = N - a' on the even fine rows and N - 1 - a' on the odd ones.  No division by a
// small number occurs anywhere (unlike the usual cosine-transform-by-FFT trick).  The adjoint kernel is the exact
// transpose: it builds the full-length u from the two half-length inputs, and both output columns receive the same
// transformed sequence (times their p_phi); the component of the neighbour it contains has the opposite symmetry
// and cancels in the fold Gtilde[k] + (-1)^m Gtilde[N - k] that the adjoint Legendre kernel starts with (a10).
// The factor 1/2 is folded into the deconvolution table.
template <int N, typename C>
__global__ void __launch_bounds__(ChainCfg<N>::T)
k_theta_chain_syn(int L, int M, int nrow_half, const double2* __restrict__ ft, const double* __restrict__ pph,
                  const ChainTables tb, C* __restrict__ h) {
    using namespace fftsm;
    constexpr int T = ChainCfg<N>::T, E = ChainCfg<N>::E, RL = last_radix(N / 2);
    extern __shared__ __align__(16) double2 s_col[];
    const int tid = threadIdx.x;
    const int npair = M / 2 + 1;
    for (int mp = blockIdx.x; mp < npair; mp += gridDim.x) {
        const int ma = 2 * mp, mb = 2 * mp + 1;
        const bool has_b = mb <= M;
        const double2* cola = ft + (int64_t)ma * N;
        const double2* colb = ft + (int64_t)(has_b ? mb : ma) * N;
        if (mp + (int)gridDim.x < npair) {
            const int ncol = (2 * (mp + (int)gridDim.x) + 1 <= M) ? 2 : 1;
            prefetch_l2(cola + 2 * (int64_t)gridDim.x * N, ncol * N * (int)sizeof(double2), tid, T);
        }
        const double pa = pph[ma], pb = has_b ? pph[mb] : 0.0;
        __syncthreads();   // previous pair's stores have read s_col
        // a3: forward transform of the pair; its radix-2 stage is fused with the load (unrolled: 16 loads in flight)
#pragma unroll 4
        for (int i = tid; i < N / 2; i += T) {
            const double2 a0 = cola[i], a1 = cola[i + N / 2], b0 = colb[i], b1 = colb[i + N / 2];
            const double2 a = make_double2(fma(pb, b0.x, pa * a0.x), fma(pb, b0.y, pa * a0.y));
            const double2 b = make_double2(fma(pb, b1.x, pa * a1.x), fma(pb, b1.y, pa * a1.y));
            s_col[pad(i)] = make_double2(a.x + b.x, a.y + b.y);
            s_col[pad(i + N / 2)] = cmul(make_double2(a.x - b.x, a.y - b.y), tb.tw2[i]);
        }
        __syncthreads();
        DevExec<N, -1> fwd{s_col, tb.stw, tid};
        forward_stages<N / 2>(fwd);
        // a4: deconvolve and truncate.  The last forward stage leaves the spectrum in registers (entry e of
        // thread tid sits at digit-reversed position RL (tid + T (e / RL)) + e % RL; tables are laid out [e][tid])
        double2 c[E];
        last_stage_to_regs<N, RL, -1, E>(s_col, tid, T, c);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double f = tb.fpos[e * T + tid];     // p_theta(k) / (2 Ntheta), zero outside |k| <= lmax
            c[e] = make_double2(c[e].x * f, c[e].y * f);
        }
        // a5 (theta): rows a = 2a' + parity, one inverse transform of the pair per parity
#pragma unroll 1
        for (int par = 0; par < 2; ++par) {
            __syncthreads();
            if (par) {   // the spectrum is not needed again after parity 1: twiddle it in place
#pragma unroll
                for (int e = 0; e < E; ++e) c[e] = cmul(c[e], tb.twpar[e * T + tid]);
            }
            first_stage_from_regs<N, RL, +1, E>(s_col, tid, T, c);
            __syncthreads();
            DevExec<N, +1> inv{s_col, tb.stw, tid};
            inverse_stages<N / 2>(inv);
            for (int i = tid; i < N / 2; i += T) {     // last inverse stage, in place (a thread owns its two slots)
                const double2 z0 = s_col[pad(i)], z1 = cmul(s_col[pad(i + N / 2)], cconj(tb.tw2[i]));
                s_col[pad(i)] = make_double2(z0.x + z1.x, z0.y + z1.y);
                s_col[pad(i + N / 2)] = make_double2(z0.x - z1.x, z0.y - z1.y);
            }
            __syncthreads();
            // separate the two columns by their mirror parity; only rows a = 2a' + par < nrow_half are stored
            C* outa = h + ((int64_t)ma * 2 + par) * N;
            C* outb = h + ((int64_t)mb * 2 + par) * N;
            for (int ap = tid; 2 * ap + par < nrow_half && ap < N; ap += T) {
                const int mir = par ? N - 1 - ap : (ap == 0 ? 0 : N - ap);
                const double2 u = s_col[pad(ap)], v = s_col[pad(mir)];
                C va, vb;
                va.x = u.x + v.x;
                va.y = u.y + v.y;
                vb.x = u.x - v.x;
                vb.y = u.y - v.y;
                outa[ap] = va;
                if (has_b) outb[ap] = vb;
            }
        }
    }
}

template <int N, typename C>
__global__ void __launch_bounds__(ChainCfg<N>::T)
k_theta_chain_adj(int L, int M, int nrow_half, const C* __restrict__ h, const double* __restrict__ pph,
                  const ChainTables tb, double2* __restrict__ ft) {
    using namespace fftsm;
    constexpr int T = ChainCfg<N>::T, E = ChainCfg<N>::E, RL = last_radix(N / 2);
    extern __shared__ __align__(16) double2 s_col[];
    const int tid = threadIdx.x;
    const int npair = M / 2 + 1;
    auto ld = [](const C* ptr, int idx) {
        const C v = ptr[idx];
        return make_double2((double)v.x, (double)v.y);
    };
    for (int mp = blockIdx.x; mp < npair; mp += gridDim.x) {
        const int ma = 2 * mp, mb = 2 * mp + 1;
        const bool has_b = mb <= M;
        if (mp + (int)gridDim.x < npair) {
            const C* nxt = h + ((int64_t)(ma + 2 * gridDim.x) * 2) * N;
            const int rows = min(N, (nrow_half + 1) / 2);
            const int nblk = (ma + 2 * (int)gridDim.x + 1 <= M) ? 4 : 2;
            for (int q = 0; q < nblk; ++q) prefetch_l2(nxt + (int64_t)q * N, rows * (int)sizeof(C), tid, T);
        }
        double2 acc[E];
#pragma unroll
        for (int e = 0; e < E; ++e) acc[e] = make_double2(0.0, 0.0);
#pragma unroll 1
        for (int par = 0; par < 2; ++par) {
            const C* ina = h + ((int64_t)ma * 2 + par) * N;
            const C* inb = h + ((int64_t)(has_b ? mb : ma) * 2 + par) * N;
            const double sb = has_b ? 1.0 : 0.0;
            __syncthreads();
            // transpose of the separation: u[j] = ha[j] + hb[j] (j below the mirror point), ha[mirror j] - hb[mirror j]
            // above it, 2 ha at the self-mirrored rows 0 and N/2 of parity 0; rows beyond nrow_half do not exist (N is
            // the half fine length, nrow_half = N + 1).  The radix-2 stage of the forward transform is fused in.
#pragma unroll 4
            for (int i = tid; i < N / 2; i += T) {
                double2 a, b;
                if (par == 0) {
                    const double2 xa = ld(ina, i), xb = ld(inb, i);
                    const double2 ya = ld(ina, N / 2 - i), yb = ld(inb, N / 2 - i);
                    a = i == 0 ? make_double2(2.0 * xa.x, 2.0 * xa.y) : make_double2(fma(sb, xb.x, xa.x), fma(sb, xb.y, xa.y));
                    b = i == 0 ? make_double2(2.0 * ya.x, 2.0 * ya.y) : make_double2(fma(-sb, yb.x, ya.x), fma(-sb, yb.y, ya.y));
                } else {
                    const double2 xa = ld(ina, i), xb = ld(inb, i);
                    const double2 ya = ld(ina, N / 2 - 1 - i), yb = ld(inb, N / 2 - 1 - i);
                    a = make_double2(fma(sb, xb.x, xa.x), fma(sb, xb.y, xa.y));
                    b = make_double2(fma(-sb, yb.x, ya.x), fma(-sb, yb.y, ya.y));
                }
                s_col[pad(i)] = make_double2(a.x + b.x, a.y + b.y);
                s_col[pad(i + N / 2)] = cmul(make_double2(a.x - b.x, a.y - b.y), tb.tw2[i]);
            }
            __syncthreads();
            DevExec<N, -1> fwd{s_col, tb.stw, tid};
            forward_stages<N / 2>(fwd);
            double2 v[E];
            last_stage_to_regs<N, RL, -1, E>(s_col, tid, T, v);
#pragma unroll
            for (int e = 0; e < E; ++e) {
                if (par) v[e] = cmul(v[e], cconj(tb.twpar[e * T + tid]));
                acc[e].x += v[e].x;
                acc[e].y += v[e].y;
            }
        }
        __syncthreads();
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double f = tb.fpos[e * T + tid];
            acc[e] = make_double2(acc[e].x * f, acc[e].y * f);
        }
        first_stage_from_regs<N, RL, +1, E>(s_col, tid, T, acc);
        __syncthreads();
        DevExec<N, +1> inv{s_col, tb.stw, tid};
        inverse_stages<N / 2>(inv);
        const double pa = pph[ma], pb = has_b ? pph[mb] : 0.0;
        double2* outa = ft + (int64_t)ma * N;
        double2* outb = ft + (int64_t)mb * N;
        for (int i = tid; i < N / 2; i += T) {
            const double2 z0 = s_col[pad(i)], z1 = cmul(s_col[pad(i + N / 2)], cconj(tb.tw2[i]));
            const double2 x0 = make_double2(z0.x + z1.x, z0.y + z1.y), x1 = make_double2(z0.x - z1.x, z0.y - z1.y);
            outa[i] = make_double2(pa * x0.x, pa * x0.y);
            outa[i + N / 2] = make_double2(pa * x1.x, pa * x1.y);
            if (has_b) {
                outb[i] = make_double2(pb * x0.x, pb * x0.y);
                outb[i + N / 2] = make_double2(pb * x1.x, pb * x1.y);
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Cluster-pair variant of the fused chains.  After the radix-2 stage that is fused with the load, the even- and
// the odd-frequency half of a column are independent transforms of length H = N/2 all the way to the last
// (radix-2) stage of the inverse transform.  Two CTAs of a thread-block cluster take one half each (68 KB of
// shared memory at N = 8192: two or three independent CTAs per SM whose load / stage / store phases overlap,
// where the single-CTA kernel holds an SM alone; and a 16384-point FP64 column, which no single SM can hold,
// fits as two halves), and combine the halves in that last stage through distributed shared memory.
// ---------------------------------------------------------------------------------------------
constexpr int half_threads(int h) { return h >= 512 ? h / 16 : 32; }

template <int N>
struct HalfCfg {
    static constexpr int H = N / 2;
    static constexpr int T = half_threads(H);
    static constexpr int E = H / T;
    static constexpr size_t SMEM = sizeof(double2) * (size_t)fftsm::padded_len(H);
    static constexpr int CTAS = 512 / T > 8 ? 8 : 512 / T;   // CTAs per SM at 128 registers per thread
};

template <int N, int SIGN>
struct HalfExec {   // stages on ONE half (array length N/2); stage tables are those of the full length N
    double2* s;
    const double2* stw;
    int tid;
    template <int R, int NS>
    __device__ __forceinline__ void dif() {
        fftsm::stage_dif<N / 2, R, NS, SIGN>(s, tid, HalfCfg<N>::T, stw + fftsm::stage_table_offset(N, NS));
        __syncthreads();
    }
    template <int R, int NS>
    __device__ __forceinline__ void dit() {
        fftsm::stage_dit<N / 2, R, NS, SIGN>(s, tid, HalfCfg<N>::T, stw + fftsm::stage_table_offset(N, NS));
        __syncthreads();
    }
};

template <int N, typename C>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(HalfCfg<N>::T, HalfCfg<N>::CTAS)
k_theta_chain2_syn(int L, int M, int nrow_half, const double2* __restrict__ ft, const double* __restrict__ pph,
                   const ChainTables tb, C* __restrict__ h) {
    using namespace fftsm;
    namespace cg = cooperative_groups;
    constexpr int H = HalfCfg<N>::H, T = HalfCfg<N>::T, E = HalfCfg<N>::E, RL = last_radix(H);
    extern __shared__ __align__(16) double2 s_col[];
    cg::cluster_group cluster = cg::this_cluster();
    const int d0 = (int)cluster.block_rank();          // 0: even frequencies, 1: odd frequencies
    double2* s_even = d0 == 0 ? s_col : cluster.map_shared_rank(s_col, 0);
    double2* s_odd = d0 == 1 ? s_col : cluster.map_shared_rank(s_col, 1);
    const int tid = threadIdx.x;
    const int ncl = gridDim.x / 2;
    const double* fpos = tb.fpos + d0 * H;
    const double2* twpar = tb.twpar + d0 * H;
    const int npair = M / 2 + 1;                       // even / odd column pairs, as in k_theta_chain_syn
    for (int mp = blockIdx.x / 2; mp < npair; mp += ncl) {
        const int ma = 2 * mp, mb = 2 * mp + 1;
        const bool has_b = mb <= M;
        const double2* cola = ft + (int64_t)ma * N;
        const double2* colb = ft + (int64_t)(has_b ? mb : ma) * N;
        if (mp + ncl < npair) {
            const int64_t nxt = (int64_t)(ma + 2 * ncl + ((2 * (mp + ncl) + 1 <= M) ? d0 : 0)) * N;
            prefetch_l2(ft + nxt, N * (int)sizeof(double2), tid, T);
        }
        const double pa = pph[ma], pb = has_b ? pph[mb] : 0.0;
        // a3: this CTA's half of the radix-2 stage, fused with the load of the pair
        for (int i = tid; i < H; i += T) {
            const double2 a0 = cola[i], a1 = cola[i + H], b0 = colb[i], b1 = colb[i + H];
            const double2 a = make_double2(fma(pb, b0.x, pa * a0.x), fma(pb, b0.y, pa * a0.y));
            const double2 b = make_double2(fma(pb, b1.x, pa * a1.x), fma(pb, b1.y, pa * a1.y));
            s_col[pad(i)] = d0 ? cmul(make_double2(a.x - b.x, a.y - b.y), tb.tw2[i]) : make_double2(a.x + b.x, a.y + b.y);
        }
        __syncthreads();
        HalfExec<N, -1> fwd{s_col, tb.stw, tid};
        forward_stages<H>(fwd);
        double2 c[E];
        last_stage_to_regs<H, RL, -1, E>(s_col, tid, T, c);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double f = fpos[e * T + tid];
            c[e] = make_double2(c[e].x * f, c[e].y * f);
        }
#pragma unroll 1
        for (int par = 0; par < 2; ++par) {
            if (par) {
#pragma unroll
                for (int e = 0; e < E; ++e) c[e] = cmul(c[e], twpar[e * T + tid]);
            }
            // (a thread overwrites exactly the positions it read in the last forward stage; for parity 1 the
            //  cluster.sync that ends parity 0 orders it after every read of this buffer)
            first_stage_from_regs<H, RL, +1, E>(s_col, tid, T, c);
            __syncthreads();
            HalfExec<N, +1> inv{s_col, tb.stw, tid};
            inverse_stages<H>(inv);
            cluster.sync();                            // both halves complete
            // last inverse stage across the pair, in place: u[i] goes to the even CTA's slot i, u[i + H] to the odd
            // CTA's slot i; this CTA does i in [d0 H/2, (d0+1) H/2), nobody else touches those slots
            for (int i = d0 * (H / 2) + tid; i < (d0 + 1) * (H / 2); i += T) {
                const double2 z0 = s_even[pad(i)], z1 = cmul(s_odd[pad(i)], cconj(tb.tw2[i]));
                s_even[pad(i)] = make_double2(z0.x + z1.x, z0.y + z1.y);
                s_odd[pad(i)] = make_double2(z0.x - z1.x, z0.y - z1.y);
            }
            cluster.sync();
            // separate the two columns by mirror parity: the mirror of row a' is u[N - a'] = odd slot H - a' on the
            // even fine rows, u[N - 1 - a'] = odd slot H - 1 - a' on the odd ones
            C* outa = h + ((int64_t)ma * 2 + par) * N;
            C* outb = h + ((int64_t)mb * 2 + par) * N;
            for (int ap = d0 * (H / 2) + tid; ap < (d0 + 1) * (H / 2); ap += T) {
                if (2 * ap + par >= nrow_half) break;
                const double2 u = s_even[pad(ap)];
                const double2 v = par ? s_odd[pad(H - 1 - ap)] : (ap == 0 ? u : s_odd[pad(H - ap)]);
                C va, vb;
                va.x = u.x + v.x;
                va.y = u.y + v.y;
                vb.x = u.x - v.x;
                vb.y = u.y - v.y;
                outa[ap] = va;
                if (has_b) outb[ap] = vb;
            }
            if (par == 0 && d0 == 0 && tid == 0 && 2 * H < nrow_half) {   // row a' = H = N/2 mirrors onto itself
                const double2 u = s_odd[pad(0)];
                C va, vb;
                va.x = 2.0 * u.x;
                va.y = 2.0 * u.y;
                vb.x = 0;
                vb.y = 0;
                outa[H] = va;
                if (has_b) outb[H] = vb;
            }
            cluster.sync();                            // the peer has read this CTA's half
        }
    }
}

template <int N, typename C>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(HalfCfg<N>::T, HalfCfg<N>::CTAS)
k_theta_chain2_adj(int L, int M, int nrow_half, const C* __restrict__ h, const double* __restrict__ pph,
                   const ChainTables tb, double2* __restrict__ ft) {
    using namespace fftsm;
    namespace cg = cooperative_groups;
    constexpr int H = HalfCfg<N>::H, T = HalfCfg<N>::T, E = HalfCfg<N>::E, RL = last_radix(H);
    extern __shared__ __align__(16) double2 s_col[];
    cg::cluster_group cluster = cg::this_cluster();
    const int d0 = (int)cluster.block_rank();
    const double2* s_even = d0 == 0 ? s_col : cluster.map_shared_rank(s_col, 0);
    const double2* s_odd = d0 == 1 ? s_col : cluster.map_shared_rank(s_col, 1);
    const int tid = threadIdx.x;
    const int ncl = gridDim.x / 2;
    const double* fpos = tb.fpos + d0 * H;
    const double2* twpar = tb.twpar + d0 * H;
    const int npair = M / 2 + 1;
    auto ld = [](const C* ptr, int idx) {
        const C v = ptr[idx];
        return make_double2((double)v.x, (double)v.y);
    };
    for (int mp = blockIdx.x / 2; mp < npair; mp += ncl) {
        const int ma = 2 * mp, mb = 2 * mp + 1;
        const bool has_b = mb <= M;
        const double sb = has_b ? 1.0 : 0.0;
        double2 acc[E];
#pragma unroll
        for (int e = 0; e < E; ++e) acc[e] = make_double2(0.0, 0.0);
#pragma unroll 1
        for (int par = 0; par < 2; ++par) {
            const C* ina = h + ((int64_t)ma * 2 + par) * N;
            const C* inb = h + ((int64_t)(has_b ? mb : ma) * 2 + par) * N;
            if (par) __syncthreads();                  // the last forward stage of parity 0 has read s_col
            // transpose of the separation (see k_theta_chain_adj), this CTA's half of the radix-2 stage fused in
            for (int i = tid; i < H; i += T) {
                double2 a, b;
                if (par == 0) {
                    const double2 xa = ld(ina, i), xb = ld(inb, i);
                    const double2 ya = ld(ina, H - i), yb = ld(inb, H - i);
                    a = i == 0 ? make_double2(2.0 * xa.x, 2.0 * xa.y) : make_double2(fma(sb, xb.x, xa.x), fma(sb, xb.y, xa.y));
                    b = i == 0 ? make_double2(2.0 * ya.x, 2.0 * ya.y) : make_double2(fma(-sb, yb.x, ya.x), fma(-sb, yb.y, ya.y));
                } else {
                    const double2 xa = ld(ina, i), xb = ld(inb, i);
                    const double2 ya = ld(ina, H - 1 - i), yb = ld(inb, H - 1 - i);
                    a = make_double2(fma(sb, xb.x, xa.x), fma(sb, xb.y, xa.y));
                    b = make_double2(fma(-sb, yb.x, ya.x), fma(-sb, yb.y, ya.y));
                }
                s_col[pad(i)] = d0 ? cmul(make_double2(a.x - b.x, a.y - b.y), tb.tw2[i]) : make_double2(a.x + b.x, a.y + b.y);
            }
            __syncthreads();
            HalfExec<N, -1> fwd{s_col, tb.stw, tid};
            forward_stages<H>(fwd);
            double2 v[E];
            last_stage_to_regs<H, RL, -1, E>(s_col, tid, T, v);
#pragma unroll
            for (int e = 0; e < E; ++e) {
                if (par) v[e] = cmul(v[e], cconj(twpar[e * T + tid]));
                acc[e].x += v[e].x;
                acc[e].y += v[e].y;
            }
        }
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const double f = fpos[e * T + tid];
            acc[e] = make_double2(acc[e].x * f, acc[e].y * f);
        }
        first_stage_from_regs<H, RL, +1, E>(s_col, tid, T, acc);
        __syncthreads();
        HalfExec<N, +1> inv{s_col, tb.stw, tid};
        inverse_stages<H>(inv);
        cluster.sync();
        const double pa = pph[ma], pb = has_b ? pph[mb] : 0.0;
        double2* outa = ft + (int64_t)ma * N;
        double2* outb = ft + (int64_t)mb * N;
        for (int i = d0 * (H / 2) + tid; i < (d0 + 1) * (H / 2); i += T) {
            const double2 z0 = s_even[pad(i)], z1 = cmul(s_odd[pad(i)], cconj(tb.tw2[i]));
            const double2 x0 = make_double2(z0.x + z1.x, z0.y + z1.y), x1 = make_double2(z0.x - z1.x, z0.y - z1.y);
            outa[i] = make_double2(pa * x0.x, pa * x0.y);
            outa[i + H] = make_double2(pa * x1.x, pa * x1.y);
            if (has_b) {
                outb[i] = make_double2(pb * x0.x, pb * x0.y);
                outb[i + H] = make_double2(pb * x1.x, pb * x1.y);
            }
        }
        cluster.sync();
    }
}

// ---------------------------------------------------------------------------------------------
// Fused phi transform (a5 phi / a9 phi) for n_phi/2 = N a power of two <= 8192: ONE kernel per direction does what
// k_h_to_z + cuFFT (and cuFFT + k_z_to_h) do in two passes over the 1 GB grid.  A CTA takes a grid row: it gathers the
// row's half spectrum X[m] = H[m][parity][a'] (m <= mmax), forms the length-N complex sequence of the half-length
// real-FFT trick (see k_h_to_z) directly at the digit-reversed positions the inverse chain of fft_smem.cuh expects,
// transforms in shared memory and stores the real row with coalesced 16-byte stores; the adjoint loads the row,
// transforms forward, and scatters the post-processed Y[m] back to H.  The gathers / scatters are 16-byte accesses
// at a stride of one H column; rows of one parity are taken in order by neighbouring CTAs, so the other half of each
// 32-byte sector is served from / merged in L2.
// ---------------------------------------------------------------------------------------------
struct PhiTables {
    const double2* tw2;     // exp(-2 pi i i/N), i < N/2
    const double2* stw;     // per-stage twiddles of length N (fftsm::stage_table_offset)
    const double2* twz;     // W^m = exp(2 pi i m / n_phi), m <= mmax
};

// grid row index of the i-th row a CTA loop visits: all even rows a = 2a' in order, then all odd ones
__device__ __forceinline__ int phi_row_of(int i, int nrow_half) {
    const int n_even = (nrow_half + 1) / 2;
    return i < n_even ? 2 * i : 2 * (i - n_even) + 1;
}

template <int N, typename C>
__global__ void __launch_bounds__(ChainCfg<N>::T)
k_phi_syn(int M, int nh, int nrow_half, const C* __restrict__ h, const PhiTables tb, C* __restrict__ grid) {
    using namespace fftsm;
    constexpr int T = ChainCfg<N>::T, RL = last_radix(N / 2);
    extern __shared__ __align__(16) double2 s_col[];
    const int tid = threadIdx.x;
    for (int it = blockIdx.x; it < nrow_half; it += gridDim.x) {
        const int a = phi_row_of(it, nrow_half), par = a & 1, ap = a >> 1;
        __syncthreads();   // the previous row's stores have read s_col
        for (int k = M + 1 + tid; k <= N - M - 1; k += T) s_col[pad(pos_of_freq<N>(k))] = make_double2(0.0, 0.0);
        for (int m = tid; m <= M; m += T) {
            const C xc = h[((int64_t)m * 2 + par) * nh + ap];
            const double xr = (double)xc.x, xi = (double)xc.y;
            if (m == 0) {          // X[0] is real for a real row; its imaginary part is ignored
                s_col[pad(pos_of_freq<N>(0))] = make_double2(xr, xr);
            } else {
                const double2 w = tb.twz[m];
                s_col[pad(pos_of_freq<N>(m))] = make_double2(xr * (1.0 - w.y) - xi * w.x, xr * w.x + xi * (1.0 - w.y));
                s_col[pad(pos_of_freq<N>(N - m))] = make_double2(xr * (1.0 + w.y) + xi * w.x, xr * w.x - xi * (1.0 + w.y));
            }
        }
        if (it + (int)gridDim.x < nrow_half) {               // next row's half spectrum -> L2 while this one is transformed
            const int a2 = phi_row_of(it + (int)gridDim.x, nrow_half);
            for (int m = tid; m <= M; m += T)
                asm volatile("prefetch.global.L2 [%0];" ::"l"(h + ((int64_t)m * 2 + (a2 & 1)) * nh + (a2 >> 1)));
        }
        __syncthreads();
        stage_dit<N, RL, RL, +1>(s_col, tid, T, tb.stw);     // first inverse stage: stride 1, no twiddles
        __syncthreads();
        DevExec<N, +1> inv{s_col, tb.stw, tid};
        inverse_stages<N / 2>(inv);
        C* row = grid + (int64_t)a * N;                      // the real row viewed as N pairs (x[2j], x[2j+1])
        for (int i = tid; i < N / 2; i += T) {
            const double2 z0 = s_col[pad(i)], z1 = cmul(s_col[pad(i + N / 2)], cconj(tb.tw2[i]));
            C o0, o1;
            o0.x = z0.x + z1.x;
            o0.y = z0.y + z1.y;
            o1.x = z0.x - z1.x;
            o1.y = z0.y - z1.y;
            row[i] = o0;
            row[i + N / 2] = o1;
        }
    }
}

template <int N, typename C>
__global__ void __launch_bounds__(ChainCfg<N>::T)
k_phi_adj(int M, int nh, int nrow_half, const C* __restrict__ grid, const PhiTables tb, C* __restrict__ h) {
    using namespace fftsm;
    constexpr int T = ChainCfg<N>::T, RL = last_radix(N / 2);
    extern __shared__ __align__(16) double2 s_col[];
    const int tid = threadIdx.x;
    for (int it = blockIdx.x; it < nrow_half; it += gridDim.x) {
        const int a = phi_row_of(it, nrow_half), par = a & 1, ap = a >> 1;
        const C* row = grid + (int64_t)a * N;
        __syncthreads();
        for (int i = tid; i < N / 2; i += T) {               // radix-2 stage of the forward transform, fused with the load
            const C ac = row[i], bc = row[i + N / 2];
            const double2 x0 = make_double2((double)ac.x, (double)ac.y), x1 = make_double2((double)bc.x, (double)bc.y);
            s_col[pad(i)] = make_double2(x0.x + x1.x, x0.y + x1.y);
            s_col[pad(i + N / 2)] = cmul(make_double2(x0.x - x1.x, x0.y - x1.y), tb.tw2[i]);
        }
        if (it + (int)gridDim.x < nrow_half)                 // next row -> L2 while this one is transformed
            prefetch_l2(grid + (int64_t)phi_row_of(it + (int)gridDim.x, nrow_half) * N, N * (int)sizeof(C), tid, T);
        __syncthreads();
        DevExec<N, -1> fwd{s_col, tb.stw, tid};
        forward_stages<N / 2>(fwd);
        stage_dif<N, RL, RL, -1>(s_col, tid, T, tb.stw);     // last forward stage, in place
        __syncthreads();
        for (int m = tid; m <= M; m += T) {                  // post-processing of the real FFT (see k_z_to_h)
            const double2 A = s_col[pad(pos_of_freq<N>(m))], Bq = s_col[pad(pos_of_freq<N>(m == 0 ? 0 : N - m))];
            const double2 w = tb.twz[m];
            const double bx = Bq.x, by = -Bq.y;              // B = conj Zf[N - m]
            const double dx = A.x - bx, dy = A.y - by;
            C out;
            out.x = 0.5 * ((A.x + bx) + (w.x * dy - w.y * dx));
            out.y = 0.5 * ((A.y + by) - (w.x * dx + w.y * dy));
            h[((int64_t)m * 2 + par) * nh + ap] = out;
        }
    }
}

// The same two kernels at N = 8192 on the register-tiled transform of fft_reg.cuh.  The radix-2 split of the length-N
// transform gives two INDEPENDENT 4096-point transforms (even / odd outputs of the inverse, even / odd frequencies of
// the forward one; Zf[m] and its partner Zf[N - m] of the real-FFT post-processing have the same parity), so a work
// item is (grid row, half): one CTA of 256 threads, 16 points per thread in registers, two exchanges through 70 KB of
// shared memory.  Two such CTAs fit an SM (registers), so the loads / stores of one overlap the transform of the
// other, which the one-CTA-per-SM kernels above cannot do.
template <typename C>
__global__ void __launch_bounds__(256, 2)
k_phi_syn_r(int M, int nh, int nrow_half, const C* __restrict__ h, const PhiTables tb, C* __restrict__ grid) {
    using namespace fftsm;
    constexpr int N = 8192, H = N / 2;
    extern __shared__ __align__(16) double2 s_half[];
    const int th = threadIdx.x;
    const double2* tw4096 = tb.stw + stage_table_offset(N, 4096);
    const double2* tw256 = tb.stw + stage_table_offset(N, 256);
    for (int item = blockIdx.x; item < 2 * nrow_half; item += gridDim.x) {
        const int hf = item & 1, a = phi_row_of(item >> 1, nrow_half), par = a & 1, ap = a >> 1;
        const C* hrow = h + (int64_t)par * nh + ap;          // X[m] = hrow[m * 2 nh]
        double2 x[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            // Z[q] and Z[q + N/2] of the half-length real-FFT sequence (see k_h_to_z), q = th + 256 j
            const int q = th + 256 * j, mq = H - q;
            double2 zlo = make_double2(0.0, 0.0), zhi = make_double2(0.0, 0.0);
            if (q <= M) {
                const C xc = hrow[(int64_t)q * 2 * nh];
                const double xr = (double)xc.x, xi = (double)xc.y;
                if (q == 0) {
                    zlo = make_double2(xr, xr);              // X[0] is real for a real row
                } else {
                    const double2 w = tb.twz[q];
                    zlo = make_double2(xr * (1.0 - w.y) - xi * w.x, xr * w.x + xi * (1.0 - w.y));
                }
            }
            if (q > 0 && mq <= M) {                          // Z[N - m], m = N/2 - q
                const C xc = hrow[(int64_t)mq * 2 * nh];
                const double xr = (double)xc.x, xi = (double)xc.y;
                const double2 w = tb.twz[mq];
                zhi = make_double2(xr * (1.0 + w.y) + xi * w.x, xr * w.x - xi * (1.0 + w.y));
            }
            // radix-2 split of the inverse transform: even outputs from Z[q] + Z[q + N/2], odd ones from the twiddled difference
            x[j] = hf ? cmul(make_double2(zlo.x - zhi.x, zlo.y - zhi.y), cconj(tb.tw2[q]))
                      : make_double2(zlo.x + zhi.x, zlo.y + zhi.y);
        }
        __syncthreads();                                     // the previous item's last exchange has been read
        fftreg::fft4096<+1>(x, s_half, th, tw4096, tw256);
        C* row = grid + (int64_t)a * N;                      // the real row viewed as N pairs (x[2j], x[2j+1])
#pragma unroll
        for (int c = 0; c < 16; ++c) {
            const double2 v = x[bitrev(c, 16)];
            C o;
            o.x = v.x;
            o.y = v.y;
            row[2 * (th + 256 * c) + hf] = o;
        }
    }
}

template <typename C>
__global__ void __launch_bounds__(256, 2)
k_phi_adj_r(int M, int nh, int nrow_half, const C* __restrict__ grid, const PhiTables tb, C* __restrict__ h) {
    using namespace fftsm;
    constexpr int N = 8192, H = N / 2;
    extern __shared__ __align__(16) double2 s_half[];
    const int th = threadIdx.x;
    const double2* tw4096 = tb.stw + stage_table_offset(N, 4096);
    const double2* tw256 = tb.stw + stage_table_offset(N, 256);
    for (int item = blockIdx.x; item < 2 * nrow_half; item += gridDim.x) {
        const int hf = item & 1, a = phi_row_of(item >> 1, nrow_half), par = a & 1, ap = a >> 1;
        const C* row = grid + (int64_t)a * N;
        double2 x[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) {                       // radix-2 split of the forward transform, fused with the load
            const int i = th + 256 * j;
            const C ac = row[i], bc = row[i + H];
            const double2 x0 = make_double2((double)ac.x, (double)ac.y), x1 = make_double2((double)bc.x, (double)bc.y);
            x[j] = hf ? cmul(make_double2(x0.x - x1.x, x0.y - x1.y), tb.tw2[i]) : make_double2(x0.x + x1.x, x0.y + x1.y);
        }
        __syncthreads();                                     // the previous item's post-processing has read s_half
        fftreg::fft4096<-1>(x, s_half, th, tw4096, tw256);
        __syncthreads();                                     // every thread is past its last read of the exchange buffer
#pragma unroll
        for (int c = 0; c < 16; ++c) s_half[pad(th + 256 * c)] = x[bitrev(c, 16)];   // Zf[2 q + hf] at q
        __syncthreads();
        // post-processing of the real FFT (see k_z_to_h) for the m of this half's parity: m = 2 q + hf, and its partner
        // N - m = 2 (N/2 - q - hf) + hf lives in the same half
#pragma unroll 4
        for (int j = 0; j < 16; ++j) {
            const int q = th + 256 * j, m = 2 * q + hf;
            if (m > M) break;
            const int qp = (m == 0) ? 0 : H - q - hf;
            const double2 A = s_half[pad(q)], Bq = s_half[pad(qp)];
            const double2 w = tb.twz[m];
            const double bx = Bq.x, by = -Bq.y;              // B = conj Zf[N - m]
            const double dx = A.x - bx, dy = A.y - by;
            C out;
            out.x = 0.5 * ((A.x + bx) + (w.x * dy - w.y * dx));
            out.y = 0.5 * ((A.y + by) - (w.x * dx + w.y * dy));
            h[((int64_t)m * 2 + par) * nh + ap] = out;
        }
    }
}

template <typename C>
int launch_phi_r(bool* attr_set, bool adjoint, int M, int nh, int nrow_half, int n_sm, const PhiTables& tb, C* h, C* grid,
                 cudaStream_t s) {
    constexpr int SMEM = fftreg::HSMEM * (int)sizeof(double2);
    if (!attr_set[adjoint]) {
        if (adjoint) NUSHT_CUDA_TRY(cudaFuncSetAttribute(k_phi_adj_r<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM));
        else NUSHT_CUDA_TRY(cudaFuncSetAttribute(k_phi_syn_r<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM));
        attr_set[adjoint] = true;
    }
    const int blocks = std::min(2 * nrow_half, 2 * n_sm);
    if (adjoint) k_phi_adj_r<C><<<blocks, 256, SMEM, s>>>(M, nh, nrow_half, grid, tb, h);
    else k_phi_syn_r<C><<<blocks, 256, SMEM, s>>>(M, nh, nrow_half, h, tb, grid);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}

template <int N, typename C>
int launch_phi(bool* attr_set, bool adjoint, int M, int nh, int nrow_half, int n_sm, const PhiTables& tb, C* h, C* grid,
               cudaStream_t s) {
    if (!attr_set[adjoint]) {
        if (adjoint)
            NUSHT_CUDA_TRY(cudaFuncSetAttribute(k_phi_adj<N, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ChainCfg<N>::SMEM));
        else
            NUSHT_CUDA_TRY(cudaFuncSetAttribute(k_phi_syn<N, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ChainCfg<N>::SMEM));
        attr_set[adjoint] = true;
    }
    const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(8, (size_t)(200 * 1024) / (ChainCfg<N>::SMEM + 1024)));
    const int blocks = std::min(nrow_half, n_sm * per_sm);
    if (adjoint) k_phi_adj<N, C><<<blocks, ChainCfg<N>::T, ChainCfg<N>::SMEM, s>>>(M, nh, nrow_half, grid, tb, h);
    else k_phi_syn<N, C><<<blocks, ChainCfg<N>::T, ChainCfg<N>::SMEM, s>>>(M, nh, nrow_half, h, tb, grid);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}

template <typename C>
int dispatch_phi(nusht_plan_s* p, bool adjoint, cudaStream_t s) {
    const int n = p->ng.nph / 2;
    PhiTables tb;
    tb.tw2 = p->d_phitab;
    tb.stw = p->d_phitab + n / 2;
    tb.twz = p->d_twz;
    if (n == 8192 && !getenv("NUSHT_PHI_SMEM"))       // register-tiled transform (NUSHT_PHI_SMEM keeps the stage-by-stage one: tests)
        return launch_phi_r<C>(p->phi_attr_set, adjoint, p->mmax, p->ng.nth / 2, p->ng.nrow_half, p->n_sm, tb, (C*)p->d_h,
                               (C*)p->d_grid, s);
    switch (n) {
#define NUSHT_PHI(NN) \
    case NN:          \
        return launch_phi<NN, C>(p->phi_attr_set, adjoint, p->mmax, p->ng.nth / 2, p->ng.nrow_half, p->n_sm, tb, (C*)p->d_h, (C*)p->d_grid, s);
        NUSHT_PHI(128) NUSHT_PHI(256) NUSHT_PHI(512) NUSHT_PHI(1024) NUSHT_PHI(2048) NUSHT_PHI(4096) NUSHT_PHI(8192)
#undef NUSHT_PHI
    }
    return NUSHT_ERR_UNSUPPORTED;
}

// position -> frequency of the forward chain for a run-time N (host; mirrors fftsm::freq_of_pos)
static int chain_freq_of_pos(int n, int p) {
    int q = p / (n / 2), mul = 2, ns = n / 2;
    p %= n / 2;
    while (ns >= 16) {
        q += mul * (p / (ns / 16));
        p %= ns / 16;
        mul *= 16;
        ns /= 16;
    }
    return q + mul * p;
}

template <int N, typename C>
int launch_chain(bool* attr_set, bool adjoint, int L, int M, int nrow_half, int n_sm, double2* ft, const double* pph,
                 const ChainTables& tb, C* h, cudaStream_t s) {
    // the attribute is per device: the flag lives in the plan (one device), not in the process
    if (!attr_set[adjoint]) {
        if (adjoint)
            NUSHT_CUDA_TRY(cudaFuncSetAttribute(k_theta_chain_adj<N, C>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                (int)ChainCfg<N>::SMEM));
        else
            NUSHT_CUDA_TRY(cudaFuncSetAttribute(k_theta_chain_syn<N, C>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                (int)ChainCfg<N>::SMEM));
        attr_set[adjoint] = true;
    }
    // persistent: as many CTAs as fit at once (shared memory bound), columns dealt round robin
    const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(8, (size_t)(200 * 1024) / (ChainCfg<N>::SMEM + 1024)));
    const int grid = std::min(M / 2 + 1, n_sm * per_sm);   // one CTA iteration per column pair
    if (adjoint)
        k_theta_chain_adj<N, C><<<grid, ChainCfg<N>::T, ChainCfg<N>::SMEM, s>>>(L, M, nrow_half, h, pph, tb, ft);
    else
        k_theta_chain_syn<N, C><<<grid, ChainCfg<N>::T, ChainCfg<N>::SMEM, s>>>(L, M, nrow_half, ft, pph, tb, h);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}

template <int N, typename C>
int launch_chain2(bool* attr_set, bool adjoint, int L, int M, int nrow_half, int n_sm, double2* ft, const double* pph,
                  const ChainTables& tb, C* h, cudaStream_t s) {
    if (!attr_set[adjoint]) {
        if (adjoint)
            NUSHT_CUDA_TRY(cudaFuncSetAttribute(k_theta_chain2_adj<N, C>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                (int)HalfCfg<N>::SMEM));
        else
            NUSHT_CUDA_TRY(cudaFuncSetAttribute(k_theta_chain2_syn<N, C>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                (int)HalfCfg<N>::SMEM));
        attr_set[adjoint] = true;
    }
    // persistent pairs: as many CTAs as fit at once (shared memory, 128 registers per thread), columns round robin
    const size_t by_smem = (size_t)(200 * 1024) / (HalfCfg<N>::SMEM + 1024);
    const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(HalfCfg<N>::CTAS, by_smem));
    const int grid = 2 * std::max(1, std::min(M / 2 + 1, n_sm * per_sm / 2));   // one cluster iteration per column pair
    if (adjoint)
        k_theta_chain2_adj<N, C><<<grid, HalfCfg<N>::T, HalfCfg<N>::SMEM, s>>>(L, M, nrow_half, h, pph, tb, ft);
    else
        k_theta_chain2_syn<N, C><<<grid, HalfCfg<N>::T, HalfCfg<N>::SMEM, s>>>(L, M, nrow_half, ft, pph, tb, h);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}

template <typename C>
int dispatch_chain(nusht_plan_s* p, bool adjoint, C* h, cudaStream_t s) {
    const int n = p->lg.nth2;
    ChainTables tb;
    tb.tw2 = p->d_tw2n;
    tb.stw = p->d_tw2n + n / 2;
    tb.twpar = p->d_tw2n + n / 2 + fftsm::stage_table_len(n);
    tb.fpos = reinterpret_cast<const double*>(tb.twpar + n);
    if (p->theta_chain == 2) {
        switch (n) {
#define NUSHT_CHAIN2(NN) \
    case NN:             \
        return launch_chain2<NN, C>(p->chain_attr_set, adjoint, p->lmax, p->mmax, p->ng.nrow_half, p->n_sm, p->d_ft, p->d_pph, tb, h, s);
            NUSHT_CHAIN2(2048) NUSHT_CHAIN2(4096) NUSHT_CHAIN2(8192) NUSHT_CHAIN2(16384)
#undef NUSHT_CHAIN2
        }
        return NUSHT_ERR_UNSUPPORTED;
    }
    switch (n) {
#define NUSHT_CHAIN(NN) \
    case NN:            \
        return launch_chain<NN, C>(p->chain_attr_set, adjoint, p->lmax, p->mmax, p->ng.nrow_half, p->n_sm, p->d_ft, p->d_pph, tb, h, s);
        NUSHT_CHAIN(128) NUSHT_CHAIN(256) NUSHT_CHAIN(512) NUSHT_CHAIN(1024) NUSHT_CHAIN(2048) NUSHT_CHAIN(4096)
        NUSHT_CHAIN(8192)
#undef NUSHT_CHAIN
    }
    return NUSHT_ERR_UNSUPPORTED;
}

}  // namespace

template <typename T>
static int f_alloc(T** ptr, size_t bytes, nusht_plan_s* p) {
    if (bytes == 0) bytes = 16;
    NUSHT_CUDA_TRY(cudaMalloc((void**)ptr, bytes));
    p->workspace_bytes += (int64_t)bytes;
    return NUSHT_OK;
}

int fourier_build(nusht_plan_s* p) {
    const int L = p->lmax, M = p->mmax;
    const NufftGeom& g = p->ng;
    const int nth2 = p->lg.nth2;
    const bool f64 = p->dtype == NUSHT_F64;
    const size_t csz = f64 ? 16 : 8, rsz = f64 ? 8 : 4;

    // deconvolution tables (host, extended precision inside nufft_kernel_ft); 1/Ntheta folded into p_theta
    std::vector<double> pth(2 * L + 1), pph(M + 1);
    nufft_kernel_ft(p, 0.0, g.nth);     // (builds its quadrature nodes once, before the threads start)
    nusht_parallel_for(L + 1, [&](int lo, int hi) {
        for (int k = lo; k < hi; ++k) {
            const double v = 1.0 / (nufft_kernel_ft(p, (double)k, g.nth) * (double)nth2);
            pth[L + k] = v;
            pth[L - k] = v;
        }
    });
    nusht_parallel_for(M + 1, [&](int lo, int hi) {
        for (int m = lo; m < hi; ++m) pph[m] = 1.0 / nufft_kernel_ft(p, (double)m, g.nph);
    });
    NUSHT_TRY(f_alloc(&p->d_pth, sizeof(double) * (2 * L + 1), p));
    NUSHT_TRY(f_alloc(&p->d_pph, sizeof(double) * (M + 1), p));
    NUSHT_CUDA_TRY(cudaMemcpy(p->d_pth, pth.data(), sizeof(double) * (2 * L + 1), cudaMemcpyHostToDevice));
    NUSHT_CUDA_TRY(cudaMemcpy(p->d_pph, pph.data(), sizeof(double) * (M + 1), cudaMemcpyHostToDevice));

    const size_t hbytes = (size_t)(M + 1) * (size_t)g.nth * csz;
    const size_t gbytes = (size_t)g.nrow_half * (size_t)g.nph * rsz;
    if (p->fourier_general) {
        // sigma != 2 exists to save memory: H[m][a] and the fine grid are never live together (synthesis: H -> Z, then
        // Z -> grid; adjoint: grid -> Z, then Z -> H), so they share one allocation
        NUSHT_TRY(f_alloc(&p->d_h, std::max(hbytes, gbytes), p));
        p->d_grid = p->d_h;
        NUSHT_CUDA_TRY(cudaMemset(p->d_h, 0, std::max(hbytes, gbytes)));
    } else {
        NUSHT_TRY(f_alloc(&p->d_h, hbytes, p));
        NUSHT_TRY(f_alloc(&p->d_grid, gbytes, p));
        NUSHT_CUDA_TRY(cudaMemset(p->d_h, 0, hbytes));
        NUSHT_CUDA_TRY(cudaMemset(p->d_grid, 0, gbytes));
    }

    if (p->fourier_general) {
        // sigma != 2: plain cuFFT chain (see k_deconv_pad_gen)
        p->theta_chain = 0;
        p->theta_fused = false;
        const size_t zbytes = (size_t)g.nrow_half * (size_t)(g.nph / 2 + 1) * csz;
        NUSHT_TRY(f_alloc(&p->d_z, zbytes, p));
        // the four plans run one after the other on the transform's stream: ONE work area, sized for the largest
        // (this variant exists to save memory; non-power-of-two lengths need a work area of the size of their data)
        size_t ws = 0, wmax = 0;
        int n1[1] = {nth2}, n2[1] = {g.nth}, n3[1] = {g.nph};
        cufftHandle* hs[4] = {&p->fft_theta_coarse, &p->fft_theta_fine, &p->fft_phi, &p->fft_phi_r2c};
        for (int i = 0; i < 4; ++i) {
            NUSHT_CUFFT_TRY(cufftCreate(hs[i]));
            NUSHT_CUFFT_TRY(cufftSetAutoAllocation(*hs[i], 0));
        }
        NUSHT_CUFFT_TRY(cufftMakePlanMany(p->fft_theta_coarse, 1, n1, nullptr, 1, nth2, nullptr, 1, nth2, CUFFT_Z2Z, M + 1, &ws));
        wmax = std::max(wmax, ws);
        NUSHT_CUFFT_TRY(cufftMakePlanMany(p->fft_theta_fine, 1, n2, nullptr, 1, g.nth, nullptr, 1, g.nth,
                                          f64 ? CUFFT_Z2Z : CUFFT_C2C, M + 1, &ws));
        wmax = std::max(wmax, ws);
        NUSHT_CUFFT_TRY(cufftMakePlanMany(p->fft_phi, 1, n3, nullptr, 1, 0, nullptr, 1, 0, f64 ? CUFFT_Z2D : CUFFT_C2R,
                                          g.nrow_half, &ws));
        wmax = std::max(wmax, ws);
        NUSHT_CUFFT_TRY(cufftMakePlanMany(p->fft_phi_r2c, 1, n3, nullptr, 1, 0, nullptr, 1, 0, f64 ? CUFFT_D2Z : CUFFT_R2C,
                                          g.nrow_half, &ws));
        wmax = std::max(wmax, ws);
        NUSHT_TRY(f_alloc(&p->d_fftwork, wmax, p));
        for (int i = 0; i < 4; ++i) NUSHT_CUFFT_TRY(cufftSetWorkArea(*hs[i], p->d_fftwork));
        p->have_fft = true;
        return NUSHT_OK;
    }

    // fused theta chains: coarse length == half fine length, a power of two.  theta_chain = 1: one CTA per
    // column (128 <= N <= 8192, the default there: 0.73 / 0.84 ms against 0.76 / 0.87 ms at N = 8192);
    // 2: a cluster pair per column (2048 <= N <= 16384; the default at 16384, where one SM cannot hold a column)
    {
        const bool pow2 = (g.nth / 2 == nth2) && (nth2 & (nth2 - 1)) == 0;
        p->theta_chain = 0;
        if (pow2 && nth2 >= 128 && nth2 <= 8192) p->theta_chain = 1;
        else if (pow2 && nth2 == 16384) p->theta_chain = 2;
        // NUSHT_THETA_CHAIN = cufft | single | cluster overrides the choice where the variant exists (tests
        // compare the three)
        const char* ev = getenv("NUSHT_THETA_CHAIN");
        if (ev && strcmp(ev, "cufft") == 0) p->theta_chain = 0;
        if (ev && strcmp(ev, "single") == 0 && pow2 && nth2 >= 128 && nth2 <= 8192) p->theta_chain = 1;
        if (ev && strcmp(ev, "cluster") == 0 && pow2 && nth2 >= 2048 && nth2 <= 16384) p->theta_chain = 2;
        p->theta_fused = p->theta_chain != 0;
    }
    if (p->theta_fused) {
        // one buffer: tw2 [N/2] | stage tables | twpar [N] | fpos [N doubles]
        const int n = nth2, nst = fftsm::stage_table_len(n);
        std::vector<double2> tb((size_t)n / 2 + nst + n + (n + 1) / 2);
        const long double PI_L = 3.14159265358979323846264338327950288L;
        auto unit = [&](long double turns) {   // exp(2 pi i turns)
            return make_double2((double)cosl(2.0L * PI_L * turns), (double)sinl(2.0L * PI_L * turns));
        };
        for (int i = 0; i < n / 2; ++i) tb[i] = unit(-(long double)i / (long double)n);
        {
            size_t o = (size_t)n / 2;
            for (int ns = n / 2; ns >= 32; ns /= 16)
                for (int i = 0; i < ns / 16; ++i) tb[o++] = unit(-(long double)i / (long double)ns);
        }
        double2* twpar = tb.data() + n / 2 + nst;
        double* fpos = reinterpret_cast<double*>(twpar + n);
        // entry e of thread t <-> position RL (t + T (e / RL)) + e % RL, stored at [e][t] (coalesced)
        // (cluster pair: the same per half d0, stored at [d0][e][t])
        const int nhalf = p->theta_chain == 2 ? 2 : 1, len = n / nhalf;
        const int T = p->theta_chain == 2 ? half_threads(len) : chain_threads(n), E = len / T;
        const int RL = fftsm::last_radix(n / 2);
        for (int d0 = 0; d0 < nhalf; ++d0)
            for (int e = 0; e < E; ++e)
                for (int t = 0; t < T; ++t) {
                    const int pos = d0 * len + RL * (t + T * (e / RL)) + e % RL;
                    const int f = chain_freq_of_pos(n, pos), k = f < n / 2 ? f : f - n;
                    const size_t at = (size_t)d0 * len + (size_t)e * T + t;
                    twpar[at] = unit((long double)k / (long double)(2 * n));
                    // (column pairs: the 1/2 of their separation is folded in here)
                    fpos[at] = (k >= -L && k <= L) ? 0.5 * pth[k + L] : 0.0;
                }
        NUSHT_TRY(f_alloc(&p->d_tw2n, sizeof(double2) * tb.size(), p));
        NUSHT_CUDA_TRY(cudaMemcpy(p->d_tw2n, tb.data(), sizeof(double2) * tb.size(), cudaMemcpyHostToDevice));
        int dev = 0;
        NUSHT_CUDA_TRY(cudaGetDevice(&dev));
        NUSHT_CUDA_TRY(cudaDeviceGetAttribute(&p->n_sm, cudaDevAttrMultiProcessorCount, dev));
    }

    // fused phi transform: n_phi / 2 a power of two in [128, 8192] next to a fused theta chain (NUSHT_PHI=cufft
    // keeps the cuFFT path for the tests, which compare the two)
    {
        const int nz = g.nph / 2;
        // Measured at config 3 (n_phi / 2 = 8192): adjoint 0.86 ms fused against 0.92 ms (cuFFT 0.59 + k_z_to_h 0.32);
        // synthesis 0.94-0.97 ms fused against 0.88 ms (k_h_to_z 0.27 + cuFFT 0.61): one CTA per SM cannot overlap its
        // phases and the radix-16 stages through shared memory cost about 12 us per 8192-point row, as much as cuFFT's
        // register-tiled transform plus the extra pass.  Default: fused in the adjoint only; NUSHT_PHI = fused | cufft
        // forces both directions (tests compare them).
        const char* ev = getenv("NUSHT_PHI");
        // (FP32 plans keep cuFFT unless forced: its binary32 transform takes 0.37 ms where the fused kernel, which
        //  computes in binary64 whatever the storage type, takes 0.83 ms)
        const bool forced = ev && strcmp(ev, "fused") == 0;
        p->phi_fused = p->theta_fused && (nz & (nz - 1)) == 0 && nz >= 128 && nz <= 8192 && M < nz / 2 &&
                       !(ev && strcmp(ev, "cufft") == 0) && (f64 || forced);
        p->phi_fused_syn = p->phi_fused && forced;
        if (p->phi_fused) {
            const int nst = fftsm::stage_table_len(nz);
            std::vector<double2> tb((size_t)nz / 2 + nst);
            const long double PI_L = 3.14159265358979323846264338327950288L;
            auto unit = [&](long double turns) {
                return make_double2((double)cosl(2.0L * PI_L * turns), (double)sinl(2.0L * PI_L * turns));
            };
            for (int i = 0; i < nz / 2; ++i) tb[i] = unit(-(long double)i / (long double)nz);
            size_t o = (size_t)nz / 2;
            for (int ns = nz / 2; ns >= 32; ns /= 16)
                for (int i = 0; i < ns / 16; ++i) tb[o++] = unit(-(long double)i / (long double)ns);
            NUSHT_TRY(f_alloc(&p->d_phitab, sizeof(double2) * tb.size(), p));
            NUSHT_CUDA_TRY(cudaMemcpy(p->d_phitab, tb.data(), sizeof(double2) * tb.size(), cudaMemcpyHostToDevice));
        }
    }

    // cuFFT plans
    size_t ws = 0, wtot = 0;
    if (!p->theta_fused) {
        int n[1] = {nth2};
        NUSHT_CUFFT_TRY(cufftCreate(&p->fft_theta_coarse));
        NUSHT_CUFFT_TRY(cufftMakePlanMany(p->fft_theta_coarse, 1, n, nullptr, 1, nth2, nullptr, 1, nth2, CUFFT_Z2Z,
                                          M + 1, &ws));
        wtot += ws;
    }
    if (!p->theta_fused) {
        int n[1] = {g.nth / 2};   // two half-length transforms per m (see k_deconv_pad)
        NUSHT_CUFFT_TRY(cufftCreate(&p->fft_theta_fine));
        NUSHT_CUFFT_TRY(cufftMakePlanMany(p->fft_theta_fine, 1, n, nullptr, 1, g.nth / 2, nullptr, 1, g.nth / 2,
                                          f64 ? CUFFT_Z2Z : CUFFT_C2C, 2 * (M + 1), &ws));
        wtot += ws;
    }
    {
        // phi pass: one complex transform of length n_phi/2 per grid row, in place (see k_h_to_z)
        int n[1] = {g.nph / 2};
        if (!p->phi_fused || !p->phi_fused_syn) {
            NUSHT_CUFFT_TRY(cufftCreate(&p->fft_phi));
            NUSHT_CUFFT_TRY(cufftMakePlanMany(p->fft_phi, 1, n, nullptr, 1, g.nph / 2, nullptr, 1, g.nph / 2,
                                              f64 ? CUFFT_Z2Z : CUFFT_C2C, g.nrow_half, &ws));
            wtot += ws;
        }
        std::vector<double2> tw(M + 1);
        const long double PI_L = 3.14159265358979323846264338327950288L;
        for (int m = 0; m <= M; ++m) {
            const long double ang = 2.0L * PI_L * (long double)m / (long double)g.nph;
            tw[m] = make_double2((double)cosl(ang), (double)sinl(ang));
        }
        NUSHT_TRY(f_alloc(&p->d_twz, sizeof(double2) * (M + 1), p));
        NUSHT_CUDA_TRY(cudaMemcpy(p->d_twz, tw.data(), sizeof(double2) * (M + 1), cudaMemcpyHostToDevice));
    }
    p->workspace_bytes += (int64_t)wtot;
    p->have_fft = true;
    return NUSHT_OK;
}

#define REC(i)                                                   \
    do {                                                         \
        if (ev) NUSHT_CUDA_TRY(cudaEventRecord(ev[(i)], s));     \
    } while (0)

// synthesis: d_ft (Ftilde) -> d_grid.  ev (optional) = events at the boundaries of stages 2..5:
// ev[0] before a3, ev[1] after a3, ev[2] after a4, ev[3] after a5-theta, ev[4] after a5-phi.
static int fourier_synthesis_general(nusht_plan_s* p, cudaStream_t s, cudaEvent_t* ev) {
    const int L = p->lmax, M = p->mmax;
    const NufftGeom& g = p->ng;
    const int nth2 = p->lg.nth2, nzc = g.nph / 2 + 1;
    const bool f64 = p->dtype == NUSHT_F64;
    REC(0);
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_theta_coarse, s));
    NUSHT_CUFFT_TRY(cufftExecZ2Z(p->fft_theta_coarse, (cufftDoubleComplex*)p->d_ft, (cufftDoubleComplex*)p->d_ft, CUFFT_FORWARD));
    REC(1);
    {
        dim3 grid((g.nth + 255) / 256, M + 1);
        if (f64) k_deconv_pad_gen<double><<<grid, 256, 0, s>>>(L, M, nth2, g.nth, p->d_ft, p->d_pth, p->d_pph, (double2*)p->d_h);
        else k_deconv_pad_gen<float><<<grid, 256, 0, s>>>(L, M, nth2, g.nth, p->d_ft, p->d_pth, p->d_pph, (float2*)p->d_h);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    REC(2);
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_theta_fine, s));
    if (f64) NUSHT_CUFFT_TRY(cufftExecZ2Z(p->fft_theta_fine, (cufftDoubleComplex*)p->d_h, (cufftDoubleComplex*)p->d_h, CUFFT_INVERSE));
    else NUSHT_CUFFT_TRY(cufftExecC2C(p->fft_theta_fine, (cufftComplex*)p->d_h, (cufftComplex*)p->d_h, CUFFT_INVERSE));
    REC(3);
    {
        dim3 grid((g.nrow_half + 31) / 32, (nzc + 31) / 32);
        if (f64) k_h_to_zc<double2><<<grid, 256, 0, s>>>(M, g.nth, g.nrow_half, nzc, (const double2*)p->d_h, (double2*)p->d_z);
        else k_h_to_zc<float2><<<grid, 256, 0, s>>>(M, g.nth, g.nrow_half, nzc, (const float2*)p->d_h, (float2*)p->d_z);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_phi, s));
    if (f64) NUSHT_CUFFT_TRY(cufftExecZ2D(p->fft_phi, (cufftDoubleComplex*)p->d_z, (double*)p->d_grid));
    else NUSHT_CUFFT_TRY(cufftExecC2R(p->fft_phi, (cufftComplex*)p->d_z, (float*)p->d_grid));
    REC(4);
    return NUSHT_OK;
}

static int fourier_adjoint_general(nusht_plan_s* p, cudaStream_t s, cudaEvent_t* ev) {
    const int L = p->lmax, M = p->mmax;
    const NufftGeom& g = p->ng;
    const int nth2 = p->lg.nth2, nzc = g.nph / 2 + 1;
    const bool f64 = p->dtype == NUSHT_F64;
    REC(0);
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_phi_r2c, s));
    if (f64) NUSHT_CUFFT_TRY(cufftExecD2Z(p->fft_phi_r2c, (double*)p->d_grid, (cufftDoubleComplex*)p->d_z));
    else NUSHT_CUFFT_TRY(cufftExecR2C(p->fft_phi_r2c, (float*)p->d_grid, (cufftComplex*)p->d_z));
    {
        dim3 grid((g.nth + 31) / 32, (M + 32) / 32);
        if (f64) k_zc_to_h<double2><<<grid, 256, 0, s>>>(M, g.nth, g.nrow_half, nzc, (const double2*)p->d_z, (double2*)p->d_h);
        else k_zc_to_h<float2><<<grid, 256, 0, s>>>(M, g.nth, g.nrow_half, nzc, (const float2*)p->d_z, (float2*)p->d_h);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    REC(1);
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_theta_fine, s));
    if (f64) NUSHT_CUFFT_TRY(cufftExecZ2Z(p->fft_theta_fine, (cufftDoubleComplex*)p->d_h, (cufftDoubleComplex*)p->d_h, CUFFT_FORWARD));
    else NUSHT_CUFFT_TRY(cufftExecC2C(p->fft_theta_fine, (cufftComplex*)p->d_h, (cufftComplex*)p->d_h, CUFFT_FORWARD));
    REC(2);
    {
        dim3 grid((nth2 + 255) / 256, M + 1);
        if (f64) k_deconv_trunc_gen<double><<<grid, 256, 0, s>>>(L, M, nth2, g.nth, (const double2*)p->d_h, p->d_pth, p->d_pph, p->d_ft);
        else k_deconv_trunc_gen<float><<<grid, 256, 0, s>>>(L, M, nth2, g.nth, (const float2*)p->d_h, p->d_pth, p->d_pph, p->d_ft);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    REC(3);
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_theta_coarse, s));
    NUSHT_CUFFT_TRY(cufftExecZ2Z(p->fft_theta_coarse, (cufftDoubleComplex*)p->d_ft, (cufftDoubleComplex*)p->d_ft, CUFFT_INVERSE));
    REC(4);
    return NUSHT_OK;
}

int fourier_synthesis(nusht_plan_s* p, cudaStream_t s, cudaEvent_t* ev) {
    if (p->fourier_general) return fourier_synthesis_general(p, s, ev);
    const int L = p->lmax, M = p->mmax;
    const NufftGeom& g = p->ng;
    const int nth2 = p->lg.nth2;
    const bool f64 = p->dtype == NUSHT_F64;
    REC(0);
    if (p->theta_fused) {
        REC(1);
        REC(2);
        if (f64)
            NUSHT_TRY(dispatch_chain<double2>(p, false, (double2*)p->d_h, s));
        else
            NUSHT_TRY(dispatch_chain<float2>(p, false, (float2*)p->d_h, s));
    } else {
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_theta_coarse, s));
    NUSHT_CUFFT_TRY(cufftExecZ2Z(p->fft_theta_coarse, (cufftDoubleComplex*)p->d_ft, (cufftDoubleComplex*)p->d_ft,
                                 CUFFT_FORWARD));
    REC(1);
    {
        dim3 grid((g.nth / 2 + 255) / 256, M + 1);
        if (f64)
            k_deconv_pad<double><<<grid, 256, 0, s>>>(L, M, nth2, g.nth / 2, p->d_ft, p->d_pth, p->d_pph, (double2*)p->d_h);
        else
            k_deconv_pad<float><<<grid, 256, 0, s>>>(L, M, nth2, g.nth / 2, p->d_ft, p->d_pth, p->d_pph, (float2*)p->d_h);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    REC(2);
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_theta_fine, s));
    if (f64)
        NUSHT_CUFFT_TRY(cufftExecZ2Z(p->fft_theta_fine, (cufftDoubleComplex*)p->d_h, (cufftDoubleComplex*)p->d_h,
                                     CUFFT_INVERSE));
    else
        NUSHT_CUFFT_TRY(cufftExecC2C(p->fft_theta_fine, (cufftComplex*)p->d_h, (cufftComplex*)p->d_h, CUFFT_INVERSE));
    }
    REC(3);
    if (p->phi_fused_syn) {
        if (f64) NUSHT_TRY(dispatch_phi<double2>(p, false, s));
        else NUSHT_TRY(dispatch_phi<float2>(p, false, s));
        REC(4);
        return NUSHT_OK;
    }
    {
        // H -> pre-processed rows of the grid buffer, then one in-place complex transform per row
        const int nz = g.nph / 2;
        dim3 grid(2 * ((g.nth / 2 + 31) / 32), (M + 32) / 32);
        if (f64)
            k_h_to_z<double2><<<grid, 256, 0, s>>>(M, g.nth / 2, g.nrow_half, nz, p->d_twz, (const double2*)p->d_h,
                                                    (double2*)p->d_grid);
        else
            k_h_to_z<float2><<<grid, 256, 0, s>>>(M, g.nth / 2, g.nrow_half, nz, p->d_twz, (const float2*)p->d_h,
                                                   (float2*)p->d_grid);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_phi, s));
    if (f64)
        NUSHT_CUFFT_TRY(cufftExecZ2Z(p->fft_phi, (cufftDoubleComplex*)p->d_grid, (cufftDoubleComplex*)p->d_grid,
                                     CUFFT_INVERSE));
    else
        NUSHT_CUFFT_TRY(cufftExecC2C(p->fft_phi, (cufftComplex*)p->d_grid, (cufftComplex*)p->d_grid, CUFFT_INVERSE));
    REC(4);
    return NUSHT_OK;
}

// adjoint: d_grid -> d_ft (Gtilde).  ev[0] before R2C, ev[1] after R2C, ev[2] after fine theta FFT,
// ev[3] after truncate/deconvolve, ev[4] after the coarse inverse FFT.
int fourier_adjoint(nusht_plan_s* p, cudaStream_t s, cudaEvent_t* ev) {
    if (p->fourier_general) return fourier_adjoint_general(p, s, ev);
    const int L = p->lmax, M = p->mmax;
    const NufftGeom& g = p->ng;
    const int nth2 = p->lg.nth2;
    const bool f64 = p->dtype == NUSHT_F64;
    REC(0);
    if (p->phi_fused) {
        if (f64) NUSHT_TRY(dispatch_phi<double2>(p, true, s));
        else NUSHT_TRY(dispatch_phi<float2>(p, true, s));
    } else {
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_phi, s));
    if (f64)
        NUSHT_CUFFT_TRY(cufftExecZ2Z(p->fft_phi, (cufftDoubleComplex*)p->d_grid, (cufftDoubleComplex*)p->d_grid,
                                     CUFFT_FORWARD));
    else
        NUSHT_CUFFT_TRY(cufftExecC2C(p->fft_phi, (cufftComplex*)p->d_grid, (cufftComplex*)p->d_grid, CUFFT_FORWARD));
    }
    if (!p->phi_fused) {
        // post-processing + transpose to H[m][parity][a'], zero-extended in theta to the full period
        const int nz = g.nph / 2;
        dim3 grid(2 * ((g.nth / 2 + 31) / 32), (M + 32) / 32);
        if (f64)
            k_z_to_h<double2><<<grid, 256, 0, s>>>(M, g.nth / 2, g.nrow_half, nz, !p->theta_fused, p->d_twz, (const double2*)p->d_grid,
                                                    (double2*)p->d_h);
        else
            k_z_to_h<float2><<<grid, 256, 0, s>>>(M, g.nth / 2, g.nrow_half, nz, !p->theta_fused, p->d_twz, (const float2*)p->d_grid,
                                                   (float2*)p->d_h);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    REC(1);
    if (p->theta_fused) {
        if (f64)
            NUSHT_TRY(dispatch_chain<double2>(p, true, (double2*)p->d_h, s));
        else
            NUSHT_TRY(dispatch_chain<float2>(p, true, (float2*)p->d_h, s));
        REC(2);
        REC(3);
        REC(4);
        return NUSHT_OK;
    }
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_theta_fine, s));
    if (f64)
        NUSHT_CUFFT_TRY(cufftExecZ2Z(p->fft_theta_fine, (cufftDoubleComplex*)p->d_h, (cufftDoubleComplex*)p->d_h,
                                     CUFFT_FORWARD));
    else
        NUSHT_CUFFT_TRY(cufftExecC2C(p->fft_theta_fine, (cufftComplex*)p->d_h, (cufftComplex*)p->d_h, CUFFT_FORWARD));
    REC(2);
    {
        dim3 grid((nth2 + 255) / 256, M + 1);
        if (f64)
            k_deconv_trunc<double><<<grid, 256, 0, s>>>(L, M, nth2, g.nth / 2, (const double2*)p->d_h, p->d_pth, p->d_pph,
                                                        p->d_ft);
        else
            k_deconv_trunc<float><<<grid, 256, 0, s>>>(L, M, nth2, g.nth / 2, (const float2*)p->d_h, p->d_pth, p->d_pph,
                                                       p->d_ft);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    REC(3);
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_theta_coarse, s));
    NUSHT_CUFFT_TRY(cufftExecZ2Z(p->fft_theta_coarse, (cufftDoubleComplex*)p->d_ft, (cufftDoubleComplex*)p->d_ft,
                                 CUFFT_INVERSE));
    REC(4);
    return NUSHT_OK;
}
#undef REC

void fourier_free(nusht_plan_s* p) {
    if (p->fft_theta_coarse) cufftDestroy(p->fft_theta_coarse);
    if (p->fft_theta_fine) cufftDestroy(p->fft_theta_fine);
    if (p->fft_phi) cufftDestroy(p->fft_phi);
    if (p->fft_phi_r2c) cufftDestroy(p->fft_phi_r2c);
    p->fft_theta_coarse = p->fft_theta_fine = p->fft_phi = p->fft_phi_r2c = 0;
    cudaFree(p->d_z);
    cudaFree(p->d_phitab);
    p->d_phitab = nullptr;
    cudaFree(p->d_fftwork);
    p->d_z = nullptr;
    p->d_fftwork = nullptr;
    if (p->d_grid == p->d_h) p->d_grid = nullptr;      // sigma != 2: one allocation
    cudaFree(p->d_pth); cudaFree(p->d_pph); cudaFree(p->d_h); cudaFree(p->d_twz); cudaFree(p->d_grid); cudaFree(p->d_tw2n);
    p->d_tw2n = nullptr;
    p->d_pth = p->d_pph = nullptr;
    p->d_h = p->d_grid = nullptr;
    p->d_twz = nullptr;
}
