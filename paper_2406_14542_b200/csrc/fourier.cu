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

#include <vector>

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

// a5 / a9 layout change between the theta pass (H[m][parity][a'], a = 2a' + parity) and the phi pass
// (Ht[a][m], m contiguous, row length mp = n_phi/2 + 1): 32 x 32 tiles through shared memory.
// Only rows a <= n_theta/2 (theta in [0, pi]) and columns m <= mmax are moved.
template <typename C>
__global__ void __launch_bounds__(256)
k_h_to_ht(int M, int nh, int nrow_half, int mp, const C* __restrict__ h, C* __restrict__ ht) {
    __shared__ C tile[32][33];
    // blockIdx.x enumerates (parity, 32 values of a')
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
        if (m <= M && ap0 + r < nh && a < nrow_half) ht[(int64_t)a * mp + m] = tile[tx][r];
    }
}

// transpose back, fused with the zero-extension of the theta axis to the full period (the
// transpose of "keep rows 0 .. n_theta/2"): H[m][parity][a'] = Ht[2a' + parity][m] for rows <= n_theta/2, 0 beyond
template <typename C>
__global__ void __launch_bounds__(256)
k_ht_to_h(int M, int nh, int nrow_half, int mp, const C* __restrict__ ht, C* __restrict__ h) {
    __shared__ C tile[32][33];
    const int nblk = (nh + 31) / 32;
    const int par = blockIdx.x / nblk, ap0 = (blockIdx.x % nblk) * 32, m0 = blockIdx.y * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int a = 2 * (ap0 + r) + par, m = m0 + tx;
        if (m <= M && a < nrow_half) tile[r][tx] = ht[(int64_t)a * mp + m];
    }
    __syncthreads();
    C zero;
    zero.x = 0;
    zero.y = 0;
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
        const int m = m0 + r, ap = ap0 + tx;
        if (m <= M && ap < nh) h[((int64_t)m * 2 + par) * nh + ap] = (2 * ap + par < nrow_half) ? tile[tx][r] : zero;
    }
}

// plan-time probe: does any word of columns m > M of Ht differ from zero?
__global__ void k_tail_nonzero(int M, int nrow_half, int mp, int words_per_elem, const unsigned long long* __restrict__ ht,
                               int* __restrict__ flag) {
    const int64_t tail = (int64_t)(mp - M - 1) * words_per_elem;
    const int64_t total = (int64_t)nrow_half * tail;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const int64_t a = i / tail, q = i - a * tail;
        if (ht[(a * mp + M + 1) * words_per_elem + q] != 0ull) *flag = 1;
    }
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
    for (int k = 0; k <= L; ++k) {
        const double v = 1.0 / (nufft_kernel_ft(p, (double)k, g.nth) * (double)nth2);
        pth[L + k] = v;
        pth[L - k] = v;
    }
    for (int m = 0; m <= M; ++m) pph[m] = 1.0 / nufft_kernel_ft(p, (double)m, g.nph);
    NUSHT_TRY(f_alloc(&p->d_pth, sizeof(double) * (2 * L + 1), p));
    NUSHT_TRY(f_alloc(&p->d_pph, sizeof(double) * (M + 1), p));
    NUSHT_CUDA_TRY(cudaMemcpy(p->d_pth, pth.data(), sizeof(double) * (2 * L + 1), cudaMemcpyHostToDevice));
    NUSHT_CUDA_TRY(cudaMemcpy(p->d_pph, pph.data(), sizeof(double) * (M + 1), cudaMemcpyHostToDevice));

    const int mp = g.nph / 2 + 1;
    const size_t hbytes = (size_t)(M + 1) * (size_t)g.nth * csz;
    const size_t htbytes = (size_t)g.nrow_half * (size_t)mp * csz;
    const size_t gbytes = (size_t)g.nrow_half * (size_t)g.nph * rsz;
    NUSHT_TRY(f_alloc(&p->d_h, hbytes, p));
    NUSHT_TRY(f_alloc(&p->d_ht, htbytes, p));
    NUSHT_TRY(f_alloc(&p->d_ht_adj, htbytes, p));   // R2C output of the adjoint (fills columns m > mmax too)
    NUSHT_TRY(f_alloc(&p->d_grid, gbytes, p));
    NUSHT_CUDA_TRY(cudaMemset(p->d_h, 0, hbytes));
    NUSHT_CUDA_TRY(cudaMemset(p->d_ht, 0, htbytes));
    NUSHT_CUDA_TRY(cudaMemset(p->d_grid, 0, gbytes));

    // cuFFT plans
    size_t ws = 0, wtot = 0;
    {
        int n[1] = {nth2};
        NUSHT_CUFFT_TRY(cufftCreate(&p->fft_theta_coarse));
        NUSHT_CUFFT_TRY(cufftMakePlanMany(p->fft_theta_coarse, 1, n, nullptr, 1, nth2, nullptr, 1, nth2, CUFFT_Z2Z,
                                          M + 1, &ws));
        wtot += ws;
    }
    {
        int n[1] = {g.nth / 2};   // two half-length transforms per m (see k_deconv_pad)
        NUSHT_CUFFT_TRY(cufftCreate(&p->fft_theta_fine));
        NUSHT_CUFFT_TRY(cufftMakePlanMany(p->fft_theta_fine, 1, n, nullptr, 1, g.nth / 2, nullptr, 1, g.nth / 2,
                                          f64 ? CUFFT_Z2Z : CUFFT_C2C, 2 * (M + 1), &ws));
        wtot += ws;
    }
    {
        // phi pass on the transposed buffer Ht[a][m]: contiguous rows of mp complex <-> n_phi reals
        int n[1] = {g.nph};
        int inembed[1] = {mp}, onembed[1] = {g.nph};
        NUSHT_CUFFT_TRY(cufftCreate(&p->fft_phi_c2r));
        NUSHT_CUFFT_TRY(cufftMakePlanMany(p->fft_phi_c2r, 1, n, inembed, 1, mp, onembed, 1, g.nph,
                                          f64 ? CUFFT_Z2D : CUFFT_C2R, g.nrow_half, &ws));
        wtot += ws;
        NUSHT_CUFFT_TRY(cufftCreate(&p->fft_phi_r2c));
        NUSHT_CUFFT_TRY(cufftMakePlanMany(p->fft_phi_r2c, 1, n, onembed, 1, g.nph, inembed, 1, mp,
                                          f64 ? CUFFT_D2Z : CUFFT_R2C, g.nrow_half, &ws));
        wtot += ws;
    }
    // Columns m > mmax of Ht are zero and must stay so for the C2R.  cuFFT is allowed to overwrite the
    // input of an out-of-place C2R: probe once whether this plan does; if it does, they are re-zeroed
    // on every synthesis, otherwise never again.
    p->c2r_clobbers_input = false;
    if (mp - M - 1 > 0) {
        int* d_flag = nullptr;
        NUSHT_CUDA_TRY(cudaMalloc((void**)&d_flag, sizeof(int)));
        NUSHT_CUDA_TRY(cudaMemset(d_flag, 0, sizeof(int)));
        NUSHT_CUDA_TRY(cudaMemset2D(p->d_ht, (size_t)mp * csz, 0x3c, (size_t)(M + 1) * csz, (size_t)g.nrow_half));
        if (f64)
            NUSHT_CUFFT_TRY(cufftExecZ2D(p->fft_phi_c2r, (cufftDoubleComplex*)p->d_ht, (cufftDoubleReal*)p->d_grid));
        else
            NUSHT_CUFFT_TRY(cufftExecC2R(p->fft_phi_c2r, (cufftComplex*)p->d_ht, (cufftReal*)p->d_grid));
        k_tail_nonzero<<<1024, 256>>>(M, g.nrow_half, mp, (int)(csz / 8), (const unsigned long long*)p->d_ht, d_flag);
        int flag = 0;
        NUSHT_CUDA_TRY(cudaMemcpy(&flag, d_flag, sizeof(int), cudaMemcpyDeviceToHost));
        cudaFree(d_flag);
        p->c2r_clobbers_input = flag != 0;
        NUSHT_CUDA_TRY(cudaMemset(p->d_ht, 0, htbytes));
        NUSHT_CUDA_TRY(cudaMemset(p->d_grid, 0, gbytes));
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
int fourier_synthesis(nusht_plan_s* p, cudaStream_t s, cudaEvent_t* ev) {
    const int L = p->lmax, M = p->mmax;
    const NufftGeom& g = p->ng;
    const int nth2 = p->lg.nth2;
    const bool f64 = p->dtype == NUSHT_F64;
    const size_t csz = f64 ? 16 : 8;
    REC(0);
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
        NUSHT_CUDA_TRY(cudaGetLastError());
    }
    REC(2);
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_theta_fine, s));
    if (f64)
        NUSHT_CUFFT_TRY(cufftExecZ2Z(p->fft_theta_fine, (cufftDoubleComplex*)p->d_h, (cufftDoubleComplex*)p->d_h,
                                     CUFFT_INVERSE));
    else
        NUSHT_CUFFT_TRY(cufftExecC2C(p->fft_theta_fine, (cufftComplex*)p->d_h, (cufftComplex*)p->d_h, CUFFT_INVERSE));
    REC(3);
    {
        // H[m][a] -> Ht[a][m] (rows theta in [0, pi] only), then the phi C2R on contiguous rows
        const int mp = g.nph / 2 + 1;
        dim3 grid(2 * ((g.nth / 2 + 31) / 32), (M + 32) / 32);
        if (f64)
            k_h_to_ht<double2><<<grid, 256, 0, s>>>(M, g.nth / 2, g.nrow_half, mp, (const double2*)p->d_h, (double2*)p->d_ht);
        else
            k_h_to_ht<float2><<<grid, 256, 0, s>>>(M, g.nth / 2, g.nrow_half, mp, (const float2*)p->d_h, (float2*)p->d_ht);
        NUSHT_CUDA_TRY(cudaGetLastError());
        if (p->c2r_clobbers_input && mp - M - 1 > 0)
            NUSHT_CUDA_TRY(cudaMemset2DAsync((char*)p->d_ht + (size_t)(M + 1) * csz, (size_t)mp * csz, 0,
                                             (size_t)(mp - M - 1) * csz, (size_t)g.nrow_half, s));
    }
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_phi_c2r, s));
    if (f64)
        NUSHT_CUFFT_TRY(cufftExecZ2D(p->fft_phi_c2r, (cufftDoubleComplex*)p->d_ht, (cufftDoubleReal*)p->d_grid));
    else
        NUSHT_CUFFT_TRY(cufftExecC2R(p->fft_phi_c2r, (cufftComplex*)p->d_ht, (cufftReal*)p->d_grid));
    REC(4);
    return NUSHT_OK;
}

// adjoint: d_grid -> d_ft (Gtilde).  ev[0] before R2C, ev[1] after R2C, ev[2] after fine theta FFT,
// ev[3] after truncate/deconvolve, ev[4] after the coarse inverse FFT.
int fourier_adjoint(nusht_plan_s* p, cudaStream_t s, cudaEvent_t* ev) {
    const int L = p->lmax, M = p->mmax;
    const NufftGeom& g = p->ng;
    const int nth2 = p->lg.nth2;
    const bool f64 = p->dtype == NUSHT_F64;
    const size_t csz = f64 ? 16 : 8;
    REC(0);
    NUSHT_CUFFT_TRY(cufftSetStream(p->fft_phi_r2c, s));
    if (f64)
        NUSHT_CUFFT_TRY(cufftExecD2Z(p->fft_phi_r2c, (cufftDoubleReal*)p->d_grid, (cufftDoubleComplex*)p->d_ht_adj));
    else
        NUSHT_CUFFT_TRY(cufftExecR2C(p->fft_phi_r2c, (cufftReal*)p->d_grid, (cufftComplex*)p->d_ht_adj));
    {
        // Ht[a][m] -> H[m][a] for m <= mmax, zero-extended in theta to the full period
        const int mp = g.nph / 2 + 1;
        dim3 grid(2 * ((g.nth / 2 + 31) / 32), (M + 32) / 32);
        if (f64)
            k_ht_to_h<double2><<<grid, 256, 0, s>>>(M, g.nth / 2, g.nrow_half, mp, (const double2*)p->d_ht_adj, (double2*)p->d_h);
        else
            k_ht_to_h<float2><<<grid, 256, 0, s>>>(M, g.nth / 2, g.nrow_half, mp, (const float2*)p->d_ht_adj, (float2*)p->d_h);
        NUSHT_CUDA_TRY(cudaGetLastError());
    }
    REC(1);
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
        NUSHT_CUDA_TRY(cudaGetLastError());
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
    if (p->fft_phi_c2r) cufftDestroy(p->fft_phi_c2r);
    if (p->fft_phi_r2c) cufftDestroy(p->fft_phi_r2c);
    p->fft_theta_coarse = p->fft_theta_fine = p->fft_phi_c2r = p->fft_phi_r2c = 0;
    cudaFree(p->d_pth); cudaFree(p->d_pph); cudaFree(p->d_h); cudaFree(p->d_ht); cudaFree(p->d_ht_adj); cudaFree(p->d_grid);
    p->d_pth = p->d_pph = nullptr;
    p->d_h = p->d_ht = p->d_ht_adj = p->d_grid = nullptr;
}
