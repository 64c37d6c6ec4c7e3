// fft_reg.cuh -- register-tiled complex FFT of 4096 = 16 x 16 x 16 points by 256 threads, the core of the fused
// phi transform of fourier.cu at n_phi / 2 = 8192.
//
// fft_smem.cuh runs every radix-16 stage from and to shared memory (five sweeps of the array per 8192-point
// transform).  Here a thread keeps its 16 points in registers through all three stages and shared memory is only the
// exchange between them (two sweeps):
//   index i = i0 + 16 i1 + 256 i2,  frequency q = a + 16 b + 256 c  (all digits 0..15)
//   stage 1  thread (i0, i1) holds i2 = 0..15:  DFT16 over i2 -> a,  times W_4096^{(i0 + 16 i1) a}
//   exchange thread (i0, i1) writes [t + 256 a], thread (i0, a) reads i1 = 0..15 at [i0 + 16 i1 + 256 a]
//   stage 2  DFT16 over i1 -> b,  times W_256^{i0 b}
//   exchange thread (i0, a) writes [t + 256 b], thread (a, b) reads i0 = 0..15 at [16 t + i0]
//   stage 3  DFT16 over i0 -> c;  thread t = a + 16 b holds X[t + 256 c], c = 0..15
// so input AND output are in natural order with the thread index as the fast (coalesced) index: no digit reversal,
// and the inverse transform is the same code with the sign of the exponent flipped.  Element p of the exchange buffer
// sits at p + p/16 (fftsm::pad): the stride-16 reads of the second exchange are then conflict-free.
//
// The phases are separate __host__ __device__ functions so that tests/fft_smem_host_check.cu can run the "threads"
// one after the other on a CPU against a direct DFT.
#pragma once
#include "fft_smem.cuh"

namespace fftreg {

using fftsm::bitrev;
using fftsm::cconj;
using fftsm::cmul;
using fftsm::dft_reg;
using fftsm::pad;

constexpr int HLEN = 4096;                                  // points per transform
constexpr int HTHREADS = 256;                               // threads per transform
constexpr int HSMEM = HLEN + HLEN / 16;                     // padded exchange buffer, in double2

// multiply output k of a DFT16 (left at x[bitrev(k)]) by w1^k
template <int SIGN>
FFTSM_HD void twiddle16(double2 (&x)[16], double2 w1) {
    if (SIGN > 0) w1 = cconj(w1);
    double2 w = w1;
#pragma unroll
    for (int k = 1; k < 16; ++k) {
        x[bitrev(k, 16)] = cmul(x[bitrev(k, 16)], w);
        if (k + 1 < 16) w = cmul(w, w1);
    }
}

// phase A: stage 1 + first half of exchange 1.  x[i2] = input at index t + 256 i2.  tw4096[t] = exp(-2 pi i t/4096).
template <int SIGN>
FFTSM_HD void phase_a(double2 (&x)[16], double2* s, int t, const double2* __restrict__ tw4096) {
    dft_reg<16, SIGN>(x);
    twiddle16<SIGN>(x, tw4096[t]);
#pragma unroll
    for (int a = 0; a < 16; ++a) s[pad(t + 256 * a)] = x[bitrev(a, 16)];
}

// phase B1 (after a barrier): second half of exchange 1
FFTSM_HD void phase_b1(double2 (&x)[16], const double2* s, int t) {
    const int i0 = t & 15, a = t >> 4;
#pragma unroll
    for (int i1 = 0; i1 < 16; ++i1) x[i1] = s[pad(i0 + 16 * i1 + 256 * a)];
}

// phase B2 (after a barrier: every thread has read): stage 2 + first half of exchange 2.  tw256[i0] = exp(-2 pi i i0/256).
template <int SIGN>
FFTSM_HD void phase_b2(double2 (&x)[16], double2* s, int t, const double2* __restrict__ tw256) {
    dft_reg<16, SIGN>(x);
    twiddle16<SIGN>(x, tw256[t & 15]);
#pragma unroll
    for (int b = 0; b < 16; ++b) s[pad(t + 256 * b)] = x[bitrev(b, 16)];
}

// phase C (after a barrier): second half of exchange 2 + stage 3.  On return X[t + 256 c] is in x[bitrev(c)].
template <int SIGN>
FFTSM_HD void phase_c(double2 (&x)[16], const double2* s, int t) {
#pragma unroll
    for (int i0 = 0; i0 < 16; ++i0) x[i0] = s[pad(16 * t + i0)];
    dft_reg<16, SIGN>(x);
}

#ifdef __CUDACC__
// the whole transform for the 256 threads that share `s`; every thread of the CTA must call it (barriers)
template <int SIGN>
__device__ __forceinline__ void fft4096(double2 (&x)[16], double2* s, int t, const double2* __restrict__ tw4096,
                                        const double2* __restrict__ tw256) {
    phase_a<SIGN>(x, s, t, tw4096);
    __syncthreads();
    phase_b1(x, s, t);
    __syncthreads();
    phase_b2<SIGN>(x, s, t, tw256);
    __syncthreads();
    phase_c<SIGN>(x, s, t);
}
#endif

}  // namespace fftreg
