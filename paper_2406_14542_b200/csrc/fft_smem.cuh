// fft_smem.cuh -- power-of-two complex FFT of one column held in shared memory, used by the fused
// theta chains of fourier.cu (SURVEY.md 8(a) rows a3-a5 theta / a9 theta).
//
// Structure (N = 2^k, 128 <= N <= 8192 in FP64): a decimation-in-frequency forward transform
//   stage 0   radix 2, fused with the load of the column from global memory,
//   stage i   radix 16 while the remaining sub-transform length is >= 16, then one radix 2/4/8 stage,
// leaves X[q] at the DIGIT-REVERSED position p (freq_of_pos below).  The inverse transform is the
// transposed (decimation-in-time) chain with conjugated twiddles: it takes digit-reversed input and
// produces natural order, so no permutation pass is ever executed: the spectrum is scaled, truncated
// and twiddled in place between the two.  Every stage keeps its butterfly (R complex numbers) in
// registers; stages exchange data through shared memory, element p at index p + p/16 (padding makes
// the stride-16 stage conflict-free).  Twiddles: one table W[j] = exp(-2 pi i j / (2N)), j < 2N
// (plan time, extended precision); the R-1 twiddles of a butterfly are powers of one table entry.
//
// The functions are __host__ __device__ so that the stage structure can be checked on a CPU by
// running the "threads" one after the other (tests/test_fft_smem_cpu.py builds such a harness).
#pragma once
#include <cuda_runtime.h>

namespace fftsm {

#define FFTSM_HD __host__ __device__ __forceinline__

FFTSM_HD int pad(int p) { return p + (p >> 4); }
__host__ __device__ constexpr int padded_len(int n) { return n + (n >> 4); }

FFTSM_HD double2 cmul(double2 a, double2 b) {
    return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
}
FFTSM_HD double2 cconj(double2 a) { return make_double2(a.x, -a.y); }

__host__ __device__ constexpr int bitrev(int j, int r) {   // reverse the log2(r) bits of j
    int out = 0;
    for (int b = 1; b < r; b <<= 1) {
        out = (out << 1) | (j & 1);
        j >>= 1;
    }
    return out;
}

// cos(2 pi j/16), sin(2 pi j/16), j = 0..7
FFTSM_HD double cos16(int j) {
    constexpr double C[8] = {1.0, 0.92387953251128673848, 0.70710678118654752440, 0.38268343236508977173,
                             0.0, -0.38268343236508977173, -0.70710678118654752440, -0.92387953251128673848};
    return C[j];
}
FFTSM_HD double sin16(int j) {
    constexpr double S[8] = {0.0, 0.38268343236508977173, 0.70710678118654752440, 0.92387953251128673848,
                             1.0, 0.92387953251128673848, 0.70710678118654752440, 0.38268343236508977173};
    return S[j];
}

// In-register DFT of R points, sign SIGN in the exponent; radix-2 DIF stages with compile-time
// twiddles.  Output j is left in x[bitrev(j, R)].
template <int R, int SIGN>
FFTSM_HD void dft_reg(double2 (&x)[R]) {
#pragma unroll
    for (int len = R; len >= 2; len >>= 1) {
#pragma unroll
        for (int b = 0; b < R; b += len) {
#pragma unroll
            for (int j = 0; j < len / 2; ++j) {
                const double2 u = x[b + j], v = x[b + j + len / 2];
                x[b + j] = make_double2(u.x + v.x, u.y + v.y);
                const double dx = u.x - v.x, dy = u.y - v.y;
                const int a = j * (16 / len);   // angle index: 2 pi a / 16
                if (a == 0) {
                    x[b + j + len / 2] = make_double2(dx, dy);
                } else if (a == 4) {            // multiply by SIGN * i
                    x[b + j + len / 2] = SIGN > 0 ? make_double2(-dy, dx) : make_double2(dy, -dx);
                } else {
                    const double c = cos16(a), s = SIGN * sin16(a);
                    x[b + j + len / 2] = make_double2(fma(dx, c, -dy * s), fma(dx, s, dy * c));
                }
            }
        }
    }
}

// frequency held at (unpadded) position p after the forward passes on a sub-transform of length NS
template <int NS>
FFTSM_HD int freq_of_pos_sub(int p) {
    if constexpr (NS >= 16) {
        return p / (NS / 16) + 16 * freq_of_pos_sub<NS / 16>(p % (NS / 16));
    } else {
        return p;   // a single stage of radix NS (or NS == 1)
    }
}
template <int N>
FFTSM_HD int freq_of_pos(int p) {
    return p / (N / 2) + 2 * freq_of_pos_sub<N / 2>(p % (N / 2));
}

// the inverse map: (unpadded) position that holds frequency q after the forward passes, i.e. where the inverse chain
// expects it.  Used by kernels that GENERATE a spectrum and can place each entry where the inverse transform wants it.
template <int NS>
FFTSM_HD int pos_of_freq_sub(int q) {
    if constexpr (NS >= 16) {
        return (q % 16) * (NS / 16) + pos_of_freq_sub<NS / 16>(q / 16);
    } else {
        return q;
    }
}
template <int N>
FFTSM_HD int pos_of_freq(int q) {
    return (q & 1) * (N / 2) + pos_of_freq_sub<N / 2>(q >> 1);
}

// One DIF stage of radix R on every sub-transform of length NS of the array (N elements, T threads).
// SIGN = -1: forward.  tw = stage table of NS/R entries exp(-2 pi i i/NS), i < NS/R (stage_table_offset).
template <int N, int R, int NS, int SIGN>
FFTSM_HD void stage_dif(double2* s, int tid, int T, const double2* __restrict__ tw) {
    constexpr int SUB = NS / R;
#pragma unroll 1
    for (int b = tid; b < N / R; b += T) {
        const int i = b % SUB, base = (b / SUB) * NS + i;
        double2 x[R];
#pragma unroll
        for (int j = 0; j < R; ++j) x[j] = s[pad(base + j * SUB)];
        dft_reg<R, SIGN>(x);
        s[pad(base)] = x[0];
        if constexpr (SUB > 1) {
            double2 w1 = tw[i];                          // exp(-2 pi i i/NS)
            if (SIGN > 0) w1 = cconj(w1);
            double2 w = w1;
#pragma unroll
            for (int j = 1; j < R; ++j) {
                s[pad(base + j * SUB)] = cmul(x[bitrev(j, R)], w);
                if (j + 1 < R) w = cmul(w, w1);
            }
        } else {
#pragma unroll
            for (int j = 1; j < R; ++j) s[pad(base + j * SUB)] = x[bitrev(j, R)];
        }
    }
}

// The transposed stage (decimation in time): twiddle the inputs, then the R-point DFT.
template <int N, int R, int NS, int SIGN>
FFTSM_HD void stage_dit(double2* s, int tid, int T, const double2* __restrict__ tw) {
    constexpr int SUB = NS / R;
#pragma unroll 1
    for (int b = tid; b < N / R; b += T) {
        const int i = b % SUB, base = (b / SUB) * NS + i;
        double2 x[R];
        x[0] = s[pad(base)];
        if constexpr (SUB > 1) {
            double2 w1 = tw[i];
            if (SIGN > 0) w1 = cconj(w1);
            double2 w = w1;
#pragma unroll
            for (int j = 1; j < R; ++j) {
                x[j] = cmul(s[pad(base + j * SUB)], w);
                if (j + 1 < R) w = cmul(w, w1);
            }
        } else {
#pragma unroll
            for (int j = 1; j < R; ++j) x[j] = s[pad(base + j * SUB)];
        }
        dft_reg<R, SIGN>(x);
#pragma unroll
        for (int j = 0; j < R; ++j) s[pad(base + j * SUB)] = x[bitrev(j, R)];
    }
}

// Compact per-stage twiddle tables, concatenated: the stage on sub-transforms of length NS (radix
// 16, NS >= 32) reads NS/16 entries exp(-2 pi i i/NS) starting at stage_table_offset(N, NS).
__host__ __device__ constexpr int stage_table_offset(int n, int ns) {
    int off = 0;
    for (int s = n / 2; s > ns; s /= 16) off += s / 16;
    return off;
}
__host__ __device__ constexpr int stage_table_len(int n) {
    int off = 0;
    for (int s = n / 2; s >= 32; s /= 16) off += s / 16;
    return off;
}

// radix of the last forward stage (= first inverse stage) on sub-transforms of length NS0 = N/2; its
// stride is 1, it has no twiddles, and thread `tid` of T owns butterflies b = tid + T u: positions R b + j.
__host__ __device__ constexpr int last_radix(int ns0) {
    int ns = ns0;
    while (ns > 16) ns /= 16;
    return ns;   // 16 when ns0 is a power of 16, else 2, 4 or 8
}

// last forward stage: shared memory -> registers (c[u * R + j] = output j of butterfly tid + T u)
template <int N, int R, int SIGN, int E>
FFTSM_HD void last_stage_to_regs(const double2* s, int tid, int T, double2 (&c)[E]) {
#pragma unroll
    for (int u = 0; u < E / R; ++u) {
        const int base = (tid + T * u) * R;
        double2 x[R];
#pragma unroll
        for (int j = 0; j < R; ++j) x[j] = s[pad(base + j)];
        dft_reg<R, SIGN>(x);
#pragma unroll
        for (int j = 0; j < R; ++j) c[u * R + j] = x[bitrev(j, R)];
    }
}
// first inverse stage: registers -> shared memory
template <int N, int R, int SIGN, int E>
FFTSM_HD void first_stage_from_regs(double2* s, int tid, int T, const double2 (&c)[E]) {
#pragma unroll
    for (int u = 0; u < E / R; ++u) {
        const int base = (tid + T * u) * R;
        double2 x[R];
#pragma unroll
        for (int j = 0; j < R; ++j) x[j] = c[u * R + j];
        dft_reg<R, SIGN>(x);
#pragma unroll
        for (int j = 0; j < R; ++j) s[pad(base + j)] = x[bitrev(j, R)];
    }
}

// Stage drivers.  Exec supplies `template <int R, int NS> void dif()` / `dit()`: run one stage for
// all threads and synchronise (the device executor of fourier.cu; a sequential loop on the host).
// The last forward / first inverse stage (sub-transform length last_radix) is NOT run by these: the
// caller does it between shared memory and registers with the two functions above.
template <int NS, class Exec>
FFTSM_HD void forward_stages(Exec& ex) {   // after the fused radix-2 stage: sub-transforms of length NS
    if constexpr (NS > 16) {
        ex.template dif<16, NS>();
        forward_stages<NS / 16>(ex);
    }
}
template <int NS, class Exec>
FFTSM_HD void inverse_stages(Exec& ex) {   // mirror image; the fused radix-2 stage follows
    if constexpr (NS > 16) {
        inverse_stages<NS / 16>(ex);
        ex.template dit<16, NS>();
    }
}

}  // namespace fftsm
