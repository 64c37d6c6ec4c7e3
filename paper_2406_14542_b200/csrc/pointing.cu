// pointing.cu -- deflected positions for CMB weak lensing (arXiv 2406.14542 Appendix C, Eq. C1,
// PAPER.md:303-314, the Eq. C1 half: the deflection field (alpha_theta, alpha_phi)
// of Eq. C2 is an input here).
//
//   n' = cos(a) n + (sin(a)/a) (a_theta e_theta + a_phi e_phi),   a = sqrt(a_theta^2 + a_phi^2)
//   n = (sin t cos p, sin t sin p, cos t),  e_theta = (cos t cos p, cos t sin p, -sin t),  e_phi = (-sin p, cos p, 0)
//   theta' = atan2(|n'_xy|, n'_z),  phi' = atan2(n'_y, n'_x) mod 2 pi
//
// One thread per point, FP64 throughout ("double precision accuracy on the pointing").  The x and y
// components are formed in the frame rotated by -phi about z (u = n'.(cos p, sin p, 0), v = n'.e_phi), so that
// phi' = phi + atan2(v, u): two sincos instead of three and no cancellation in phi' for small deflections.
// HBM floor: 4 loads + 2 stores of 8 bytes per point, all coalesced; what binds is the issue rate of the FP64
// elementary functions (the first version: two sincos, two atan2, two sqrt, a division, about 500 instructions per
// point).  Lensing deflections are arcminutes, so the common case is served by short series and the
// general functions stay for the rest, per lane:
//   * sin(a)/a and cos(a) as even polynomials in a^2 for a < 1/4 (no sqrt, no sincos, no division);
//   * theta' = theta + atan2(rho cos t - z sin t, z cos t + rho sin t), rho = |n'_xy| (the rotation angle in the
//     meridian plane of n'), and phi' = phi + atan2(v, u): both arguments are small unless the point sits next to a
//     pole, and atan(x) is a 6-term odd series for |x| < 0.03 (truncation 4e-20).
// The CPU oracle (oracle/oracle.py) writes out the Cartesian form of Eq. C1 in long double and shares nothing with
// this file.
#include <math.h>

#include "nusht_internal.cuh"

namespace {

constexpr double PT_TWO_PI = 6.283185307179586476925286766559;
constexpr double PT_PI = 3.14159265358979323846;
constexpr int PT_THREADS = 256;

// atan(x) for |x| < 0.03: x (1 - x^2/3 + x^4/5 - x^6/7 + x^8/9 - x^10/11), next term 0.03^12 / 13 = 4e-20
__device__ __forceinline__ double atan_small(double x) {
    const double y = x * x;
    double p = -1.0 / 11.0;
    p = fma(p, y, 1.0 / 9.0);
    p = fma(p, y, -1.0 / 7.0);
    p = fma(p, y, 1.0 / 5.0);
    p = fma(p, y, -1.0 / 3.0);
    return fma(x * y, p, x);
}

__global__ void __launch_bounds__(PT_THREADS)
k_pointing(int64_t npts, const double* __restrict__ theta, const double* __restrict__ phi,
           const double* __restrict__ a_theta, const double* __restrict__ a_phi, double* theta_out,
           double* phi_out) {
    const int64_t stride = (int64_t)gridDim.x * PT_THREADS;
    for (int64_t i = (int64_t)blockIdx.x * PT_THREADS + threadIdx.x; i < npts; i += stride) {
        const double t = theta[i], p = phi[i], at = a_theta[i], ap = a_phi[i];
        const double a2 = fma(at, at, ap * ap);           // angles: no overflow to guard against
        double st, ct, sinc, ca;
        sincos(t, &st, &ct);
        if (a2 < 0.0625) {
            // sin(a)/a = sum (-a^2)^k / (2k+1)!,  cos(a) = sum (-a^2)^k / (2k)!;  a^2 <= 1/16: 7 and 8 terms reach 1e-17
            double q = 1.0 / 6227020800.0;                     // 1/13!
            q = fma(q, -a2, 1.0 / 39916800.0);                 // 1/11!
            q = fma(q, -a2, 1.0 / 362880.0);                   // 1/9!
            q = fma(q, -a2, 1.0 / 5040.0);
            q = fma(q, -a2, 1.0 / 120.0);
            q = fma(q, -a2, 1.0 / 6.0);
            sinc = fma(q, -a2, 1.0);
            double c = 1.0 / 87178291200.0;                    // 1/14!
            c = fma(c, -a2, 1.0 / 479001600.0);                // 1/12!
            c = fma(c, -a2, 1.0 / 3628800.0);                  // 1/10!
            c = fma(c, -a2, 1.0 / 40320.0);
            c = fma(c, -a2, 1.0 / 720.0);
            c = fma(c, -a2, 1.0 / 24.0);
            c = fma(c, -a2, 0.5);
            ca = fma(c, -a2, 1.0);
        } else {
            const double a = sqrt(a2);
            double sa;
            sincos(a, &sa, &ca);
            sinc = sa / a;
        }
        // components of n' along (cos p, sin p, 0), e_phi and z
        const double bt = sinc * at;
        const double u = fma(ca, st, bt * ct);
        const double v = sinc * ap;
        const double z = fma(ca, ct, -bt * st);
        const double rho = sqrt(fma(u, u, v * v));
        // theta' = atan2(rho, z) = theta + (angle from n to n' in the meridian plane of n')
        // (two rounded products, not an FMA: with zero deflection rho = sin t and z = cos t exactly, and the
        //  difference must then be exactly zero so that theta' == theta)
        const double sd = __dsub_rn(__dmul_rn(rho, ct), __dmul_rn(z, st)), cd = fma(z, ct, rho * st);
        double t2;
        if (fabs(sd) < 0.03 * cd) t2 = t + atan_small(sd / cd);
        else t2 = atan2(rho, z);
        t2 = fmin(fmax(t2, 0.0), PT_PI);
        double p2 = p + ((fabs(v) < 0.03 * u) ? atan_small(v / u) : atan2(v, u));
        p2 -= PT_TWO_PI * floor(p2 * (1.0 / PT_TWO_PI));
        if (p2 < 0.0) p2 = 0.0;
        if (p2 >= PT_TWO_PI) p2 -= PT_TWO_PI;
        theta_out[i] = t2;
        phi_out[i] = p2;
    }
}

}  // namespace

extern "C" int nusht_pointing(int64_t npts, const double* theta, const double* phi, const double* alpha_theta,
                              const double* alpha_phi, double* theta_out, double* phi_out, void* stream) {
    if (npts < 0) return NUSHT_ERR_INVALID_ARG;
    if (npts == 0) return NUSHT_OK;
    if (!theta || !phi || !alpha_theta || !alpha_phi || !theta_out || !phi_out) return NUSHT_ERR_INVALID_ARG;
    int dev = 0, n_sm = 0;
    NUSHT_CUDA_TRY(cudaGetDevice(&dev));
    NUSHT_CUDA_TRY(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    // persistent grid: 8 CTAs of 256 threads per SM (all 2048 thread slots), grid-stride loop
    int64_t blocks = (npts + PT_THREADS - 1) / PT_THREADS;
    if (blocks > (int64_t)n_sm * 8) blocks = (int64_t)n_sm * 8;
    k_pointing<<<(unsigned)blocks, PT_THREADS, 0, (cudaStream_t)stream>>>(npts, theta, phi, alpha_theta, alpha_phi,
                                                                         theta_out, phi_out);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}
