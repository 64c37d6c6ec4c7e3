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
// HBM-bound: 4 loads + 2 stores of 8 bytes per point, all coalesced.  The CPU oracle (oracle/oracle.py) writes
// out the Cartesian form of Eq. C1 in long double and shares nothing with this file.
#include <math.h>

#include "nusht_internal.cuh"

namespace {

constexpr double PT_TWO_PI = 6.283185307179586476925286766559;
constexpr int PT_THREADS = 256;

__global__ void __launch_bounds__(PT_THREADS)
k_pointing(int64_t npts, const double* __restrict__ theta, const double* __restrict__ phi,
           const double* __restrict__ a_theta, const double* __restrict__ a_phi, double* theta_out,
           double* phi_out) {
    const int64_t stride = (int64_t)gridDim.x * PT_THREADS;
    for (int64_t i = (int64_t)blockIdx.x * PT_THREADS + threadIdx.x; i < npts; i += stride) {
        const double t = theta[i], p = phi[i], at = a_theta[i], ap = a_phi[i];
        const double a = sqrt(fma(at, at, ap * ap));      // angles: no overflow to guard against
        double st, ct, sa, ca;
        sincos(t, &st, &ct);
        sincos(a, &sa, &ca);
        const double sinc = (a > 0.0) ? sa / a : 1.0;
        // components of n' along (cos p, sin p, 0), e_phi and z
        const double u = fma(ca, st, sinc * at * ct);
        const double v = sinc * ap;
        const double z = fma(ca, ct, -sinc * at * st);
        const double t2 = atan2(sqrt(fma(u, u, v * v)), z);
        double p2 = p + atan2(v, u);
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
