// legendre.cu -- ring Legendre stage of the nuSHT (operators S, D and their transposes; arXiv
// 2406.14542 Eq. 5-6).
//
//   synthesis:  F_m(theta_k) = sum_{l=m}^{lmax} a_lm Pbar_lm(theta_k) on the Clenshaw-Curtis rings
//               theta_k = pi k/(N_r-1), written directly in doubled (DFS) form
//               Ftilde[m][r] = F_m(theta_r) (r < N_r),  (-1)^m F_m(theta_{Ntheta-r}) (r >= N_r).
//   adjoint:    c_lm = sum_k Pbar_lm(theta_k) G_m[k],  G = fold(Gtilde)  (no quadrature weights).
//
// Pbar_lm is generated on the fly with the x^2-stepping recurrence of the paper's
// ref. [42] (Ishioka 2018), derived here from  x Pbar_l = c_{l+1} Pbar_{l+1} + c_l Pbar_{l-1},
// c_l^2 = (l^2-m^2)/(4 l^2-1):
//   even class  q_n = Pbar_{m+2n}:   q_{n+1} = A_n (x^2 - D_n) q_n - C_n q_{n-1}
//   scaled      q_n = sigma_n qh_n:  qh_{n+1} = (alpha_n x^2 + beta_n) qh_n + qh_{n-1}      (2 FMA)
//               evaluated as  t_n = (alpha_n + beta_n) - alpha_n sin^2(theta):  next to the poles x^2 = cos^2(theta)
//               rounds with an absolute error of 1e-16, the SAME error for every n of a ring, i.e. a coherent
//               shift of theta by 1e-16 / sin(2 theta) that grows to l * shift in the phase of Pbar_lm; sin^2 is
//               small there and carries a relative error instead.  Next to the EQUATOR the roles
//               swap (the x^2-stepping recurrence has double characteristic roots at theta = 0, pi/2 and pi): there
//               sin^2 is the one that rounds coherently, so blocks of ring pairs with theta >= pi/4 use
//               t_n = beta_n + alpha_n cos^2(theta).  Two tables, (-alpha_n, alpha_n + beta_n) and (alpha_n, beta_n);
//               a warp fetches its tiles from the one its block uses, and the per-pair operand table holds sin^2 or
//               cos^2 accordingly.  One FMA per step either way.
//   odd class   Pbar_{m+2n+1} = (x q_n - c_{m+2n} Pbar_{m+2n-1})/c_{m+2n+1}  is folded into the
//               coefficients once per transform (O(lmax^2)):  sum_n b_n Pbar_{m+2n+1} =
//               x sum_j (r_j/c_{m+2j+1}) q_j,  r_j = b_j - rho_j r_{j+1},  rho_j = c_{m+2j+2}/c_{m+2j+3}.
// One thread owns R north/south ring pairs (Pbar_lm(pi-theta) = (-1)^{l+m} Pbar_lm(theta)): per pair
// and per two l it issues 2 FMA of recurrence and 4 FMA of accumulation.  Underflow of
// Pbar_mm ~ sin^m(theta) is handled with a per-pair power-of-two exponent counter: while it is
// positive the pair is "dead" (true value < 2^-96, LIVE_BITS below) and contributes nothing.
//
// The CPU oracle (oracle/) uses the plain three-term recurrence in l and shares nothing with this file.
#include <math.h>
#include <stdio.h>

#include <algorithm>
#include <mutex>
#include <utility>
#include <vector>

#include "nusht_internal.cuh"

namespace {

constexpr int LEG_CHUNK = 8;       // n-steps between exponent checks
constexpr int LEG_R = 4;           // ring pairs per thread
// synthesis: one warp per CTA, so that warps with different live/dead histories never wait for each other
constexpr int SYN_THREADS = 32;
constexpr int SYN_WARPS = SYN_THREADS / 32;
constexpr int SYN_TN = 128;
// adjoint: one warp per CTA as well; more ring pairs per thread halve the cost of the cross-lane reduction
constexpr int ADJ_R = 5;           // adjoint: 5 pairs per thread amortise the cross-lane reduction (still 128 registers, 16 warps/SM)
constexpr int ADJ_TN = 128;
constexpr int ADJ_CHUNK = 8;       // n-steps per transposing reduction / exponent check
__host__ __device__ constexpr int adj_min_ctas(int r, int c) { return r <= 4 ? (c <= 2 ? 22 : (c <= 4 ? 18 : 16)) : (r == 5 ? 13 : (r == 6 ? 12 : (c <= 2 ? 12 : 10))); }
// A ring pair is "in range" once |Pbar_lm| >= 2^-LIVE_BITS; below that its terms are dropped.  The test runs once
// per chunk of 8 n-steps, over which Pbar grows by less than 2^32, so the largest dropped term is below
// 2^(32 - LIVE_BITS) = 2^-64 = 5e-20 relative to Pbar = O(1): no FP64 result can resolve it (LIVE_BITS = 64
// would drop terms up to 2^-32 and fails the stage test; 128 costs 0.07 ms per direction at lmax = 4095).  With
// the counter at 1 the stored value is the true one times 2^512, so the pair comes into range when it passes
// 2^(512 - LIVE_BITS).
constexpr int LIVE_BITS = 96;
constexpr double SCALE_UP_LIMIT = 1.6923032801030364e+125;   // 2^(512 - LIVE_BITS) = 2^416
constexpr double SCALE_DOWN = 7.458340731200207e-155;      // 2^-512

struct LegParams {
    // b_split: blocks bx >= b_split use the cos^2 form of t_n (header), and so do the remainder pairs iff
    // nblk >= b_split.  (The struct must not grow: k_legendre_adjoint sits exactly at its 128-register budget and
    // ptxas starts spilling inside its FMA loop when the parameter block gets larger; the cos^2 table is therefore
    // reached as ab + eoff[mmax + 1], the second half of one allocation.)
    int lmax, mmax, nr, nth2, npairs, b_split;
    int nblk, rem;   // main blocks of 32 R pairs per m; left-over pairs handled by the remainder blocks
    // fast-forward table (plan time): for warp (m, block) the first n-step (multiple of LEG_CHUNK) at which
    // one of its ring pairs is in range, and the scaled recurrence state of its pairs at that step
    const int* ff_n;
    const double2* ff_p;   // (p0, p1) per (m, block, r, lane)
    const int* ff_e;       // exponent counter
    // work list of the synthesis (plan time): CTA i takes items[i] = (block of ring pairs, m), longest first
    const int2* items;
    const int64_t* eoff;
    const double2* ab;
    const double* x2;      // sin^2(theta_j) per ring pair (the operand of the x^2-stepping recurrence, header)
    const double* x;
    const double2* logsin;
    const double2* logkap;
    // ring-list mode (rSHT on caller ring grids, ring.cu): pair j = (north ring pn[j], south ring ps[j] or -1);
    // rows of F[m][.] then have nth2 = nrings entries and are NOT doubled
    const int* pn;
    const int* ps;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra.uni WAIT_DONE;\n"
        "bra.uni WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// TMA 1-D bulk copy global -> shared, completion signalled on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ---------------------------------------------------------------------------------------------
// plan-time tables, one thread per m (sequential in n: sigma is a two-step product)
// ---------------------------------------------------------------------------------------------
__global__ void k_legendre_tables(int L, int M, const int64_t* __restrict__ eoff, double2* __restrict__ ab,
                                  double2* __restrict__ abx, double* __restrict__ sig, double* __restrict__ sodd, double* __restrict__ rho) {
    int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m > M) return;
    const int ne = (L - m) / 2 + 1;
    const int64_t o = eoff[m];
    auto c2 = [m](int l) -> double {   // c_l^2, exact integer numerator/denominator
        double num = (double)((long long)(l - m) * (long long)(l + m));
        double den = 4.0 * (double)l * (double)l - 1.0;
        return num / den;
    };
    double sg_prev = 0.0, sg = 1.0;
    for (int n = 0; n < ne; ++n) {
        const int l = m + 2 * n;
        const double c2l = (n == 0) ? 0.0 : c2(l);
        const double c2lm1 = (n == 0) ? 0.0 : c2(l - 1);
        const double c2l1 = c2(l + 1), c2l2 = c2(l + 2), c2l3 = c2(l + 3);
        const double A = 1.0 / sqrt(c2l1 * c2l2);
        const double D = c2l1 + c2l;
        const double C = sqrt(c2l * c2lm1) * A;
        const double sg_next = (n == 0) ? 1.0 : -C * sg_prev;
        const double alpha = A * sg / sg_next;
        ab[o + n] = make_double2(-alpha, alpha * (1.0 - D));   // t_n = ab.y + ab.x sin^2(theta) = alpha (x^2 - D)
        abx[o + n] = make_double2(alpha, -alpha * D);          // t_n = abx.y + abx.x cos^2(theta)
        sig[o + n] = sg;
        sodd[o + n] = sg / sqrt(c2l1);
        rho[o + n] = sqrt(c2l2 / c2l3);
        sg_prev = sg;
        sg = sg_next;
    }
}

// ---------------------------------------------------------------------------------------------
// a1 prologue: alm -> (ae, ao): even-class scaling and odd-class fold, one WARP per m.
//   ae_j = a_{m+2j} sigma_j;   r_j = a_{m+2j+1} - rho_j r_{j+1};   ao_j = r_j sodd_j
// The first-order recurrence in j is evaluated 32 entries at a time as a warp suffix scan of the
// affine maps r -> b_j - rho_j r (|rho_j| < 1, so the composition is as stable as the sequential
// form), carrying r across tiles from high j to low j.  All loads and stores are coalesced.
// ---------------------------------------------------------------------------------------------
constexpr int PREP_THREADS = 128;

// (Lio: band limit of the caller's alm layout; Lio < L only in ring plans built one degree higher, where the
//  coefficients above Lio read as zero)
template <typename T>
__global__ void __launch_bounds__(PREP_THREADS)
k_alm_prep(int L, int Lio, int M, const int64_t* __restrict__ eoff, const T* __restrict__ alm,
           const double* __restrict__ sig, const double* __restrict__ sodd,
           const double* __restrict__ rho, double4* __restrict__ aeo) {
    const int m = blockIdx.x * (PREP_THREADS / 32) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (m > M) return;
    const int ne = (L - m) / 2 + 1;
    const int no = (L - m + 1) / 2;
    const int64_t o = eoff[m];
    const T* col = alm + 2 * ((int64_t)m * (2 * Lio + 1 - m) / 2);   // col[2*l], col[2*l+1] for l >= m
    double cre = 0.0, cim = 0.0;   // r_{j+1} entering the tile from above
    for (int base = ((ne - 1) / 32) * 32; base >= 0; base -= 32) {
        const int j = base + lane;
        const bool in = j < ne;
        double are = 0.0, aim = 0.0, bre = 0.0, bim = 0.0, S = 0.0, sg = 0.0, so = 0.0;
        if (in) {
            const int le = m + 2 * j;
            if (le <= Lio) {
                are = (double)col[2 * le];
                aim = (double)col[2 * le + 1];
            }
            if (j < no && le + 1 <= Lio) {
                bre = (double)col[2 * le + 2];
                bim = (double)col[2 * le + 3];
            }
            S = -rho[o + j];
            sg = sig[o + j];
            so = sodd[o + j];
        }
        // suffix scan: after it, r_j = B + S * (r entering the tile)
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const double S2 = __shfl_down_sync(0xffffffffu, S, d);
            const double B2re = __shfl_down_sync(0xffffffffu, bre, d);
            const double B2im = __shfl_down_sync(0xffffffffu, bim, d);
            if (lane + d < 32) {
                bre = fma(S, B2re, bre);
                bim = fma(S, B2im, bim);
                S *= S2;
            }
        }
        const double rre = fma(S, cre, bre), rim = fma(S, cim, bim);
        if (in) {
            double4 v;
            v.x = are * sg;
            v.y = aim * sg;
            v.z = rre * so;
            v.w = rim * so;
            if (m == 0) { v.y = 0.0; v.w = 0.0; }   // Im(a_l0) is ignored (G3)
            aeo[o + j] = v;
        }
        cre = __shfl_sync(0xffffffffu, rre, 0);
        cim = __shfl_sync(0xffffffffu, rim, 0);
    }
}

// a11 epilogue: (e~, o~) -> alm.  c_{m+2n} = sigma_n e~_n;  u_n = sodd_n o~_n;
//   v_n = u_n - rho_{n-1} v_{n-1};  c_{m+2n+1} = v_n   (transpose of the fold above), one warp
// per m, prefix scan of the affine maps v -> u_n - rho_{n-1} v.
template <typename T>
__global__ void __launch_bounds__(PREP_THREADS)
k_alm_post(int L, int Lio, int M, const int64_t* __restrict__ eoff, const double4* __restrict__ eo,
           const double* __restrict__ sig, const double* __restrict__ sodd,
           const double* __restrict__ rho, T* __restrict__ alm) {
    const int m = blockIdx.x * (PREP_THREADS / 32) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (m > M) return;
    const int ne = (L - m) / 2 + 1;
    const int no = (L - m + 1) / 2;
    const int64_t o = eoff[m];
    T* col = alm + 2 * ((int64_t)m * (2 * Lio + 1 - m) / 2);
    double cre = 0.0, cim = 0.0;   // v_{n-1} entering the tile from below
    for (int base = 0; base < ne; base += 32) {
        const int n = base + lane;
        const bool in = n < ne;
        double ere = 0.0, eim = 0.0, ure = 0.0, uim = 0.0, S = 0.0;
        if (in) {
            const double4 v = eo[o + n];
            const double sg = sig[o + n], so = sodd[o + n];
            ere = v.x * sg;
            eim = v.y * sg;
            ure = v.z * so;
            uim = v.w * so;
            S = (n > 0) ? -rho[o + n - 1] : 0.0;
        }
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const double S2 = __shfl_up_sync(0xffffffffu, S, d);
            const double U2re = __shfl_up_sync(0xffffffffu, ure, d);
            const double U2im = __shfl_up_sync(0xffffffffu, uim, d);
            if (lane >= d) {
                ure = fma(S, U2re, ure);
                uim = fma(S, U2im, uim);
                S *= S2;
            }
        }
        const double vre = fma(S, cre, ure), vim = fma(S, cim, uim);
        if (in) {
            const int le = m + 2 * n;
            if (le <= Lio) {
                col[2 * le] = (T)ere;
                col[2 * le + 1] = (m == 0) ? (T)0 : (T)eim;
            }
            if (n < no && le + 1 <= Lio) {
                col[2 * le + 2] = (T)vre;
                col[2 * le + 3] = (m == 0) ? (T)0 : (T)vim;
            }
        }
        cre = __shfl_sync(0xffffffffu, vre, 31);
        cim = __shfl_sync(0xffffffffu, vim, 31);
    }
}

// ---------------------------------------------------------------------------------------------
// per-pair seed: qh_0 = Pbar_mm(theta_j) = (-1)^m 2^(lk_m + m log2 sin theta_j), as p * 2^(-512 e)
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void seed_pair(const LegParams& P, int m, int j, bool valid, double& p, int& e) {
    p = 0.0;
    e = 0;
    if (!valid) return;
    const double2 lk = P.logkap[m];
    if (m == 0) {
        p = exp2(lk.x + lk.y);
        return;
    }
    const double2 ls = P.logsin[j];
    if (ls.x < -1e300) return;   // a pole ring (log2 sin theta = -inf in the table): Pbar_lm = 0 for m > 0
    const double dm = (double)m;
    // (mh + err) = m * ls.x exactly;  s = mh + lk.x with two-sum error err2
    const double mh = dm * ls.x;
    const double err = fma(dm, ls.x, -mh);
    const double s = mh + lk.x;
    const double bb = s - mh;
    const double err2 = (mh - (s - bb)) + (lk.x - bb);
    const double low = err + err2 + fma(dm, ls.y, lk.y);
    int ee = 0;
    if (s < -(double)LIVE_BITS) ee = (int)floor((-s - (double)LIVE_BITS) * (1.0 / 512.0)) + 1;
    const double expo = s + 512.0 * (double)ee;      // exact: s has < 2^16 magnitude
    const double ip = rint(expo);
    const double fr = (expo - ip) + low;
    p = scalbn(exp2(fr), (int)ip);
    if (m & 1) p = -p;
    e = ee;
}

// a2 for one ring pair: north = E + x O, south = E - x O; mirror rows carry (-1)^m (phi -> phi + pi)
// (Fig. 1)
template <bool RING>
__device__ __forceinline__ void write_pair(const LegParams& P, double2* row, double sgn, int j, double ere,
                                           double eim, double ore_, double oim) {
    const double x = P.x[j];
    const double2 nv = make_double2(fma(x, ore_, ere), fma(x, oim, eim));
    const double2 sv = make_double2(fma(-x, ore_, ere), fma(-x, oim, eim));
    if (RING) {                    // ring list: F[m][ring], no doubling
        row[P.pn[j]] = nv;
        const int rs = P.ps[j];
        if (rs >= 0) row[rs] = sv;
        return;
    }
    const int ks = P.nr - 1 - j;   // south ring index
    row[j] = nv;
    if (j != 0) row[P.nth2 - j] = make_double2(sgn * nv.x, sgn * nv.y);
    if (ks != j) {
        row[ks] = sv;
        if (j != 0) row[P.nth2 - ks] = make_double2(sgn * sv.x, sgn * sv.y);
    }
}

// a10 for one ring pair (D^T): G[k] = Gt[k] + (-1)^m Gt[Ntheta-k] away from the poles, then the even /
// odd (in l - m) combinations of the north and south ring
template <bool RING>
__device__ __forceinline__ void fold_pair(const LegParams& P, const double2* __restrict__ row, double sgn, int j,
                                          double& ere, double& eim, double& ore_, double& oim) {
    if (RING) {                    // ring list: G[m][ring] as it is (weights applied upstream)
        const double2 gn = row[P.pn[j]];
        const int rs = P.ps[j];
        const double2 gs = rs >= 0 ? row[rs] : make_double2(0.0, 0.0);
        const double x = P.x[j];
        ere = gn.x + gs.x;
        eim = gn.y + gs.y;
        ore_ = x * (gn.x - gs.x);
        oim = x * (gn.y - gs.y);
        return;
    }
    const int kn = j, ks = P.nr - 1 - j;
    double2 gn = row[kn];
    if (kn != 0) {
        const double2 t = row[P.nth2 - kn];
        gn.x = fma(sgn, t.x, gn.x);
        gn.y = fma(sgn, t.y, gn.y);
    }
    double2 gs = make_double2(0.0, 0.0);
    if (ks != kn) {
        gs = row[ks];
        if (kn != 0) {
            const double2 t = row[P.nth2 - ks];
            gs.x = fma(sgn, t.x, gs.x);
            gs.y = fma(sgn, t.y, gs.y);
        }
    }
    const double x = P.x[j];
    ere = gn.x + gs.x;
    eim = gn.y + gs.y;
    ore_ = x * (gn.x - gs.x);
    oim = x * (gn.y - gs.y);
}

// Remainder ring pairs.  With N_r = 2^k + 1 rings there are 2^(k-1) + 1 pairs: one more than a whole
// number of 32 R blocks.  Rather than a 17th warp per m with a single busy lane, the last block
// column of the grid takes the `rem` left-over pairs of 32/rem different m per warp, one (m, pair)
// per lane, each lane streaming its own coefficient column from global memory.
template <bool RING>
__device__ void synth_remainder(const LegParams& P, const double4* __restrict__ aeo, double2* __restrict__ ft, int j0,
                                int rem, int by) {
    const int gid = by * 32 + threadIdx.x;
    const int m = gid / rem, j = j0 + gid % rem;
    if (m > P.mmax) return;
    const int ne = (P.lmax - m) / 2 + 1;
    const int64_t o = P.eoff[m];
    double p0 = 0.0, p1;
    int ex;
    seed_pair(P, m, j, true, p1, ex);
    const double x2 = P.x2[j];
    double ere = 0.0, eim = 0.0, ore_ = 0.0, oim = 0.0;
    for (int n = 0; n < ne; ++n) {
        const double2 ab = P.ab[o + n + (P.nblk >= P.b_split ? P.eoff[P.mmax + 1] : 0)];
        const double t = fma(ab.x, x2, ab.y);
        if (ex == 0) {
            const double4 c = aeo[o + n];
            ere = fma(c.x, p1, ere);
            eim = fma(c.y, p1, eim);
            ore_ = fma(c.z, p1, ore_);
            oim = fma(c.w, p1, oim);
        }
        const double pn = fma(t, p1, p0);
        p0 = p1;
        p1 = pn;
        if (ex > 0 && (n & 7) == 7 && fabs(p1) > SCALE_UP_LIMIT) {
            p1 *= SCALE_DOWN;
            p0 *= SCALE_DOWN;
            ex -= 1;
        }
    }
    write_pair<RING>(P, ft + (int64_t)m * P.nth2, (m & 1) ? -1.0 : 1.0, j, ere, eim, ore_, oim);
}

template <bool RING>
__device__ void adjoint_remainder(const LegParams& P, const double2* __restrict__ gt, double4* __restrict__ eo, int j0,
                                  int rem, int by) {
    const int gid = by * 32 + threadIdx.x;
    const int m = gid / rem, j = j0 + gid % rem;
    if (m > P.mmax) return;
    const int ne = (P.lmax - m) / 2 + 1;
    const int64_t o = P.eoff[m];
    double p0 = 0.0, p1;
    int ex;
    seed_pair(P, m, j, true, p1, ex);
    const double x2 = P.x2[j];
    double ere, eim, ore_, oim;
    fold_pair<RING>(P, gt + (int64_t)m * P.nth2, (m & 1) ? -1.0 : 1.0, j, ere, eim, ore_, oim);
    for (int n = 0; n < ne; ++n) {
        const double2 ab = P.ab[o + n];          // the launch hands over the table of this block's form
        const double t = fma(ab.x, x2, ab.y);
        if (ex == 0) {
            double* out = reinterpret_cast<double*>(eo + o + n);
            atomicAdd(out + 0, p1 * ere);
            atomicAdd(out + 1, p1 * eim);
            atomicAdd(out + 2, p1 * ore_);
            atomicAdd(out + 3, p1 * oim);
        }
        const double pn = fma(t, p1, p0);
        p0 = p1;
        p1 = pn;
        if (ex > 0 && (n & 3) == 3 && fabs(p1) > SCALE_UP_LIMIT) {
            p1 *= SCALE_DOWN;
            p0 *= SCALE_DOWN;
            ex -= 1;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// plan time: fast-forward table.  While every ring pair of a warp is still below range (Pbar_mm ~
// sin^m theta underflows for most (m, ring)), the transform kernels would only advance the
// recurrence.  That part does not depend on the data, so it is run once here: the warp advances
// chunk by chunk exactly as the transform kernels do, stops at the first chunk boundary where a
// pair is in range, and stores the step and the state.  The transforms start from there; a warp
// whose pairs never come into range before lmax does no work at all.
// ---------------------------------------------------------------------------------------------
template <int R>
__global__ void __launch_bounds__(32)
k_legendre_fastforward(LegParams P, int* __restrict__ ff_n, double2* __restrict__ ff_p, int* __restrict__ ff_e) {
    const int m = blockIdx.y, lane = threadIdx.x;
    const int ne = (P.lmax - m) / 2 + 1;
    const int64_t o = P.eoff[m];
    const int jb = blockIdx.x * (32 * R);
    const bool xform = (int)blockIdx.x >= P.b_split;
    double x2[R], p0[R], p1[R];
    int ex[R];
    bool valid[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int j = jb + r * 32 + lane;
        valid[r] = j < P.npairs;
        x2[r] = valid[r] ? P.x2[j] : 0.0;
        seed_pair(P, m, j, valid[r], p1[r], ex[r]);
        p0[r] = 0.0;
    }
    int n = 0;
    for (; n < ne; n += LEG_CHUNK) {
        bool any_live = false;
#pragma unroll
        for (int r = 0; r < R; ++r) any_live |= (valid[r] && ex[r] == 0);
        if (__any_sync(0xffffffffu, any_live)) break;
        const int ns = min(LEG_CHUNK, ne - n);
        for (int i = 0; i < ns; ++i) {
            const double2 ab = P.ab[o + n + i + (xform ? P.eoff[P.mmax + 1] : 0)];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const double t = fma(ab.x, x2[r], ab.y);
                const double pn = fma(t, p1[r], p0[r]);
                p0[r] = p1[r];
                p1[r] = pn;
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (ex[r] > 0 && fabs(p1[r]) > SCALE_UP_LIMIT) {
                p1[r] *= SCALE_DOWN;
                p0[r] *= SCALE_DOWN;
                ex[r] -= 1;
            }
        }
    }
    const int64_t w = (int64_t)m * P.nblk + blockIdx.x;
    if (lane == 0) ff_n[w] = min(n, ne);
#pragma unroll
    for (int r = 0; r < R; ++r) {
        ff_p[(w * R + r) * 32 + lane] = make_double2(p0[r], p1[r]);
        ff_e[(w * R + r) * 32 + lane] = ex[r];
    }
}

// ---------------------------------------------------------------------------------------------
// a1 + a2: Legendre synthesis with fused DFS doubling.  grid = (pair blocks, m).
// ---------------------------------------------------------------------------------------------
template <int R, bool RING>
__global__ void __launch_bounds__(SYN_THREADS)
k_legendre_synth(LegParams P, const double4* __restrict__ aeo, double2* __restrict__ ft) {
    const int2 item = P.items[blockIdx.x];
    const int bx = item.x, by = item.y;
    if (P.rem > 0 && bx == P.nblk) {
        synth_remainder<RING>(P, aeo, ft, P.nblk * (32 * R), P.rem, by);
        return;
    }
    __shared__ __align__(16) double2 s_ab[2][SYN_TN];
    __shared__ __align__(32) double4 s_aeo[2][SYN_TN];
    __shared__ __align__(8) uint64_t s_bar[2];

    const int m = by;
    const int L = P.lmax;
    const int ne = (L - m) / 2 + 1;
    const int64_t o = P.eoff[m];
    const bool xform = bx >= P.b_split;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int jb = (bx * SYN_WARPS + warp) * (32 * R);
    const int ntiles = (ne + SYN_TN - 1) / SYN_TN;
    const int64_t wff = (int64_t)m * P.nblk + bx;
    const int n_start = P.ff_n[wff];          // first step at which a pair of this warp is in range
    const int tile0 = n_start / SYN_TN;

    if (tid == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        mbar_fence_init();
    }
    __syncthreads();
    auto issue = [&](int tile) {
        const int st = (tile - tile0) & 1;
        const int cnt = min(SYN_TN, ne - tile * SYN_TN);
        mbar_expect_tx(&s_bar[st], (uint32_t)cnt * 48u);
        // blocks next to the equator take the cos^2 form of the table (header)
        bulk_g2s(&s_ab[st][0], P.ab + (xform ? P.eoff[P.mmax + 1] : 0) + o + (int64_t)tile * SYN_TN, (uint32_t)cnt * 16u, &s_bar[st]);
        bulk_g2s(&s_aeo[st][0], aeo + o + (int64_t)tile * SYN_TN, (uint32_t)cnt * 32u, &s_bar[st]);
    };
    if (tid == 0 && n_start < ne) {
        issue(tile0);
        if (tile0 + 1 < ntiles) issue(tile0 + 1);
    }

    double x2[R], p0[R], p1[R], ere[R], eim[R], ore_[R], oim[R];
    int ex[R];
    bool valid[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int j = jb + r * 32 + lane;
        valid[r] = j < P.npairs;
        x2[r] = valid[r] ? P.x2[j] : 0.0;
        const double2 pp = P.ff_p[(wff * R + r) * 32 + lane];   // state at n_start (plan-time fast-forward)
        p0[r] = pp.x;
        p1[r] = pp.y;
        ex[r] = P.ff_e[(wff * R + r) * 32 + lane];
        ere[r] = eim[r] = ore_[r] = oim[r] = 0.0;
    }
    const bool warp_has_work = jb < P.npairs;
    bool steady = false;                      // every pair of the warp in range: no more exponent bookkeeping

    for (int tile = tile0; tile < ntiles && n_start < ne; ++tile) {
        const int st = (tile - tile0) & 1;
        const int cnt = min(SYN_TN, ne - tile * SYN_TN);
        mbar_wait(&s_bar[st], (uint32_t)(((tile - tile0) >> 1) & 1));
        if (warp_has_work) {
            for (int i0 = (tile == tile0) ? n_start - tile0 * SYN_TN : 0; i0 < cnt; i0 += LEG_CHUNK) {
                const int ns = min(LEG_CHUNK, cnt - i0);
                bool w_dead = false, w_live = true;
                if (!steady) {                   // warp-uniform; exponents only ever count down to 0
                    bool any_dead = false, any_live = false;
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        any_dead |= (ex[r] > 0);
                        any_live |= (valid[r] && ex[r] == 0);
                    }
                    w_dead = __any_sync(0xffffffffu, any_dead);
                    w_live = __any_sync(0xffffffffu, any_live);
                    steady = !w_dead;
                }
                if (w_live) {
                    // some pair in range: 6 FMA per pair and step, no masks.  A pair still below range
                    // accumulates finite garbage (scaled |p1| stays below 2^448); its sums are cleared when it
                    // comes into range (below) or at the end, which drops exactly the terms < 2^-LIVE_BITS.
                    if (ns == LEG_CHUNK) {
#pragma unroll
                        for (int i = 0; i < LEG_CHUNK; ++i) {
                            const double2 ab = s_ab[st][i0 + i];
                            const double4 c = s_aeo[st][i0 + i];
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                const double t = fma(ab.x, x2[r], ab.y);
                                ere[r] = fma(c.x, p1[r], ere[r]);
                                eim[r] = fma(c.y, p1[r], eim[r]);
                                ore_[r] = fma(c.z, p1[r], ore_[r]);
                                oim[r] = fma(c.w, p1[r], oim[r]);
                                const double pn = fma(t, p1[r], p0[r]);
                                p0[r] = p1[r];
                                p1[r] = pn;
                            }
                        }
                    } else {
                        for (int i = 0; i < ns; ++i) {
                            const double2 ab = s_ab[st][i0 + i];
                            const double4 c = s_aeo[st][i0 + i];
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                const double t = fma(ab.x, x2[r], ab.y);
                                ere[r] = fma(c.x, p1[r], ere[r]);
                                eim[r] = fma(c.y, p1[r], eim[r]);
                                ore_[r] = fma(c.z, p1[r], ore_[r]);
                                oim[r] = fma(c.w, p1[r], oim[r]);
                                const double pn = fma(t, p1[r], p0[r]);
                                p0[r] = p1[r];
                                p1[r] = pn;
                            }
                        }
                    }
                } else {
                    // every pair of the warp still below range: recurrence only (2 FMA)
                    for (int i = 0; i < ns; ++i) {
                        const double2 ab = s_ab[st][i0 + i];
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const double t = fma(ab.x, x2[r], ab.y);
                            const double pn = fma(t, p1[r], p0[r]);
                            p0[r] = p1[r];
                            p1[r] = pn;
                        }
                    }
                }
                if (w_dead) {
                    // exponent bookkeeping once per chunk: growth over 8 steps is < 2^32
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        if (ex[r] > 0) {
                            if (fabs(p1[r]) > SCALE_UP_LIMIT) {
                                p1[r] *= SCALE_DOWN;
                                p0[r] *= SCALE_DOWN;
                                ex[r] -= 1;
                            }
                            ere[r] = eim[r] = ore_[r] = oim[r] = 0.0;   // nothing counted before the pair is in range
                        }
                    }
                }
            }
        }
        __syncthreads();
        if (tid == 0 && tile + 2 < ntiles) issue(tile + 2);
    }

    if (!warp_has_work) return;
#pragma unroll
    for (int r = 0; r < R; ++r)
        if (ex[r] > 0) ere[r] = eim[r] = ore_[r] = oim[r] = 0.0;   // never came into range
    // a2: fused DFS doubling
    const double sgn = (m & 1) ? -1.0 : 1.0;
    double2* row = ft + (int64_t)m * P.nth2;
#pragma unroll
    for (int r = 0; r < R; ++r)
        if (valid[r]) write_pair<RING>(P, row, sgn, jb + r * 32 + lane, ere[r], eim[r], ore_[r], oim[r]);
}

// ---------------------------------------------------------------------------------------------
// a10 + a11: fold + adjoint Legendre.  One CTA per m, looping over blocks of ring pairs; per
// n-step every thread forms 4 partial sums over its R pairs, 8 steps x 4 sums are reduced across
// the warp with a 31-shuffle transposing butterfly, across warps through shared memory, and
// accumulated into eo[m][n] by the CTA itself (deterministic, no atomics).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double shfl_xor_d(double v, int mask) {
    return __shfl_xor_sync(0xffffffffu, v, mask);
}

// One warp per CTA: the warp owns 32 R ring pairs of one m for all n, forms the 4 partial sums of
// every n-step over its rings (4 steps x 4 sums at a time, transposed through shared memory) and
// adds them to eo[m][n] with native FP64 global reductions (RED.ADD.F64); eo must be zero on entry.
// No warp ever waits for another one, whatever its mix of live and dead ring pairs.  A dead pair
// (scaled value below range) keeps G = 0 in registers, so the inner loop needs no masks; its folded
// G values are loaded when the pair comes into range.
template <int R, int C, bool RING>
__global__ void __launch_bounds__(32, adj_min_ctas(R, C))
k_legendre_adjoint(LegParams P, const double2* __restrict__ gt, double4* __restrict__ eo) {
    // plain 2-D grid (block of ring pairs, m): the blocks of one m run together and add into the same eo[m]
    // column while it is L2-resident; a work list as in the synthesis was tried (see build_work_list).
    // The host launches this kernel once per form of t_n (header): blocks [0, b_split) with the sin^2 table, blocks
    // from b_split on with P.ab pointing at the cos^2 table and P.b_split = the block offset.  (Choosing the table in
    // here instead costs the registers that make ptxas spill inside the FMA loop: the kernel sits exactly at the
    // 128 registers that four one-warp CTAs per scheduler leave.)
    const int bx = blockIdx.x + P.b_split, by = blockIdx.y;
    if (P.rem > 0 && bx == P.nblk) {
        adjoint_remainder<RING>(P, gt, eo, P.nblk * (32 * R), P.rem, by);
        return;
    }
    __shared__ __align__(16) double2 s_ab[2][ADJ_TN];
    constexpr int NV = 4 * C;             // values reduced across the warp per chunk of C steps
    __shared__ __align__(16) double s_tr[NV][34];   // row stride 272 B: 16-byte aligned rows, conflict-free LDS.128
    __shared__ __align__(8) uint64_t s_bar[2];

    const int m = by;
    const int L = P.lmax;
    const int ne = (L - m) / 2 + 1;
    const int64_t o = P.eoff[m];
    const int lane = threadIdx.x;
    const int jb = bx * (32 * R);
    const int ntiles = (ne + ADJ_TN - 1) / ADJ_TN;
    const double sgn = (m & 1) ? -1.0 : 1.0;
    const double2* row = gt + (int64_t)m * P.nth2;
    const int64_t wff = (int64_t)m * P.nblk + bx;
    const int n_start = P.ff_n[wff];          // first step at which a pair of this warp is in range
    if (n_start >= ne) return;                // never before lmax: this warp contributes nothing
    const int tile0 = n_start / ADJ_TN;

    // entries past the end of a column are read (and their results dropped): keep them finite
    for (int i = lane; i < 2 * ADJ_TN; i += 32) (&s_ab[0][0])[i] = make_double2(0.0, 0.0);
    if (lane == 0) {
        mbar_init(&s_bar[0], 1);
        mbar_init(&s_bar[1], 1);
        mbar_fence_init();
    }
    __syncwarp();
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy zero fill before the bulk copies
    auto issue = [&](int tile) {
        const int st = (tile - tile0) & 1;
        const int cnt = min(ADJ_TN, ne - tile * ADJ_TN);
        mbar_expect_tx(&s_bar[st], (uint32_t)cnt * 16u);
        bulk_g2s(&s_ab[st][0], P.ab + o + (int64_t)tile * ADJ_TN, (uint32_t)cnt * 16u, &s_bar[st]);
    };
    if (lane == 0) {
        issue(tile0);
        if (tile0 + 1 < ntiles) issue(tile0 + 1);
    }

    double x2[R], p0[R], p1[R], gere[R], geim[R], gore[R], goim[R];
    int ex[R];
    bool valid[R];
    auto load_g = [&](int j, double& ere, double& eim, double& ore_, double& oim) {
        fold_pair<RING>(P, row, sgn, j, ere, eim, ore_, oim);
    };
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int j = jb + r * 32 + lane;
        valid[r] = j < P.npairs;
        x2[r] = valid[r] ? P.x2[j] : 0.0;
        const double2 pp = P.ff_p[(wff * R + r) * 32 + lane];   // state at n_start (plan-time fast-forward)
        p0[r] = pp.x;
        p1[r] = pp.y;
        ex[r] = P.ff_e[(wff * R + r) * 32 + lane];
        gere[r] = geim[r] = gore[r] = goim[r] = 0.0;
        if (valid[r] && ex[r] == 0) load_g(j, gere[r], geim[r], gore[r], goim[r]);
    }

    bool steady = false;                      // every pair of the warp in range: no more exponent bookkeeping
    for (int tile = tile0; tile < ntiles; ++tile) {
        const int st = (tile - tile0) & 1;
        const int cnt = min(ADJ_TN, ne - tile * ADJ_TN);
        mbar_wait(&s_bar[st], (uint32_t)(((tile - tile0) >> 1) & 1));
        for (int i0 = (tile == tile0) ? n_start - tile0 * ADJ_TN : 0; i0 < cnt; i0 += C) {
            const int ns = min(C, cnt - i0);
            bool w_dead = false, w_live = true;
            if (!steady) {                       // warp-uniform; exponents only ever count down to 0
                bool any_dead = false, any_live = false;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    any_dead |= (ex[r] > 0);
                    any_live |= (valid[r] && ex[r] == 0);
                }
                w_dead = __any_sync(0xffffffffu, any_dead);
                w_live = __any_sync(0xffffffffu, any_live);
                steady = !w_dead && w_live;
            }
            if (w_live) {
                // always ADJ_CHUNK steps: beyond the end of the column the sums are dropped below and
                // the recurrence state is never used again
                double v[NV];
#pragma unroll
                for (int q = 0; q < NV; ++q) v[q] = 0.0;
#pragma unroll
                for (int i = 0; i < C; ++i) {
                    const double2 ab = s_ab[st][i0 + i];   // beyond cnt: stale or zero entries, results dropped
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const double t = fma(ab.x, x2[r], ab.y);
                        v[4 * i + 0] = fma(p1[r], gere[r], v[4 * i + 0]);
                        v[4 * i + 1] = fma(p1[r], geim[r], v[4 * i + 1]);
                        v[4 * i + 2] = fma(p1[r], gore[r], v[4 * i + 2]);
                        v[4 * i + 3] = fma(p1[r], goim[r], v[4 * i + 3]);
                        const double pn = fma(t, p1[r], p0[r]);
                        p0[r] = p1[r];
                        p1[r] = pn;
                    }
                }
                // cross-lane sums: transpose through shared memory (value q of lane l at s_tr[q][l]); the
                // 32 / NV lanes of row q = lane % NV add NV entries each and are combined by shuffles
                double tot;
                int qout;
                if (NV == 32) {
                    // values (2 qp, 2 qp + 1) of a lane travel as one 128-bit store; lane = (qp, half) then adds the pair
                    // over 16 lanes and the two halves meet in one shuffle
                    double2* tr2 = reinterpret_cast<double2*>(&s_tr[0][0]);        // [16][33] double2
#pragma unroll
                    for (int qp = 0; qp < NV / 2; ++qp) tr2[qp * 33 + lane] = make_double2(v[2 * qp], v[2 * qp + 1]);
                    __syncwarp();
                    const double2* src = tr2 + (lane & 15) * 33 + 16 * (lane >> 4);
                    double a0 = 0.0, a1 = 0.0, b0 = 0.0, b1 = 0.0;
#pragma unroll
                    for (int k = 0; k < 16; k += 2) {
                        const double2 u = src[k], w = src[k + 1];
                        a0 += u.x;
                        b0 += u.y;
                        a1 += w.x;
                        b1 += w.y;
                    }
                    double s0 = a0 + a1, s1 = b0 + b1;
                    s0 += shfl_xor_d(s0, 16);
                    s1 += shfl_xor_d(s1, 16);
                    tot = (lane < 16) ? s0 : s1;
                    qout = 2 * (lane & 15) + (lane >> 4);
                } else {
#pragma unroll
                    for (int q = 0; q < NV; ++q) s_tr[q][lane] = v[q];
                    __syncwarp();
                    const double2* src = reinterpret_cast<const double2*>(&s_tr[lane % NV][NV * (lane / NV)]);
                    double ta = 0.0, tb2 = 0.0, tc = 0.0, td = 0.0;      // four short add chains
#pragma unroll
                    for (int k = 0; k < NV / 2; k += 2) {
                        const double2 u = src[k], w = src[k + 1];
                        ta += u.x;
                        tb2 += u.y;
                        tc += w.x;
                        td += w.y;
                    }
                    tot = (ta + tb2) + (tc + td);
#pragma unroll
                    for (int sh = NV; sh < 32; sh *= 2) tot += shfl_xor_d(tot, sh);
                    qout = lane;
                }
                __syncwarp();
                if (qout < NV && (qout >> 2) < ns)      // q = 4 * step + component
                    atomicAdd(reinterpret_cast<double*>(eo + o + (int64_t)tile * ADJ_TN + i0) + qout, tot);
            } else {
                for (int i = 0; i < ns; ++i) {
                    const double2 ab = s_ab[st][i0 + i];
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const double t = fma(ab.x, x2[r], ab.y);
                        const double pn = fma(t, p1[r], p0[r]);
                        p0[r] = p1[r];
                        p1[r] = pn;
                    }
                }
            }
            if (w_dead) {
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    if (ex[r] > 0 && fabs(p1[r]) > SCALE_UP_LIMIT) {
                        p1[r] *= SCALE_DOWN;
                        p0[r] *= SCALE_DOWN;
                        ex[r] -= 1;
                        if (ex[r] == 0) load_g(jb + r * 32 + lane, gere[r], geim[r], gore[r], goim[r]);
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0 && tile + 2 < ntiles) issue(tile + 2);
    }
}

}  // namespace

// =============================================================================================
// host side
// =============================================================================================
// grid decomposition of the ring pairs for R pairs per thread (see synth_remainder)
static dim3 leg_grid(const nusht_plan_s* p, int R, LegParams& P) {
    const int per = 32 * R;
    int nblk = p->lg.npairs / per, rem = p->lg.npairs - nblk * per;
    if (rem == 0 || rem > 8 || nblk == 0) {
        nblk = (p->lg.npairs + per - 1) / per;
        rem = 0;
    }
    P.nblk = nblk;
    P.rem = rem;
    // form of t_n per block (header): pairs are ordered from the poles to the equator, so the blocks whose first pair
    // lies at theta >= pi/4 (index >= j_quarter) are the last ones
    P.b_split = (p->j_quarter + per - 1) / per;
    P.x2 = (R == ADJ_R && ADJ_R != LEG_R) ? p->d_x2a : p->d_x2;
    const int need_y = rem ? ((p->mmax + 1) * rem + 31) / 32 : 0;   // remainder warps; they fit: rem <= 8
    (void)need_y;
    return dim3(nblk + (rem ? 1 : 0), p->mmax + 1);
}

static LegParams make_params(const nusht_plan_s* p, bool adjoint_tables = false) {
    LegParams P;
    P.nblk = 0;
    P.rem = 0;
    P.lmax = p->lmax;
    P.mmax = p->mmax;
    P.nr = p->lg.nr;
    P.nth2 = p->lg.nth2;
    P.npairs = p->lg.npairs;
    P.b_split = 0;
    P.eoff = p->d_eoff;
    P.ab = p->d_ab;
    P.x2 = p->d_x2;
    P.x = p->d_x;
    P.logsin = p->d_logsin;
    P.logkap = p->d_logkap;
    P.pn = p->d_pair_n;
    P.ps = p->d_pair_s;
    const bool a = adjoint_tables && ADJ_R != LEG_R;
    P.ff_n = a ? p->d_ffa_n : p->d_ff_n;
    P.ff_p = a ? p->d_ffa_p : p->d_ff_p;
    P.ff_e = a ? p->d_ffa_e : p->d_ff_e;
    P.items = p->d_items_syn;
    return P;
}

template <typename T>
static int dev_alloc(T** ptr, size_t count, nusht_plan_s* p) {
    size_t bytes = count * sizeof(T);
    if (bytes == 0) bytes = sizeof(T);
    NUSHT_CUDA_TRY(cudaMalloc((void**)ptr, bytes));
    p->workspace_bytes += (int64_t)bytes;
    return NUSHT_OK;
}

// Work list of the synthesis kernel: one entry (block of ring pairs, m) per CTA.  A block's cost is the number of
// n-steps from its first in-range step to the end of the column, known from the fast-forward table.  The
// remainder CTAs (one lane per (m, pair), dependent global loads: long latency chains) come first, then the
// blocks by decreasing cost, so the grid drains evenly (3.07 -> 2.95 ms at lmax = 4095); blocks that never come
// into range go last and only write their zeros.  The adjoint kernel keeps its 2-D grid: it sits exactly at
// 128 registers and the list lookup made it spill (4.2 -> 4.9 ms), and its blocks of one m should run together
// anyway (they add into the same eo[m] column while it is L2-resident).
// FP64 FMAs one launch executes with R ring pairs per thread: every warp runs 6 FMA (2 recurrence + 4 accumulation)
// per lane, ring pair and n-step from its fast-forward step to the end of the column (pairs of a live warp that are
// still below range execute them too); the remainder pairs run whole columns.
static int64_t executed_fma(const nusht_plan_s* p, int R, const LegParams& P, const std::vector<int>& ffn) {
    const int M = p->mmax, L = p->lmax;
    int64_t steps = 0;
    for (int m = 0; m <= M; ++m) {
        const int ne = (L - m) / 2 + 1;
        for (int b = 0; b < P.nblk; ++b) steps += (int64_t)std::max(0, ne - ffn[(size_t)m * P.nblk + b]) * 32 * R;
        steps += (int64_t)ne * P.rem;
    }
    return 6 * steps;
}

static int build_work_list(nusht_plan_s* p, int R, const int* d_ff_n, int2** d_items, int* n_items) {
    LegParams P = make_params(p);
    leg_grid(p, R, P);
    const int M = p->mmax, L = p->lmax;
    std::vector<int> ffn((size_t)(M + 1) * P.nblk);
    NUSHT_CUDA_TRY(cudaMemcpy(ffn.data(), d_ff_n, sizeof(int) * ffn.size(), cudaMemcpyDeviceToHost));
    p->leg_fma_syn = executed_fma(p, R, P, ffn);
    if (ADJ_R != LEG_R) {
        LegParams Pa = make_params(p, true);
        leg_grid(p, ADJ_R, Pa);
        std::vector<int> ffa((size_t)(M + 1) * Pa.nblk);
        NUSHT_CUDA_TRY(cudaMemcpy(ffa.data(), p->d_ffa_n, sizeof(int) * ffa.size(), cudaMemcpyDeviceToHost));
        p->leg_fma_adj = executed_fma(p, ADJ_R, Pa, ffa);
    } else {
        p->leg_fma_adj = p->leg_fma_syn;
    }
    std::vector<int2> items;
    items.reserve(ffn.size() + (size_t)M + 1);
    if (P.rem > 0) {
        const int ny = ((M + 1) * P.rem + 31) / 32;
        for (int y = 0; y < ny; ++y) items.push_back(make_int2(P.nblk, y));
    }
    std::vector<std::pair<int, int64_t>> order;     // (cost, m * nblk + block)
    order.reserve(ffn.size());
    for (int m = 0; m <= M; ++m) {
        const int ne = (L - m) / 2 + 1;
        for (int b = 0; b < P.nblk; ++b) {
            const int cost = ne - ffn[(size_t)m * P.nblk + b];
            order.push_back(std::make_pair(cost > 0 ? cost : 0, (int64_t)m * P.nblk + b));
        }
    }
    std::stable_sort(order.begin(), order.end(),
                     [](const std::pair<int, int64_t>& a, const std::pair<int, int64_t>& b) { return a.first > b.first; });
    for (const auto& e : order) items.push_back(make_int2((int)(e.second % P.nblk), (int)(e.second / P.nblk)));
    *n_items = (int)items.size();
    NUSHT_TRY(dev_alloc(d_items, items.size(), p));
    if (!items.empty())
        NUSHT_CUDA_TRY(cudaMemcpy(*d_items, items.data(), sizeof(int2) * items.size(), cudaMemcpyHostToDevice));
    return NUSHT_OK;
}

int legendre_pair_rings(int nrings, const double* theta, int* pair_n, int* pair_s) {
    const double PI_D = 3.14159265358979323846;
    std::vector<int> order(nrings);
    for (int i = 0; i < nrings; ++i) order[i] = i;
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return theta[a] < theta[b]; });
    // two pointers from the poles inwards: the ring nearest to the north pole against the one nearest to the south
    std::vector<std::pair<double, std::pair<int, int>>> pairs;     // (distance from the nearer pole, (north, south))
    int lo = 0, hi = nrings - 1;
    while (lo <= hi) {
        const int a = order[lo], b = order[hi];
        const double dn = theta[a], ds = PI_D - theta[b];          // distances from the north / south pole
        if (lo < hi && fabs((theta[a] + theta[b]) - PI_D) <= 9.0e-16) {
            pairs.push_back({dn, {a, b}});
            ++lo;
            --hi;
        } else if (lo == hi || dn <= ds) {
            pairs.push_back({fmin(theta[a], PI_D - theta[a]), {a, -1}});
            ++lo;
        } else {
            pairs.push_back({fmin(theta[b], PI_D - theta[b]), {b, -1}});
            --hi;
        }
    }
    std::stable_sort(pairs.begin(), pairs.end(),
                     [](const std::pair<double, std::pair<int, int>>& u, const std::pair<double, std::pair<int, int>>& v) {
                         return u.first < v.first;
                     });
    for (size_t j = 0; j < pairs.size(); ++j) {
        pair_n[j] = pairs[j].second.first;
        pair_s[j] = pairs[j].second.second;
    }
    return (int)pairs.size();
}

int legendre_build_tables(nusht_plan_s* p) {
    const int L = p->lmax, M = p->mmax;
    std::vector<int> h_pn, h_ps;
    if (p->lg.ring_mode) {          // pairs of the caller's ring list (ring.cu set nr = nth2 = nrings)
        h_pn.resize(p->lg.nr);
        h_ps.resize(p->lg.nr);
        p->lg.npairs = legendre_pair_rings(p->lg.nr, p->h_ring_theta, h_pn.data(), h_ps.data());
        p->lg.has_equator = 0;
        NUSHT_TRY(dev_alloc(&p->d_pair_n, (size_t)p->lg.npairs, p));
        NUSHT_TRY(dev_alloc(&p->d_pair_s, (size_t)p->lg.npairs, p));
        NUSHT_CUDA_TRY(cudaMemcpy(p->d_pair_n, h_pn.data(), sizeof(int) * p->lg.npairs, cudaMemcpyHostToDevice));
        NUSHT_CUDA_TRY(cudaMemcpy(p->d_pair_s, h_ps.data(), sizeof(int) * p->lg.npairs, cudaMemcpyHostToDevice));
    }
    const LegendreGeom& g = p->lg;
    // column offsets
    std::vector<int64_t> eoff(M + 2);
    int64_t acc = 0;
    for (int m = 0; m <= M; ++m) {
        eoff[m] = acc;
        acc += (L - m) / 2 + 1;
    }
    eoff[M + 1] = acc;
    p->n_e_total = acc;
    NUSHT_TRY(dev_alloc(&p->d_eoff, (size_t)M + 2, p));
    NUSHT_CUDA_TRY(cudaMemcpy(p->d_eoff, eoff.data(), sizeof(int64_t) * (M + 2), cudaMemcpyHostToDevice));
    NUSHT_TRY(dev_alloc(&p->d_ab, 2 * (size_t)acc, p));     // sin^2 form, then the cos^2 form (header)
    NUSHT_TRY(dev_alloc(&p->d_sig, (size_t)acc, p));
    NUSHT_TRY(dev_alloc(&p->d_sodd, (size_t)acc, p));
    NUSHT_TRY(dev_alloc(&p->d_rho, (size_t)acc, p));
    NUSHT_TRY(dev_alloc(&p->d_aeo, (size_t)acc, p));
    NUSHT_TRY(dev_alloc(&p->d_ft, (size_t)(M + 1) * (size_t)g.nth2, p));
    {
        const int threads = 32;
        k_legendre_tables<<<(M + 1 + threads - 1) / threads, threads>>>(L, M, p->d_eoff, p->d_ab, p->d_ab + acc, p->d_sig,
                                                                         p->d_sodd, p->d_rho);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    // ring tables in extended precision on the host: theta_j = pi j/(nr-1)
    const long double PI_L = 3.14159265358979323846264338327950288L;
    std::vector<double> x2(g.npairs), x2c(g.npairs), x(g.npairs);    // sin^2, cos^2, cos of the pair's colatitude
    std::vector<double2> ls(g.npairs);
    p->j_quarter = g.npairs;
    for (int j = 0; j < g.npairs; ++j) {
        long double th = PI_L * (long double)j / (long double)(g.nr - 1);
        if (g.ring_mode) {
            // the pair's colatitude: the north ring's, averaged with the mirror of its partner (they agree to 2 ulp)
            th = (long double)p->h_ring_theta[h_pn[j]];
            if (h_ps[j] >= 0) th = 0.5L * (th + (PI_L - (long double)p->h_ring_theta[h_ps[j]]));
        }
        long double c = cosl(th), s = sinl(th);
        if (g.has_equator && j == g.npairs - 1) c = 0.0L;
        x[j] = (double)c;
        x2[j] = (double)(s * s);          // the kernels' "x2" operand is sin^2(theta) or cos^2(theta): see the header
        x2c[j] = (double)(c * c);
        if (g.has_equator && j == g.npairs - 1) { x2[j] = 1.0; x2c[j] = 0.0; }
        if (fminl(th, PI_L - th) >= 0.25L * PI_L && j < p->j_quarter) p->j_quarter = j;   // pairs run pole -> equator
        if (!(s > 0.0L)) {
            ls[j] = make_double2(-INFINITY, 0.0);   // a pole ring: seed_pair returns Pbar_lm = 0 for m > 0
            x2[j] = 0.0;
            x2c[j] = 1.0;
            x[j] = (c < 0.0L) ? -1.0 : 1.0;
        } else {
            long double v = log2l(s);
            double hi = (double)v;
            ls[j] = make_double2(hi, (double)(v - (long double)hi));
        }
    }
    std::vector<double2> lk(M + 1);
    {
        long double v = -0.5L * log2l(4.0L * PI_L);
        for (int m = 0; m <= M; ++m) {
            if (m > 0) v += 0.5L * log2l((long double)(2 * m + 1) / (long double)(2 * m));
            double hi = (double)v;
            lk[m] = make_double2(hi, (double)(v - (long double)hi));
        }
    }
    NUSHT_TRY(dev_alloc(&p->d_x2, (size_t)g.npairs, p));
    NUSHT_TRY(dev_alloc(&p->d_x2a, (size_t)g.npairs, p));
    for (int which = 0; which < 2; ++which) {
        // operand table of each decomposition: sin^2 for the blocks that use t = (alpha + beta) - alpha sin^2, cos^2
        // for the blocks (and remainder pairs) that use t = beta + alpha cos^2
        LegParams P = make_params(p);
        const int R = which ? ADJ_R : LEG_R, per = 32 * R;
        leg_grid(p, R, P);
        std::vector<double> u(g.npairs);
        for (int j = 0; j < g.npairs; ++j) {
            const bool in_rem = P.rem > 0 && j >= P.nblk * per;
            const bool xf = in_rem ? (P.nblk >= P.b_split) : (j / per >= P.b_split);
            u[j] = xf ? x2c[j] : x2[j];
        }
        NUSHT_CUDA_TRY(cudaMemcpy(which ? p->d_x2a : p->d_x2, u.data(), sizeof(double) * g.npairs, cudaMemcpyHostToDevice));
    }
    NUSHT_TRY(dev_alloc(&p->d_x, (size_t)g.npairs, p));
    NUSHT_TRY(dev_alloc(&p->d_logsin, (size_t)g.npairs, p));
    NUSHT_TRY(dev_alloc(&p->d_logkap, (size_t)M + 1, p));
    NUSHT_CUDA_TRY(cudaMemcpy(p->d_x, x.data(), sizeof(double) * g.npairs, cudaMemcpyHostToDevice));
    NUSHT_CUDA_TRY(cudaMemcpy(p->d_logsin, ls.data(), sizeof(double2) * g.npairs, cudaMemcpyHostToDevice));
    NUSHT_CUDA_TRY(cudaMemcpy(p->d_logkap, lk.data(), sizeof(double2) * (M + 1), cudaMemcpyHostToDevice));
    // fast-forward tables: one per decomposition of the ring pairs (LEG_R pairs per thread in the
    // synthesis, ADJ_R in the adjoint)
    {
        LegParams P = make_params(p);
        const dim3 grid = leg_grid(p, LEG_R, P);
        const size_t nw = (size_t)(M + 1) * (size_t)P.nblk;
        NUSHT_TRY(dev_alloc(&p->d_ff_n, nw, p));
        NUSHT_TRY(dev_alloc(&p->d_ff_p, nw * LEG_R * 32, p));
        NUSHT_TRY(dev_alloc(&p->d_ff_e, nw * LEG_R * 32, p));
        k_legendre_fastforward<LEG_R><<<dim3(P.nblk, M + 1), 32>>>(P, p->d_ff_n, p->d_ff_p, p->d_ff_e);
        NUSHT_CUDA_TRY(nusht_launched());
        (void)grid;
    }
    if (ADJ_R != LEG_R) {
        LegParams P = make_params(p);
        leg_grid(p, ADJ_R, P);
        const size_t nw = (size_t)(M + 1) * (size_t)P.nblk;
        NUSHT_TRY(dev_alloc(&p->d_ffa_n, nw, p));
        NUSHT_TRY(dev_alloc(&p->d_ffa_p, nw * ADJ_R * 32, p));
        NUSHT_TRY(dev_alloc(&p->d_ffa_e, nw * ADJ_R * 32, p));
        k_legendre_fastforward<ADJ_R><<<dim3(P.nblk, M + 1), 32>>>(P, p->d_ffa_n, p->d_ffa_p, p->d_ffa_e);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    NUSHT_CUDA_TRY(cudaDeviceSynchronize());
    NUSHT_TRY(build_work_list(p, LEG_R, p->d_ff_n, &p->d_items_syn, &p->n_items_syn));
    NUSHT_CUDA_TRY(cudaStreamCreateWithFlags(&p->s_leg_aux, cudaStreamNonBlocking));
    NUSHT_CUDA_TRY(cudaEventCreateWithFlags(&p->ev_leg_fork, cudaEventDisableTiming));
    NUSHT_CUDA_TRY(cudaEventCreateWithFlags(&p->ev_leg_join, cudaEventDisableTiming));
    return NUSHT_OK;
}

int legendre_alm_prep(nusht_plan_s* p, const void* alm, cudaStream_t s) {
    const int threads = PREP_THREADS, blocks = (p->mmax + 1 + threads / 32 - 1) / (threads / 32);
    if (p->dtype == NUSHT_F64)
        k_alm_prep<double><<<blocks, threads, 0, s>>>(p->lmax, p->lmax_io, p->mmax, p->d_eoff, (const double*)alm, p->d_sig,
                                                      p->d_sodd, p->d_rho, p->d_aeo);
    else
        k_alm_prep<float><<<blocks, threads, 0, s>>>(p->lmax, p->lmax_io, p->mmax, p->d_eoff, (const float*)alm, p->d_sig,
                                                     p->d_sodd, p->d_rho, p->d_aeo);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}

int legendre_synthesis(nusht_plan_s* p, double2* ft, cudaStream_t s) {
    LegParams P = make_params(p);
    leg_grid(p, LEG_R, P);
    if (p->n_items_syn == 0) return NUSHT_OK;
    if (p->lg.ring_mode)
        k_legendre_synth<LEG_R, true><<<p->n_items_syn, SYN_THREADS, 0, s>>>(P, p->d_aeo, ft);
    else
        k_legendre_synth<LEG_R, false><<<p->n_items_syn, SYN_THREADS, 0, s>>>(P, p->d_aeo, ft);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}

int legendre_adjoint(nusht_plan_s* p, const double2* gt, cudaStream_t s) {
    // the kernel accumulates with global reductions
    NUSHT_CUDA_TRY(cudaMemsetAsync(p->d_aeo, 0, sizeof(double4) * (size_t)p->n_e_total, s));
    LegParams P = make_params(p, true);
    const dim3 grid = leg_grid(p, ADJ_R, P);
    // one launch per form of t_n (see the kernel).  The two grids are independent (both add into eo with global
    // reductions), so the second one runs on a plan-owned side stream, forked from and joined to `s` with events:
    // they share the SMs instead of draining one after the other.
    const int nbx = (int)grid.x, split = std::min(P.b_split, nbx);
    const bool both = split > 0 && split < nbx;
    if (both) {
        NUSHT_CUDA_TRY(cudaEventRecord(p->ev_leg_fork, s));
        NUSHT_CUDA_TRY(cudaStreamWaitEvent(p->s_leg_aux, p->ev_leg_fork, 0));
    }
    for (int part = 1; part >= 0; --part) {
        LegParams Q = P;
        const int first = part ? split : 0, count = part ? nbx - split : split;
        if (count <= 0) continue;
        Q.b_split = first;                                   // block offset of this launch
        if (part) Q.ab = P.ab + p->n_e_total;                // cos^2 form of the table
        const dim3 g2(count, grid.y);
        cudaStream_t sl = (both && part == 0) ? p->s_leg_aux : s;
        if (p->lg.ring_mode)
            k_legendre_adjoint<ADJ_R, ADJ_CHUNK, true><<<g2, 32, 0, sl>>>(Q, gt, p->d_aeo);
        else
            k_legendre_adjoint<ADJ_R, ADJ_CHUNK, false><<<g2, 32, 0, sl>>>(Q, gt, p->d_aeo);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    if (both) {
        NUSHT_CUDA_TRY(cudaEventRecord(p->ev_leg_join, p->s_leg_aux));
        NUSHT_CUDA_TRY(cudaStreamWaitEvent(s, p->ev_leg_join, 0));
    }
    return NUSHT_OK;
}

int legendre_alm_post(nusht_plan_s* p, void* alm, cudaStream_t s) {
    const int threads = PREP_THREADS, blocks = (p->mmax + 1 + threads / 32 - 1) / (threads / 32);
    if (p->dtype == NUSHT_F64)
        k_alm_post<double><<<blocks, threads, 0, s>>>(p->lmax, p->lmax_io, p->mmax, p->d_eoff, p->d_aeo, p->d_sig, p->d_sodd,
                                                      p->d_rho, (double*)alm);
    else
        k_alm_post<float><<<blocks, threads, 0, s>>>(p->lmax, p->lmax_io, p->mmax, p->d_eoff, p->d_aeo, p->d_sig, p->d_sodd,
                                                     p->d_rho, (float*)alm);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}

// ---- a10 + a11 without any allocation (include/nusht.h: nusht_stage_legendre_adjoint_static) --------------------
// The even/odd accumulators of the adjoint live in a file-scope array of the library instead of the plan's d_aeo, for
// callers that cannot call cudaMalloc between set-up and tear-down.  262,656 = sum_m ((L - m)/2 + 1) at L = M = 1023.
// Every device that loads this module holds the array (8.02 MiB) until the process exits; every call on a device
// shares it (calls that overlap on the GPU race, see the header).
constexpr int64_t STATIC_EO_MAX = 262656;
static_assert(STATIC_EO_MAX * (int64_t)sizeof(double4) == NUSHT_STATIC_SCRATCH_BYTES, "header and array disagree");
static __device__ __align__(256) double4 g_static_eo[STATIC_EO_MAX];

// In host code `g_static_eo` is only the handle the runtime registered for the symbol, not an address a kernel can
// use: the device address is asked for once per device, with that device current, and cached here.
constexpr int STATIC_MAX_DEVICES = 64;
static std::mutex g_static_mu;
static double4* g_static_eo_dev[STATIC_MAX_DEVICES] = {};

static int static_eo_address(double4** out) {
    int dev = -1;
    NUSHT_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return NUSHT_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_eo_dev[dev]) {
        void* ptr = nullptr;
        NUSHT_CUDA_TRY(cudaGetSymbolAddress(&ptr, g_static_eo));
        if (!ptr) return NUSHT_ERR_CUDA;
        g_static_eo_dev[dev] = (double4*)ptr;
    }
    *out = g_static_eo_dev[dev];
    return NUSHT_OK;
}

int legendre_static_scratch(int64_t* bytes) {
    double4* eo = nullptr;
    NUSHT_TRY(static_eo_address(&eo));
    if (bytes) *bytes = STATIC_EO_MAX * (int64_t)sizeof(double4);
    return NUSHT_OK;
}

// legendre_adjoint + legendre_alm_post with `eo` = the static array: the same kernels, grids and side stream (those
// two functions are left as they are; this one repeats their launch logic)
int legendre_adjoint_static(nusht_plan_s* p, const double2* gt, void* alm, cudaStream_t s) {
    if (p->n_e_total > STATIC_EO_MAX) return NUSHT_ERR_TOO_LARGE;
    int dev = -1;
    NUSHT_CUDA_TRY(cudaGetDevice(&dev));
    if (dev != p->device) return NUSHT_ERR_INVALID_ARG;
    double4* eo = nullptr;
    NUSHT_TRY(static_eo_address(&eo));
    // the kernels accumulate with global reductions and the array holds the previous call's sums
    NUSHT_CUDA_TRY(cudaMemsetAsync(eo, 0, sizeof(double4) * (size_t)p->n_e_total, s));
    LegParams P = make_params(p, true);
    const dim3 grid = leg_grid(p, ADJ_R, P);
    const int nbx = (int)grid.x, split = std::min(P.b_split, nbx);
    const bool both = split > 0 && split < nbx;
    if (both) {
        NUSHT_CUDA_TRY(cudaEventRecord(p->ev_leg_fork, s));
        NUSHT_CUDA_TRY(cudaStreamWaitEvent(p->s_leg_aux, p->ev_leg_fork, 0));
    }
    for (int part = 1; part >= 0; --part) {
        LegParams Q = P;
        const int first = part ? split : 0, count = part ? nbx - split : split;
        if (count <= 0) continue;
        Q.b_split = first;
        if (part) Q.ab = P.ab + p->n_e_total;
        const dim3 g2(count, grid.y);
        cudaStream_t sl = (both && part == 0) ? p->s_leg_aux : s;
        if (p->lg.ring_mode)
            k_legendre_adjoint<ADJ_R, ADJ_CHUNK, true><<<g2, 32, 0, sl>>>(Q, gt, eo);
        else
            k_legendre_adjoint<ADJ_R, ADJ_CHUNK, false><<<g2, 32, 0, sl>>>(Q, gt, eo);
        NUSHT_CUDA_TRY(nusht_launched());
    }
    if (both) {
        NUSHT_CUDA_TRY(cudaEventRecord(p->ev_leg_join, p->s_leg_aux));
        NUSHT_CUDA_TRY(cudaStreamWaitEvent(s, p->ev_leg_join, 0));
    }
    const int threads = PREP_THREADS, blocks = (p->mmax + 1 + threads / 32 - 1) / (threads / 32);
    if (p->dtype == NUSHT_F64)
        k_alm_post<double><<<blocks, threads, 0, s>>>(p->lmax, p->lmax_io, p->mmax, p->d_eoff, eo, p->d_sig, p->d_sodd,
                                                      p->d_rho, (double*)alm);
    else
        k_alm_post<float><<<blocks, threads, 0, s>>>(p->lmax, p->lmax_io, p->mmax, p->d_eoff, eo, p->d_sig, p->d_sodd,
                                                     p->d_rho, (float*)alm);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}

void legendre_free(nusht_plan_s* p) {
    if (p->s_leg_aux) cudaStreamDestroy(p->s_leg_aux);
    if (p->ev_leg_fork) cudaEventDestroy(p->ev_leg_fork);
    if (p->ev_leg_join) cudaEventDestroy(p->ev_leg_join);
    p->s_leg_aux = nullptr;
    p->ev_leg_fork = p->ev_leg_join = nullptr;
    cudaFree(p->d_items_syn);
    p->d_items_syn = nullptr;
    cudaFree(p->d_pair_n); cudaFree(p->d_pair_s);
    p->d_pair_n = p->d_pair_s = nullptr;
    cudaFree(p->d_eoff); cudaFree(p->d_ab); cudaFree(p->d_sig); cudaFree(p->d_sodd); cudaFree(p->d_rho);
    cudaFree(p->d_aeo); cudaFree(p->d_ft); cudaFree(p->d_x2); cudaFree(p->d_x2a); cudaFree(p->d_x); cudaFree(p->d_logsin);
    p->d_x2a = nullptr;
    cudaFree(p->d_logkap);
    cudaFree(p->d_ff_n); cudaFree(p->d_ff_p); cudaFree(p->d_ff_e);
    cudaFree(p->d_ffa_n); cudaFree(p->d_ffa_p); cudaFree(p->d_ffa_e);
    p->d_ff_n = nullptr; p->d_ff_p = nullptr; p->d_ff_e = nullptr;
    p->d_ffa_n = nullptr; p->d_ffa_p = nullptr; p->d_ffa_e = nullptr;
    p->d_eoff = nullptr; p->d_ab = nullptr; p->d_sig = p->d_sodd = p->d_rho = nullptr; p->d_aeo = nullptr;
    p->d_ft = nullptr; p->d_x2 = p->d_x = nullptr; p->d_logsin = p->d_logkap = nullptr;
}
