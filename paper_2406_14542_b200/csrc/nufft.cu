// nufft.cu -- nonuniform part of the nuSHT (operator N and its transpose; arXiv 2406.14542
// Eq. 5-6).
//
//   a6  plan time: counting sort of the points by the origin of their kernel footprint
//   a7  type-2 interpolation   f_j = sum_{a,b<w} g[a0+a][b0+b] psi(a0+a-X_j) psi(b0+b-Y_j)
//   a8  type-1 spreading       g[a0+a][b0+b] += x_j psi(a0+a-X_j) psi(b0+b-Y_j)
// with X = theta n_theta/(2 pi), Y = phi n_phi/(2 pi), a0 = ceil(X - w/2), b0 = ceil(Y - w/2) and
// psi(x) = phi_ES(2x/w), phi_ES(z) = exp(beta (sqrt(1-z^2) - 1)) -- the "exponential of semicircle"
// kernel of the paper's ref. [38], evaluated as a piecewise polynomial of
// degree `deg` in the fractional offset (one polynomial per tap; coefficients fitted at plan time at
// Chebyshev nodes in extended precision).  The deconvolution factors (fourier.cu) are the Fourier
// transform of THIS piecewise polynomial, so the approximation is self-consistent.
//
// B200 design (differs from the shared-memory-atomics scheme of the library the paper wraps):
// the fine grid is cut into strips of 33-w patch-origin columns; one WARP owns one strip segment
// and each LANE owns one grid column of the strip (strip + halo = 32 columns).  Points are sorted
// by row of their footprint origin, so the warp walks down the strip with a w-row sliding window
// held in registers: interpolation reads every grid row once (coalesced), spreading accumulates
// in registers with no shared-memory atomics and flushes each finished row with one coalesced
// native global atomic add per lane.  The grid stores only theta in [0, pi] (n_theta/2+1 rows);
// rows beyond the poles are the DFS mirror  g[-a][b] = g[a][b + n_phi/2].
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <mutex>
#include <type_traits>
#include <vector>

#include "nusht_internal.cuh"

namespace {

constexpr double TWO_PI = 6.283185307179586476925286766559;

template <typename T>
struct KernelPoly {
    T c[NUSHT_MAX_W][NUSHT_MAX_DEG + 1];   // c[tap][power of u], u = 2 xi - 1 in [-1, 1)
};

// host copies (one per plan would be cleaner; kept in the plan through these pointers)
struct KernelHost {
    int w = 0, deg = 0;
    double beta = 0;
    long double c[NUSHT_MAX_W][NUSHT_MAX_DEG + 1];
};

__host__ __device__ constexpr int poly_degree(int w) { return w < 5 ? 5 : w; }
// row stride (in elements) of the broadcast weight table: even, with stride/2 odd, so that
// 128-bit stores by 8 consecutive lanes hit 8 different 16-byte bank groups
__host__ __device__ constexpr int kth_stride(int w) {
    int s = (w + 1) & ~1;
    if (((s / 2) & 1) == 0) s += 2;
    return s;
}

// ---------------------------------------------------------------------------------------------
// a6: point keys, histogram, scan, scatter
// ---------------------------------------------------------------------------------------------
struct SortGeom {
    int nth, nph, w, fl, mb, nstrip, nseg;
    double inv_hth, inv_hph, half_w;
};

__device__ __forceinline__ bool point_coords(const SortGeom& g, double th, double ph, double& X, double& Y,
                                             int& ra, int& cb) {
    if (!(th >= 0.0) || !(th <= 3.14159265358979323846) || !isfinite(ph)) return false;
    X = th * g.inv_hth;
    double phw = ph - TWO_PI * floor(ph * (1.0 / TWO_PI));
    if (phw < 0.0) phw = 0.0;
    Y = phw * g.inv_hph;
    if (Y >= (double)g.nph) Y -= (double)g.nph;
    // the same two expressions are re-evaluated by the interp/spread kernels from the stored (X, Y):
    // identical IEEE operations, hence identical origins.  cb may equal nph (last strip wraps).
    const int a0 = (int)ceil(X - g.half_w);
    const int b0 = (int)ceil(Y - g.half_w);
    ra = a0 + g.fl;
    cb = b0 + g.fl;
    return true;
}

__global__ void k_point_keys(SortGeom g, int64_t npts, const double* __restrict__ theta,
                             const double* __restrict__ phi, int* __restrict__ keys, int* __restrict__ ranks,
                             int* __restrict__ hist, int* __restrict__ bad) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npts) return;
    double X, Y;
    int ra, cb;
    if (!point_coords(g, theta[i], phi[i], X, Y, ra, cb)) {
        atomicAdd(bad, 1);
        keys[i] = 0;
        ranks[i] = 0;
        return;
    }
    const int seg = ra / NUSHT_SEG_ROWS, strip = cb / g.mb;
    const int key = (seg * g.nstrip + strip) * NUSHT_SEG_ROWS + (ra - seg * NUSHT_SEG_ROWS);
    keys[i] = key;
    ranks[i] = atomicAdd(&hist[key], 1);      // rank of the point inside its bin: the scatter needs no second atomic
}

constexpr int SCAN_BLOCK = 256;
constexpr int SCAN_ITEMS = 8;   // per thread
constexpr int SCAN_TILE = SCAN_BLOCK * SCAN_ITEMS;

// exclusive scan in three launches: per-tile scan + tile totals, scan of totals (one CTA), add back
__global__ void k_scan_tiles(const int* __restrict__ in, int* __restrict__ out, int* __restrict__ totals, int n) {
    __shared__ int s_warp[SCAN_BLOCK / 32];
    const int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
    int v[SCAN_ITEMS], sum = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        v[k] = (base + k < n) ? in[base + k] : 0;
        sum += v[k];
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int inc = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        int t = (lane < SCAN_BLOCK / 32) ? s_warp[lane] : 0;
#pragma unroll
        for (int d = 1; d < SCAN_BLOCK / 32; d <<= 1) {
            int u = __shfl_up_sync(0xffffffffu, t, d);
            if (lane >= d) t += u;
        }
        if (lane < SCAN_BLOCK / 32) s_warp[lane] = t;
    }
    __syncthreads();
    int run = inc - sum + (warp > 0 ? s_warp[warp - 1] : 0);
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < n) out[base + k] = run;
        run += v[k];
    }
    if (threadIdx.x == SCAN_BLOCK - 1) totals[blockIdx.x] = run;
}

__global__ void k_scan_totals(int* totals, int ntiles) {
    // single CTA, sequential over chunks of blockDim
    __shared__ int s[1024];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < ntiles; base += blockDim.x) {
        const int i = base + threadIdx.x;
        const int v = (i < ntiles) ? totals[i] : 0;
        s[threadIdx.x] = v;
        __syncthreads();
        for (int d = 1; d < blockDim.x; d <<= 1) {
            int t = (threadIdx.x >= d) ? s[threadIdx.x - d] : 0;
            __syncthreads();
            s[threadIdx.x] += t;
            __syncthreads();
        }
        if (i < ntiles) totals[i] = carry + s[threadIdx.x] - v;
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) carry += s[threadIdx.x];
        __syncthreads();
    }
}

__global__ void k_scan_add(int* __restrict__ out, const int* __restrict__ totals, int n) {
    const int i = blockIdx.x * SCAN_TILE + threadIdx.x;
    const int add = totals[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        const int q = i + k * SCAN_BLOCK;
        if (q < n) out[q] += add;
    }
}

// ---------------------------------------------------------------------------------------------
// L2-blocked un-permutation (plan-time tables + one run-time copy kernel).
// The transforms work on points in sorted order but `map` is in the caller's order, and the caller's
// order is random with respect to the grid: writing f_j straight to map[perm[j]] is npts isolated
// 4-byte stores, each a read-modify-write of a DRAM sector (1.8 ms at 67 M points in FP32, more than
// the interpolation itself).  Instead the caller's index range is cut into n_buckets ranges small
// enough to stay in the 126 MB L2 (2^22 elements); at plan time every sorted position gets a slot in
// bucket-major order (stable inside a bucket, so a warp's 32 results go to n_buckets short
// contiguous runs that L2 merges into full sectors), and at run time k_unpermute walks the slots
// in order: coalesced reads, and the random writes of one bucket all land in an L2-resident range
// whose sectors are complete before they are evicted.
// ---------------------------------------------------------------------------------------------
constexpr int BUCKET_SHIFT = 22;           // caller indices per bucket: 2^22 (16 MB of FP32; measured best of 2^22..2^24), more if that gives over 31 buckets
constexpr int BUCKET_MAX = 31;             // lane b of a warp keeps bucket b's counter
constexpr int BUCKET_CHUNK = 1024;         // consecutive sorted positions per warp
constexpr int BUCKET_WARPS = 4;

__global__ void __launch_bounds__(32 * BUCKET_WARPS)
k_bucket_count(const int* __restrict__ perm, int64_t npts, int shift, int nchunks, int* __restrict__ cnt) {
    __shared__ int s_cnt[BUCKET_WARPS][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int chunk = blockIdx.x * BUCKET_WARPS + warp;
    if (chunk >= nchunks) return;
    s_cnt[warp][lane] = 0;
    __syncwarp();
    const int64_t base = (int64_t)chunk * BUCKET_CHUNK;
    for (int r = 0; r < BUCKET_CHUNK; r += 32) {
        const int64_t i = base + r + lane;
        const int b = (i < npts) ? (perm[i] >> shift) : BUCKET_MAX;   // absent points: a bucket nobody uses
        const unsigned mask = __match_any_sync(0xffffffffu, b);
        if (lane == __ffs(mask) - 1) s_cnt[warp][b] += __popc(mask);
        __syncwarp();
    }
    if (lane < BUCKET_MAX) cnt[(int64_t)lane * nchunks + chunk] = s_cnt[warp][lane];   // bucket-major matrix
}

__global__ void __launch_bounds__(32 * BUCKET_WARPS)
k_bucket_place(const int* __restrict__ perm, int64_t npts, int shift, int nchunks, const int* __restrict__ off,
               int* __restrict__ slot, int* __restrict__ dest) {
    __shared__ int s_off[BUCKET_WARPS][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int chunk = blockIdx.x * BUCKET_WARPS + warp;
    if (chunk >= nchunks) return;
    s_off[warp][lane] = (lane < BUCKET_MAX) ? off[(int64_t)lane * nchunks + chunk] : 0;
    __syncwarp();
    const int64_t base = (int64_t)chunk * BUCKET_CHUNK;
    for (int r = 0; r < BUCKET_CHUNK; r += 32) {
        const int64_t i = base + r + lane;
        const bool has = i < npts;
        const int dst = has ? perm[i] : 0;
        const int b = has ? (dst >> shift) : BUCKET_MAX;
        const unsigned mask = __match_any_sync(0xffffffffu, b);
        const int at = s_off[warp][b] + __popc(mask & ((1u << lane) - 1u));
        __syncwarp();
        if (lane == 31 - __clz(mask)) s_off[warp][b] = at + 1;     // last lane of the group
        __syncwarp();
        if (has) {
            slot[i] = at;
            dest[at] = dst;
        }
    }
}

template <typename T>
__global__ void __launch_bounds__(256)
k_unpermute(const T* __restrict__ stage, const int* __restrict__ dest, int64_t npts, T* __restrict__ map) {
    const int64_t e = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (e < npts) map[dest[e]] = stage[e];
}

__global__ void k_item_offsets(const int* __restrict__ bin_off, int* __restrict__ item_off, int n_items,
                               int npts) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_items) item_off[i] = bin_off[(int64_t)i * NUSHT_SEG_ROWS];
    if (i == n_items) item_off[i] = npts;
}

// The scatter writes ONE 32-byte record per point (a whole DRAM sector: no read-modify-write), and k_point_unpack
// splits the records into the three arrays the transforms read, with coalesced accesses on both sides.  Writing
// px[pos], py[pos], perm[pos] directly is three isolated partial-sector writes per point: 9.9 ms at 67 M points
// against 0.44 ms for the key / histogram pass.
struct __align__(32) PointRec {
    double X, Y;
    int perm, pad0;
    long long pad1;
};

__global__ void k_point_scatter(SortGeom g, int64_t npts, const double* __restrict__ theta,
                                const double* __restrict__ phi, const int* __restrict__ keys,
                                const int* __restrict__ ranks, const int* __restrict__ bin_off,
                                PointRec* __restrict__ rec) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npts) return;
    double X, Y;
    int ra, cb;
    point_coords(g, theta[i], phi[i], X, Y, ra, cb);
    const int pos = bin_off[keys[i]] + ranks[i];
    double2* out = reinterpret_cast<double2*>(rec + pos);
    out[0] = make_double2(X, Y);
    out[1] = make_double2(__longlong_as_double((long long)(unsigned)i), 0.0);
}

__global__ void k_point_unpack(int64_t npts, const PointRec* __restrict__ rec, double* __restrict__ px,
                               double* __restrict__ py, int* __restrict__ perm) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npts) return;
    const double2* in = reinterpret_cast<const double2*>(rec + i);
    const double2 a = in[0], b = in[1];
    px[i] = a.x;
    py[i] = a.y;
    perm[i] = (int)__double_as_longlong(b.x);
}

// ---------------------------------------------------------------------------------------------
// kernel evaluation: w polynomials of degree DEG in u, coefficients read from the kernel-parameter
// constant bank (uniform operands, no loads)
// ---------------------------------------------------------------------------------------------
// The kernel is even, so tap W-1-i is tap i evaluated at -u: c[W-1-i][d] = (-1)^d c[i][d] (enforced
// exactly at plan time).  Taps i and W-1-i share the even and odd parts E_i(u^2) +- u O_i(u^2).
template <int W, typename T>
__device__ __forceinline__ void eval_taps(const KernelPoly<T>& kp, T u, T (&k)[W]) {
    constexpr int DEG = poly_degree(W);
    constexpr int DE = DEG & ~1;            // highest even power
    constexpr int DO = (DEG - 1) | 1;       // highest odd power
    const T u2 = u * u;
#pragma unroll
    for (int i = 0; i < W / 2; ++i) {
        T e = kp.c[i][DE], o = kp.c[i][DO];
#pragma unroll
        for (int d = DE - 2; d >= 0; d -= 2) e = fma(e, u2, kp.c[i][d]);
#pragma unroll
        for (int d = DO - 2; d >= 1; d -= 2) o = fma(o, u2, kp.c[i][d]);
        k[i] = fma(u, o, e);
        k[W - 1 - i] = fma(-u, o, e);
    }
    if (W & 1) {
        T e = kp.c[W / 2][DE];
#pragma unroll
        for (int d = DE - 2; d >= 0; d -= 2) e = fma(e, u2, kp.c[W / 2][d]);
        k[W / 2] = e;
    }
}

struct NufftParams {
    NufftGeom g;
    const double* px;
    const double* py;
    const int* perm;
    const int* item_off;
    int n_items;
};

// warps (= independent work items) per CTA; fewer for wide double-precision kernels so that the
// per-warp scratch stays inside the 48 KB static shared-memory window
template <int W, typename T>
__host__ __device__ constexpr int nu_warps() { return (W * (int)sizeof(T) > 96) ? 2 : 4; }

template <int W, typename T>
struct WarpScratch {
    static constexpr int SK = kth_stride(W);
    static constexpr int SP = W | 1;
    T th[32][SK];       // per point: theta-direction weights (broadcast reads, 128-bit where possible)
    T ph[32][SP];       // per point: phi-direction weights (lane-indexed reads)
    T part[32][SP];     // interp: per point, per active lane partial sums
    int oy[32];         // per point: lane of the first footprint column
};

// fine-grid row offset and mirror flag of logical row a (may lie beyond a pole)
__device__ __forceinline__ int64_t grid_row(const NufftGeom& g, int a, bool& mirror) {
    int am = a;
    if (am < 0) am += g.nth;
    if (am >= g.nth) am -= g.nth;
    mirror = am > g.nth / 2;
    return (int64_t)(mirror ? g.nth - am : am) * g.nph;
}

// fine-grid row/column of logical row a (may lie beyond a pole) for a lane
__device__ __forceinline__ int64_t grid_index(const NufftGeom& g, int a, int col_n, int col_m) {
    int am = a;
    if (am < 0) am += g.nth;
    if (am >= g.nth) am -= g.nth;
    const bool mirror = am > g.nth / 2;
    const int row = mirror ? g.nth - am : am;
    return (int64_t)row * g.nph + (mirror ? col_m : col_n);
}

// ---------------------------------------------------------------------------------------------
// per-batch prologue shared by a7 and a8: lane `lane` evaluates the 2W weights of point batch+lane
// and publishes them; returns the bit mask of points that start a new row run (points are sorted
// by the row a0 of their footprint origin inside a work item).
// ---------------------------------------------------------------------------------------------
template <typename T> struct Vec2;
template <> struct Vec2<double> { using type = double2; };
template <> struct Vec2<float> { using type = float2; };

template <int W, typename T>
__device__ __forceinline__ unsigned publish_weights(WarpScratch<W, T>& ws, const KernelPoly<T>& kp, int lane,
                                                    bool has, double X, double Y, T val, int c0, int& a0) {
    using V2 = typename Vec2<T>::type;
    const double a0d = ceil(X - 0.5 * W), b0d = ceil(Y - 0.5 * W);
    const T ut = (T)(2.0 * ((a0d + 0.5 * W) - X) - 1.0);
    const T up = (T)(2.0 * ((b0d + 0.5 * W) - Y) - 1.0);
    T k[W];
    eval_taps<W, T>(kp, ut, k);
#pragma unroll
    for (int i = 0; i + 1 < W; i += 2) {
        V2 v;
        v.x = val * k[i];
        v.y = val * k[i + 1];
        *reinterpret_cast<V2*>(&ws.th[lane][i]) = v;
    }
    if (W & 1) {
        V2 v;
        v.x = val * k[W - 1];
        v.y = 0;
        *reinterpret_cast<V2*>(&ws.th[lane][W - 1]) = v;
    }
    eval_taps<W, T>(kp, up, k);
#pragma unroll
    for (int i = 0; i < W; ++i) ws.ph[lane][i] = k[i];
    ws.oy[lane] = (int)b0d - c0;
    a0 = (int)a0d;
    const int a0_prev = __shfl_up_sync(0xffffffffu, a0, 1);
    return __ballot_sync(0xffffffffu, has && (lane == 0 || a0 != a0_prev));
}

// theta contraction of one point against the register window: two independent FMA chains
template <int W, typename T>
__device__ __forceinline__ T contract(const T* th, const T (&win)[W]) {
    using V2 = typename Vec2<T>::type;
    T acc0 = 0, acc1 = 0;
#pragma unroll
    for (int i = 0; i + 1 < W; i += 2) {
        const V2 kk = *reinterpret_cast<const V2*>(th + i);
        acc0 = fma(kk.x, win[i], acc0);
        acc1 = fma(kk.y, win[i + 1], acc1);
    }
    if (W & 1) acc0 = fma(th[W - 1], win[W - 1], acc0);
    return acc0 + acc1;
}

// ---------------------------------------------------------------------------------------------
// a7: type-2 interpolation
// ---------------------------------------------------------------------------------------------
template <int W, typename T>
__global__ void __launch_bounds__(nu_warps<W, T>() * 32)
k_interp(const __grid_constant__ NufftParams P, const __grid_constant__ KernelPoly<T> kp,
         const T* __restrict__ grid, T* __restrict__ map) {
    using WS = WarpScratch<W, T>;
    constexpr int NU_WARPS = nu_warps<W, T>();
    __shared__ __align__(16) WS s_ws[NU_WARPS];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int item = blockIdx.x * NU_WARPS + warp;
    if (item >= P.n_items) return;
    const int start = P.item_off[item], end = P.item_off[item + 1];
    if (start >= end) return;
    WS& ws = s_ws[warp];
    const NufftGeom& g = P.g;
    const int strip = item % g.nstrip;
    const int c0 = strip * g.mb - g.fl;   // global column of lane 0
    int col_n = (c0 + lane) % g.nph;
    if (col_n < 0) col_n += g.nph;
    int col_m = col_n + g.nph / 2;
    if (col_m >= g.nph) col_m -= g.nph;

    T win[W];     // win[i] = g[a_base + i][column of this lane]
    T nxt = 0;    // prefetched row a_base + W
    int a_base = INT_MIN;

    // coordinates of the next batch are loaded one batch ahead
    double Xn = 0.0, Yn = 0.0;
    if (start + lane < end) {
        Xn = P.px[start + lane];
        Yn = P.py[start + lane];
    }
    for (int batch = start; batch < end; batch += 32) {
        const int idx = batch + lane;
        const bool has = idx < end;
        const double X = Xn, Y = Yn;
        if (idx + 32 < end) {
            Xn = P.px[idx + 32];
            Yn = P.py[idx + 32];
        }
        int a0;
        const unsigned starts = publish_weights<W, T>(ws, kp, lane, has, X, Y, (T)1, c0, a0);
        __syncwarp();
        const int npt = min(32, end - batch);
        int j = 0;
        while (j < npt) {
            // ---- slide the register window down to the row of point j (warp-uniform) ----
            const int row = __shfl_sync(0xffffffffu, a0, j);
            if (row != a_base) {
                int d = (a_base == INT_MIN) ? W : row - a_base;
                if (d >= W) {
                    a_base = row;
#pragma unroll
                    for (int i = 0; i < W; ++i) win[i] = grid[grid_index(g, a_base + i, col_n, col_m)];
                    nxt = grid[grid_index(g, a_base + W, col_n, col_m)];
                } else {
#pragma unroll 1
                    for (; d > 0; --d) {
#pragma unroll
                        for (int i = 0; i + 1 < W; ++i) win[i] = win[i + 1];
                        win[W - 1] = nxt;
                        a_base += 1;
                        nxt = grid[grid_index(g, a_base + W, col_n, col_m)];
                    }
                }
            }
            // ---- the run of points whose footprint starts on this row: the window is loop-invariant,
            //      two points per iteration for instruction-level parallelism ----
            const unsigned rest = (j < 31) ? (starts >> (j + 1)) : 0u;
            const int run_end = rest ? j + __ffs(rest) : npt;
#pragma unroll 1
            for (; j + 1 < run_end; j += 2) {
                const T s0 = contract<W, T>(&ws.th[j][0], win);
                const T s1 = contract<W, T>(&ws.th[j + 1][0], win);
                const unsigned t0 = (unsigned)(lane - ws.oy[j]), t1 = (unsigned)(lane - ws.oy[j + 1]);
                const T p0 = (t0 < (unsigned)W) ? ws.ph[j][t0] : (T)0;
                const T p1 = (t1 < (unsigned)W) ? ws.ph[j + 1][t1] : (T)0;
                if (t0 < (unsigned)W) ws.part[j][t0] = s0 * p0;
                if (t1 < (unsigned)W) ws.part[j + 1][t1] = s1 * p1;
            }
            if (j < run_end) {
                const T s0 = contract<W, T>(&ws.th[j][0], win);
                const unsigned t0 = (unsigned)(lane - ws.oy[j]);
                if (t0 < (unsigned)W) ws.part[j][t0] = s0 * ws.ph[j][t0];
                ++j;
            }
        }
        __syncwarp();
        if (has) {
            T sum = 0;
#pragma unroll
            for (int t = 0; t < W; ++t) sum += ws.part[lane][t];
            map[P.perm[idx]] = sum;
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------
// a7, FP32 path at small widths (eps >= 1e-6, W <= 8): one THREAD per point, the W x W footprint
// gathered straight from the grid through L1.  The sorted order (segment, strip, row) keeps the 32
// points of a warp inside about two grid rows of one strip, so each of the W^2 load instructions
// touches two to four 128-byte lines that stay L1-resident across the footprint; per point the
// warp issues about 5 instructions instead of the ~20 of the register-window kernel, which is
// issue-bound at these widths (2.8 ms at W = 5, 7 for an HBM floor of 0.3 ms at config 5).
// Same arithmetic as k_interp: weights from eval_taps, theta contraction innermost per column is
// replaced by phi innermost per row (sum order differs: FP32 rounding only).
// ---------------------------------------------------------------------------------------------
constexpr int GATHER_THREADS = 256;

template <int W>
__global__ void __launch_bounds__(GATHER_THREADS)
k_interp_gather(const __grid_constant__ NufftParams P, const __grid_constant__ KernelPoly<float> kp, int64_t npts,
                const float* __restrict__ grid, float* __restrict__ map) {
    const int64_t idx = (int64_t)blockIdx.x * GATHER_THREADS + threadIdx.x;
    if (idx >= npts) return;
    const NufftGeom& g = P.g;
    const double X = P.px[idx], Y = P.py[idx];
    const int out = P.perm[idx];
    const double a0d = ceil(X - 0.5 * W), b0d = ceil(Y - 0.5 * W);
    const float ut = (float)(2.0 * ((a0d + 0.5 * W) - X) - 1.0);
    const float up = (float)(2.0 * ((b0d + 0.5 * W) - Y) - 1.0);
    float kt[W], kph[W];
    eval_taps<W, float>(kp, ut, kt);
    eval_taps<W, float>(kp, up, kph);
    const int a0 = (int)a0d;
    int b0 = (int)b0d;                       // in [-W/2, nph]
    if (b0 < 0) b0 += g.nph;
    if (b0 >= g.nph) b0 -= g.nph;
    int bm = b0 + g.nph / 2;                 // first column on a mirrored row (beyond a pole)
    if (bm >= g.nph) bm -= g.nph;
    // Interior footprints (no pole, no phi wrap) are read as NV aligned column PAIRS per row (64-bit loads:
    // n_phi is even, so every row starts 8-byte aligned): the W weights are shifted by the parity of b0 into
    // a (2 NV)-entry row with zeros at the ends, once per point, instead of W 32-bit loads per row.
    constexpr int NV = W / 2 + 1;
    const int q = b0 & 1, ba = b0 - q;
    const bool interior = (a0 >= 0) && (a0 + W - 1 <= g.nth / 2) && (ba + 2 * NV <= g.nph) && ((g.nph & 1) == 0);
    float sum = 0.f;
    if (interior) {
        float ks[2 * NV];
#pragma unroll
        for (int j = 0; j < 2 * NV; ++j) {
            const float lo = (j < W) ? kph[j < W ? j : 0] : 0.f;                  // q = 0: weight j
            const float hi = (j >= 1 && j - 1 < W) ? kph[(j >= 1 && j - 1 < W) ? j - 1 : 0] : 0.f;   // q = 1: weight j - 1
            ks[j] = q ? hi : lo;
        }
        const float2* src = reinterpret_cast<const float2*>(grid + (int64_t)a0 * g.nph + ba);
        const int64_t stride2 = g.nph / 2;
#pragma unroll
        for (int i = 0; i < W; ++i) {
            float r0 = 0.f, r1 = 0.f;
#pragma unroll
            for (int j = 0; j < NV; ++j) {
                const float2 v = __ldg(src + j);
                r0 = fmaf(ks[2 * j], v.x, r0);
                r1 = fmaf(ks[2 * j + 1], v.y, r1);
            }
            sum = fmaf(kt[i], r0 + r1, sum);
            src += stride2;
        }
    } else {
#pragma unroll
        for (int i = 0; i < W; ++i) {
            bool mirror;
            const int64_t base = grid_row(g, a0 + i, mirror);
            int c = mirror ? bm : b0;
            float r = 0.f;
#pragma unroll
            for (int j = 0; j < W; ++j) {
                r = fmaf(kph[j], __ldg(grid + base + c), r);
                c = (c + 1 == g.nph) ? 0 : c + 1;
            }
            sum = fmaf(kt[i], r, sum);
        }
    }
    map[out] = sum;
}

// ---------------------------------------------------------------------------------------------
// a8: type-1 spreading (grid must be zero on entry)
// ---------------------------------------------------------------------------------------------
template <int W, typename T>
__device__ __forceinline__ void spread_point(const T* th, T kph, T (&acc)[W]) {
    using V2 = typename Vec2<T>::type;
#pragma unroll
    for (int i = 0; i + 1 < W; i += 2) {
        const V2 kk = *reinterpret_cast<const V2*>(th + i);
        acc[i] = fma(kk.x, kph, acc[i]);
        acc[i + 1] = fma(kk.y, kph, acc[i + 1]);
    }
    if (W & 1) acc[W - 1] = fma(th[W - 1], kph, acc[W - 1]);
}

template <int W, typename T>
__global__ void __launch_bounds__(nu_warps<W, T>() * 32)
k_spread(const __grid_constant__ NufftParams P, const __grid_constant__ KernelPoly<T> kp,
         const T* __restrict__ map, T* __restrict__ grid) {
    using WS = WarpScratch<W, T>;
    constexpr int NU_WARPS = nu_warps<W, T>();
    __shared__ __align__(16) WS s_ws[NU_WARPS];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int item = blockIdx.x * NU_WARPS + warp;
    if (item >= P.n_items) return;
    const int start = P.item_off[item], end = P.item_off[item + 1];
    if (start >= end) return;
    WS& ws = s_ws[warp];
    const NufftGeom& g = P.g;
    const int strip = item % g.nstrip;
    const int c0 = strip * g.mb - g.fl;
    int col_n = (c0 + lane) % g.nph;
    if (col_n < 0) col_n += g.nph;
    int col_m = col_n + g.nph / 2;
    if (col_m >= g.nph) col_m -= g.nph;

    T acc[W];     // acc[i] accumulates g[a_base + i][column of this lane]
#pragma unroll
    for (int i = 0; i < W; ++i) acc[i] = 0;
    int a_base = INT_MIN;

    double Xn = 0.0, Yn = 0.0;     // one batch ahead; the index of the value two batches ahead (see k_spread_mma)
    T vn = 0;
    int pn = 0;
    if (start + lane < end) {
        Xn = P.px[start + lane];
        Yn = P.py[start + lane];
        vn = map[P.perm[start + lane]];
    }
    if (start + 32 + lane < end) pn = P.perm[start + 32 + lane];
    for (int batch = start; batch < end; batch += 32) {
        const int idx = batch + lane;
        const bool has = idx < end;
        const double X = Xn, Y = Yn;
        const T val = has ? vn : (T)0;
        if (idx + 32 < end) {
            Xn = P.px[idx + 32];
            Yn = P.py[idx + 32];
            vn = map[pn];
        }
        if (idx + 64 < end) pn = P.perm[idx + 64];
        int a0;
        // the point's value rides on the theta weights
        const unsigned starts = publish_weights<W, T>(ws, kp, lane, has, X, Y, val, c0, a0);
        __syncwarp();
        const int npt = min(32, end - batch);
        int j = 0;
        while (j < npt) {
            const int row = __shfl_sync(0xffffffffu, a0, j);
            if (row != a_base) {
                if (a_base == INT_MIN) {
                    a_base = row;
                } else {
                    int d = row - a_base;
                    if (d >= W) {
                        // flush the whole window
#pragma unroll
                        for (int i = 0; i < W; ++i) {
                            if (acc[i] != (T)0) atomicAdd(&grid[grid_index(g, a_base + i, col_n, col_m)], acc[i]);
                            acc[i] = 0;
                        }
                        a_base = row;
                    } else {
#pragma unroll 1
                        for (; d > 0; --d) {
                            if (acc[0] != (T)0) atomicAdd(&grid[grid_index(g, a_base, col_n, col_m)], acc[0]);
#pragma unroll
                            for (int i = 0; i + 1 < W; ++i) acc[i] = acc[i + 1];
                            acc[W - 1] = 0;
                            a_base += 1;
                        }
                    }
                }
            }
            const unsigned rest = (j < 31) ? (starts >> (j + 1)) : 0u;
            const int run_end = rest ? j + __ffs(rest) : npt;
#pragma unroll 1
            for (; j + 1 < run_end; j += 2) {
                const unsigned t0 = (unsigned)(lane - ws.oy[j]), t1 = (unsigned)(lane - ws.oy[j + 1]);
                const T p0 = (t0 < (unsigned)W) ? ws.ph[j][t0] : (T)0;
                const T p1 = (t1 < (unsigned)W) ? ws.ph[j + 1][t1] : (T)0;
                spread_point<W, T>(&ws.th[j][0], p0, acc);
                spread_point<W, T>(&ws.th[j + 1][0], p1, acc);
            }
            if (j < run_end) {
                const unsigned t0 = (unsigned)(lane - ws.oy[j]);
                const T p0 = (t0 < (unsigned)W) ? ws.ph[j][t0] : (T)0;
                spread_point<W, T>(&ws.th[j][0], p0, acc);
                ++j;
            }
        }
        __syncwarp();
    }
    if (a_base != INT_MIN) {
#pragma unroll
        for (int i = 0; i < W; ++i)
            if (acc[i] != (T)0) atomicAdd(&grid[grid_index(g, a_base + i, col_n, col_m)], acc[i]);
    }
}

template <typename T>
KernelPoly<T> make_device_poly(const KernelHost& h) {
    KernelPoly<T> kp;
    for (int i = 0; i < NUSHT_MAX_W; ++i)
        for (int d = 0; d <= NUSHT_MAX_DEG; ++d) kp.c[i][d] = (i < h.w && d <= h.deg) ? (T)h.c[i][d] : (T)0;
    return kp;
}

template <int W, typename T>
int launch_interp(const NufftParams& P, const KernelHost& h, const void* grid, void* map, cudaStream_t s) {
    const KernelPoly<T> kp = make_device_poly<T>(h);
    constexpr int NU_WARPS = nu_warps<W, T>();
    const int blocks = (P.n_items + NU_WARPS - 1) / NU_WARPS;
    k_interp<W, T><<<blocks, NU_WARPS * 32, 0, s>>>(P, kp, (const T*)grid, (T*)map);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}
template <int W, typename T>
int launch_spread(const NufftParams& P, const KernelHost& h, const void* map, void* grid, cudaStream_t s) {
    const KernelPoly<T> kp = make_device_poly<T>(h);
    constexpr int NU_WARPS = nu_warps<W, T>();
    const int blocks = (P.n_items + NU_WARPS - 1) / NU_WARPS;
    k_spread<W, T><<<blocks, NU_WARPS * 32, 0, s>>>(P, kp, (const T*)map, (T*)grid);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}

template <int W>
int launch_interp_gather(const NufftParams& P, const KernelHost& h, int64_t npts, const void* grid, void* map,
                         cudaStream_t s) {
    const KernelPoly<float> kp = make_device_poly<float>(h);
    const unsigned blocks = (unsigned)((npts + GATHER_THREADS - 1) / GATHER_THREADS);
    k_interp_gather<W><<<blocks, GATHER_THREADS, 0, s>>>(P, kp, npts, (const float*)grid, (float*)map);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}
int dispatch_interp_gather(int w, const NufftParams& P, const KernelHost& h, int64_t npts, const void* grid, void* map,
                           cudaStream_t s) {
    switch (w) {
#define NUSHT_CASE(WW) case WW: return launch_interp_gather<WW>(P, h, npts, grid, map, s);
        NUSHT_CASE(2) NUSHT_CASE(3) NUSHT_CASE(4) NUSHT_CASE(5) NUSHT_CASE(6) NUSHT_CASE(7) NUSHT_CASE(8)
#undef NUSHT_CASE
    }
    return NUSHT_ERR_UNSUPPORTED;
}

template <typename T>
int dispatch_interp(int w, const NufftParams& P, const KernelHost& h, const void* grid, void* map, cudaStream_t s) {
    switch (w) {
#define NUSHT_CASE(WW) case WW: return launch_interp<WW, T>(P, h, grid, map, s);
        NUSHT_CASE(2) NUSHT_CASE(3) NUSHT_CASE(4) NUSHT_CASE(5) NUSHT_CASE(6) NUSHT_CASE(7) NUSHT_CASE(8)
        NUSHT_CASE(9) NUSHT_CASE(10) NUSHT_CASE(11) NUSHT_CASE(12) NUSHT_CASE(13) NUSHT_CASE(14)
        NUSHT_CASE(15) NUSHT_CASE(16) NUSHT_CASE(17) NUSHT_CASE(18)
#undef NUSHT_CASE
    }
    return NUSHT_ERR_UNSUPPORTED;
}
template <typename T>
int dispatch_spread(int w, const NufftParams& P, const KernelHost& h, const void* map, void* grid, cudaStream_t s) {
    switch (w) {
#define NUSHT_CASE(WW) case WW: return launch_spread<WW, T>(P, h, map, grid, s);
        NUSHT_CASE(2) NUSHT_CASE(3) NUSHT_CASE(4) NUSHT_CASE(5) NUSHT_CASE(6) NUSHT_CASE(7) NUSHT_CASE(8)
        NUSHT_CASE(9) NUSHT_CASE(10) NUSHT_CASE(11) NUSHT_CASE(12) NUSHT_CASE(13) NUSHT_CASE(14)
        NUSHT_CASE(15) NUSHT_CASE(16) NUSHT_CASE(17) NUSHT_CASE(18)
#undef NUSHT_CASE
    }
    return NUSHT_ERR_UNSUPPORTED;
}

// =============================================================================================
// FP64 path: a7 / a8 on the FP64 tensor-core instruction (mma.sync m8n8k4 f64, SASS DMMA).
//
// Why: with the register-window scheme above every lane needs all W theta weights of every point,
// i.e. W*8 bytes x 32 lanes of shared-memory -> register traffic per point.  At W = 11 that is 11
// shared-memory wavefronts per point and the LSU data pipe (one wavefront per clock per SM)
// saturates (ncu: 73-90 % of peak, profiles/) long before the FP64 pipe does.  DMMA performs the
// broadcast inside the tensor core: each lane holds ONE element of the weight fragment, and one
// instruction does 256 FMA at the full FP64 rate of the SM (measured 37.1 TFLOP/s, same pipe as DFMA).
//
// Geometry.  A strip is 8*NT grid columns (NT n-tiles of 8), of which mb = 8*NT - W + 1 are
// footprint origins.  Lane = (g = lane/4, t = lane%4).  The row window has S = 4*KS slots
// (interp; KS k-steps) or S = 8*MT slots (spread; MT m-tiles), used circularly: grid row r lives
// in slot r mod S, so sliding the window never moves registers.  A tile is up to 8 (interp) or 4
// (spread) consecutive points of the row-sorted list whose origins a0 lie within S - W rows of the
// first one, so that every footprint of the tile is inside the S resident rows.
//   interp:  D[p][c] = sum_k A[p][k] B[k][c],  A[p][k] = th_p[(k - a0_p) mod S] (0 beyond W taps),
//            B[k][c] = window row in slot k at strip column c;  f_p = sum_c D[p][c] ph_p[c - b0_p].
//   spread:  C[k][c] += sum_p A[k][p] B[p][c], A[k][p] = x_p th_p[(k - a0_p) mod S],
//            B[p][c] = ph_p[c - b0_p];  finished rows are flushed with global atomics.
// Fragment layouts (PTX ISA, mma.m8n8k4.f64): A row = g, col = t; B row = t, col = g;
// C/D row = g, cols = 2t, 2t+1.  N-tile nt, column n  <->  strip column NT*n + nt, so that a lane's
// elements are contiguous columns: B lanes hold columns NT*g .. NT*g+NT-1, C/D lanes hold columns
// 2*NT*t .. 2*NT*t+2*NT-1.
// =============================================================================================
__device__ __forceinline__ void dmma_m8n8k4(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

__host__ __device__ constexpr int mma_nt(int w) { return w <= 8 ? 2 : (w <= 14 ? 3 : 4); }   // n-tiles per strip
__host__ __device__ constexpr int mma_ks(int w) { return w <= 6 ? 2 : (w <= 11 ? 3 : (w <= 14 ? 4 : 5)); }
__host__ __device__ constexpr int mma_mt(int w) { return w <= 6 ? 1 : (w <= 14 ? 2 : 3); }
// warps (work items) per CTA of the interpolation / spreading kernel: static shared memory stays below 48 KB
__host__ __device__ constexpr int mma_interp_warps(int w) { return w <= 11 ? 4 : 2; }
__host__ __device__ constexpr int mma_spread_warps(int w) { return w <= 14 ? 4 : 2; }
__host__ __device__ constexpr int mma_th_stride(int s) { return s <= 12 ? 12 : (s <= 16 ? 20 : 36); }  // = 4 or 12 mod 16

template <int W, int S>
struct MmaScratch {
    static constexpr int STH = mma_th_stride(S);
    static constexpr int SP = W | 1;
    double th[33][STH];   // per point: theta weights, zero-padded to S slots; row 32 stays zero (absent points)
    double ph[32][SP];    // per point: phi weights
    int oy[32];           // per point: strip column of the first footprint column
};

// lane `lane` evaluates the weights of its own point and publishes them; returns a0 of the point
template <int W, int S, bool SCALE>
__device__ __forceinline__ int mma_publish(MmaScratch<W, S>& ws, const KernelPoly<double>& kp, int lane, double X,
                                           double Y, double val, int c0) {
    const double a0d = ceil(X - 0.5 * W), b0d = ceil(Y - 0.5 * W);
    const double ut = 2.0 * ((a0d + 0.5 * W) - X) - 1.0;
    const double up = 2.0 * ((b0d + 0.5 * W) - Y) - 1.0;
    double k[W];
    eval_taps<W, double>(kp, ut, k);
#pragma unroll
    for (int i = 0; i < S; i += 2) {
        double2 v;
        v.x = (i < W) ? (SCALE ? val * k[i < W ? i : 0] : k[i < W ? i : 0]) : 0.0;
        v.y = (i + 1 < W) ? (SCALE ? val * k[i + 1 < W ? i + 1 : 0] : k[i + 1 < W ? i + 1 : 0]) : 0.0;
        *reinterpret_cast<double2*>(&ws.th[lane][i]) = v;
    }
    eval_taps<W, double>(kp, up, k);
#pragma unroll
    for (int i = 0; i < W; ++i) ws.ph[lane][i] = k[i];
    ws.oy[lane] = (int)b0d - c0;
    return (int)a0d;
}

// cp.async helpers (SASS LDGSTS): global -> shared without a register round trip, completion per thread
__device__ __forceinline__ void cp_async_8(void* dst_smem, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src)
                 : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

constexpr int NU_RING_ROWS = 16;   // rows of the strip staged ahead of the register window
constexpr int NU_RING_CHUNK = 8;   // rows staged per top-up

template <int NT, int RB>
struct StripRing {
    double rows[RB][8 * NT];             // row r of the strip lives in rows[(r + 48) % RB]
};

// ---------------------------------------------------------------------------------------------
// a7: type-2 interpolation, FP64 / DMMA
// Memory latency is taken off the critical path with cp.async: the strip's grid rows are staged
// 8-16 rows ahead of the register window into a per-warp shared-memory ring, and the coordinates of
// the next batch of 32 points are staged while the current batch is processed.
// ---------------------------------------------------------------------------------------------
template <int W>
__global__ void __launch_bounds__(32 * mma_interp_warps(W), mma_interp_warps(W) == 4 ? 6 : 1)
k_interp_mma(const __grid_constant__ NufftParams P, const __grid_constant__ KernelPoly<double> kp,
             const double* __restrict__ grid, double* __restrict__ map) {
    constexpr int NT = mma_nt(W), KS = mma_ks(W), S = 4 * KS, SPAN = S - W, OFF = 2 * S, NC = 8 * NT;
    // ring rows >= window slots S (a jump of the window loads S rows at once); 48 is a multiple of every RB
    constexpr int RB = S <= 12 ? 12 : (S <= 16 ? NU_RING_ROWS : 24), CH = S == 16 ? NU_RING_CHUNK : 4;
    static_assert(RB >= S && 48 % RB == 0, "staging ring too small for the register window");
    using WS = MmaScratch<W, S>;
    constexpr int NW = mma_interp_warps(W);
    __shared__ __align__(16) WS s_ws[NW];
    __shared__ __align__(16) StripRing<NT, RB> s_ring[NW];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int item = blockIdx.x * NW + warp;
    if (item >= P.n_items) return;
    const int start = P.item_off[item], end = P.item_off[item + 1];
    if (start >= end) return;
    WS& ws = s_ws[warp];
    StripRing<NT, RB>& ring = s_ring[warp];
    if (lane < WS::STH) ws.th[32][lane] = 0.0;
    const NufftGeom& g = P.g;
    const int strip = item % g.nstrip;
    const int c0 = strip * g.mb - g.fl;   // global column of strip column 0
    const int gq = lane >> 2, t = lane & 3;
    int cols_n, cols_m;                   // staging: lane < NC copies strip column `lane` of a row
    {
        int c = (c0 + min(lane, NC - 1)) % g.nph;
        if (c < 0) c += g.nph;
        cols_n = c;
        c += g.nph / 2;
        cols_m = (c >= g.nph) ? c - g.nph : c;
    }
    double win[KS][NT];                   // win[ks][nt]: row in slot 4 ks + t, strip column NT g + nt
#pragma unroll
    for (int ks = 0; ks < KS; ++ks)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) win[ks][nt] = 0.0;
    int loaded_hi = INT_MIN;              // rows [loaded_hi - S, loaded_hi) are in the register window
    int staged_hi = INT_MIN;              // cp.async issued for rows below staged_hi (those >= loaded_hi are in the ring)
    int landed_hi = INT_MIN;              // rows below landed_hi are known to have arrived

    const int r_limit = g.nth / 2 + 1 + S;   // no point touches a row >= r_limit (< 2 n_theta: grid_row is enough)
    auto stage_rows = [&](int r0, int r1) {
        r1 = min(r1, r_limit);
        int slot = (r0 + 48) % RB;
#pragma unroll 1
        for (int r = r0; r < r1; ++r) {
            const double* src;
            if ((unsigned)r <= (unsigned)(g.nth / 2)) {          // a stored row (all but the rows next to a pole)
                src = grid + ((int64_t)r * g.nph + cols_n);
            } else {
                bool mirror;
                const int64_t ro = grid_row(g, r, mirror);
                src = grid + ro + (mirror ? cols_m : cols_n);
            }
            if (lane < NC) cp_async_8(&ring.rows[slot][lane], src);
            slot = (slot + 1 == RB) ? 0 : slot + 1;
        }
    };
    int w_tq = 0, w_ks = 0, w_slot = 0;   // window bookkeeping of row loaded_hi: (r & 3, (r >> 2) % KS, ring slot)
    // coordinates of the next batch travel in registers (plain loads issued one batch ahead), so that the only
    // cp.async traffic is the row staging and no wait is needed at the top of a batch
    double Xn = 0.0, Yn = 0.0;
    int dn = 0;
    if (start + lane < end) {
        Xn = P.px[start + lane];
        Yn = P.py[start + lane];
        dn = P.perm[start + lane];
    }
    for (int batch = start; batch < end; batch += 32) {
        const int idx = batch + lane;
        const bool has = idx < end;
        const double X = has ? Xn : 0.0, Y = has ? Yn : 0.0;
        const int dst = has ? dn : 0;
        if (idx + 32 < end) {
            Xn = P.px[idx + 32];
            Yn = P.py[idx + 32];
            dn = P.perm[idx + 32];
        }
        const int a0 = mma_publish<W, S, false>(ws, kp, lane, X, Y, 1.0, c0);   // absent points: zero weight row (live)
        const int sp_own = (a0 + OFF) % S;      // window slot of the point's first row
        __syncwarp();
        const int npt = min(32, end - batch);
        int j0 = 0;
        while (j0 < npt) {
            // ---- tile: up to 8 consecutive points within SPAN rows of the first ----
            const int row0 = __shfl_sync(0xffffffffu, a0, j0);
            const unsigned fit = __ballot_sync(0xffffffffu, has && lane >= j0 && a0 - row0 <= SPAN);
            const int cnt = min(8, __popc(fit));
            const int need_hi = row0 + S;
            // ---- rows [row0, need_hi) must be in the register window; they come from the ring ----
            if (loaded_hi < need_hi) {
                if (staged_hi < need_hi) {          // first tile of the item, or the window outran the look-ahead
                    // Copies still in flight (rows [landed_hi, staged_hi)) must not target a ring slot that is staged
                    // again now: two asynchronous copies to one address may land in either order.  Row r and row
                    // r + RB share a slot, so that is the case as soon as the rows staged now reach landed_hi + RB
                    // (always, after a jump of the window past rows that were staged but never used).
                    if (landed_hi < staged_hi && need_hi - RB > landed_hi) {
                        cp_async_wait_all();
                        __syncwarp();
                        landed_hi = staged_hi;
                    }
                    stage_rows(max(staged_hi, row0), need_hi);
                    staged_hi = need_hi;
                }
                if (landed_hi < need_hi) {
                    cp_async_wait_all();
                    __syncwarp();
                    landed_hi = staged_hi;
                }
                // one row at a time: row r goes to slot 4 ks + (r & 3) of the circular register window, i.e. to the
                // lanes with t == (r & 3); static register indices + predicates only (a run-time index would put the
                // window in local memory)
                int r = max(loaded_hi, row0);
                if (r != loaded_hi) {               // jump: recompute the bookkeeping (OFF keeps the operands positive)
                    w_tq = (r + OFF) & 3;
                    w_ks = ((r + OFF) >> 2) % KS;
                    w_slot = (r + 48) % RB;
                }
#pragma unroll 1
                for (; r < need_hi; ++r) {
                    const double* src = &ring.rows[w_slot][NT * gq];
                    const bool mine = t == w_tq;
#pragma unroll
                    for (int ksi = 0; ksi < KS; ++ksi)
                        if (w_ks == ksi) {          // warp-uniform
                            if (mine) {
#pragma unroll
                                for (int nt = 0; nt < NT; ++nt) win[ksi][nt] = src[nt];
                            }
                        }
                    if (++w_tq == 4) {
                        w_tq = 0;
                        if (++w_ks == KS) w_ks = 0;
                    }
                    if (++w_slot == RB) w_slot = 0;
                }
                loaded_hi = need_hi;
                __syncwarp();                       // ring rows below loaded_hi may now be overwritten
            }
            // ---- keep the ring CH .. RB rows ahead of the window ----
            if (staged_hi + CH <= loaded_hi + RB) {
                stage_rows(staged_hi, staged_hi + CH);
                staged_hi += CH;
            }
            // ---- A fragments: theta weights of point j0 + g in circular slot order ----
            const int jp = min(j0 + gq, 31);
            const int sp = __shfl_sync(0xffffffffu, sp_own, jp);
            const bool live = gq < cnt;
            const double* thp = &ws.th[live ? jp : 32][0];      // row 32 is all zero
            double d[NT][2];
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) d[nt][0] = d[nt][1] = 0.0;
#pragma unroll
            for (int ks = 0; ks < KS; ++ks) {
                int i = 4 * ks + t - sp;
                if ((S & (S - 1)) == 0) i &= S - 1;
                else if (i < 0) i += S;
                const double a = thp[i];
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) dmma_m8n8k4(d[nt][0], d[nt][1], a, win[ks][nt]);
            }
            // ---- phi contraction: this lane holds strip columns 2 NT t .. 2 NT t + 2 NT - 1 of point g ----
            const int oy = ws.oy[jp];
            double sum = 0.0;
#pragma unroll
            for (int e = 0; e < 2; ++e)
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                    const unsigned ip = (unsigned)(NT * (2 * t + e) + nt - oy);
                    const double wgt = (ip < (unsigned)W) ? ws.ph[jp][ip] : 0.0;
                    sum = fma(d[nt][e], wgt, sum);
                }
            sum += __shfl_xor_sync(0xffffffffu, sum, 1);
            sum += __shfl_xor_sync(0xffffffffu, sum, 2);
            const int dstp = __shfl_sync(0xffffffffu, dst, jp);   // caller index of point j0 + g
            if (t == 0 && live) map[dstp] = sum;
            j0 += cnt;
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------
// a8: type-1 spreading, FP64 / DMMA (grid must be zero on entry)
// ---------------------------------------------------------------------------------------------
template <int W>
__global__ void __launch_bounds__(32 * mma_spread_warps(W))
k_spread_mma(const __grid_constant__ NufftParams P, const __grid_constant__ KernelPoly<double> kp,
             const double* __restrict__ map, double* __restrict__ grid) {
    constexpr int NT = mma_nt(W), MT = mma_mt(W), S = 8 * MT, SPAN = S - W, OFF = 2 * S, NW = mma_spread_warps(W);
    using WS = MmaScratch<W, S>;
    __shared__ __align__(16) WS s_ws[NW];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int item = blockIdx.x * NW + warp;
    if (item >= P.n_items) return;
    const int start = P.item_off[item], end = P.item_off[item + 1];
    if (start >= end) return;
    WS& ws = s_ws[warp];
    if (lane < WS::STH) ws.th[32][lane] = 0.0;
    const NufftGeom& g = P.g;
    const int strip = item % g.nstrip;
    const int c0 = strip * g.mb - g.fl;
    const int gq = lane >> 2, t = lane & 3;
    int colc_n[2 * NT], colc_m[2 * NT];   // global columns of this lane's accumulator elements
#pragma unroll
    for (int q = 0; q < 2 * NT; ++q) {
        // accumulator element (nt, e) sits at strip column NT (2t + e) + nt; q = NT e + nt
        int c = (c0 + 2 * NT * t + q) % g.nph;
        if (c < 0) c += g.nph;
        colc_n[q] = c;
        c += g.nph / 2;
        colc_m[q] = (c >= g.nph) ? c - g.nph : c;
    }
    double acc[MT][NT][2];                // acc[mt][nt][e]: slot 8 mt + g, strip column NT (2t+e) + nt
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;
    int a_lo = INT_MIN;                   // slots hold rows [a_lo, a_lo + S)

    // flush rows r0 .. r0 + n - 1 (n <= 8: one row per value of g) to the grid and clear their slots
    auto flush_group = [&](int r0, int n) {
        const int s0 = (r0 + OFF) % S;
        const int i = (gq - s0) & 7;      // slot s0 + i is the one of this group with (slot & 7) == g
        const bool rowhit = i < n;
        int s = s0 + i;
        if (s >= S) s -= S;
        bool mirror;
        const int64_t ro = grid_row(g, r0 + i, mirror);
        // static indices + predicates only: a run-time index into acc would put it in local memory
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
            const bool hit = rowhit && (mt == (s >> 3));
#pragma unroll
            for (int e = 0; e < 2; ++e)
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                    const double v = acc[mt][nt][e];
                    const int q = NT * e + nt;
                    if (hit && v != 0.0) atomicAdd(&grid[ro + (mirror ? colc_m[q] : colc_n[q])], v);
                    acc[mt][nt][e] = hit ? 0.0 : v;
                }
        }
    };
    constexpr int FG = SPAN >= 4 ? 4 : (SPAN >= 2 ? 2 : 1);   // rows flushed together
    // The window base a_lo is kept a multiple of FG, so the FG rows of a regular flush sit in ONE group of 8
    // slots: the m-tile is warp-uniform and only its 2 NT accumulators are touched.
    auto flush_aligned = [&](int r0) {
        const int s0 = (r0 + OFF) % S;    // multiple of FG
        const int i = (gq - s0) & 7;
        const bool rowhit = i < FG;
        bool mirror;
        const int64_t ro = grid_row(g, r0 + i, mirror);
        auto body = [&](auto mtc) {       // compile-time m-tile: static register indices only
            constexpr int mt = decltype(mtc)::value;
#pragma unroll
            for (int e = 0; e < 2; ++e)
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                    const double v = acc[mt][nt][e];
                    const int q = NT * e + nt;
                    if (rowhit && v != 0.0) atomicAdd(&grid[ro + (mirror ? colc_m[q] : colc_n[q])], v);
                    acc[mt][nt][e] = rowhit ? 0.0 : v;
                }
        };
        const int mtu = s0 >> 3;          // warp-uniform
        if (MT == 1 || mtu == 0) body(std::integral_constant<int, 0>{});
        else if (MT == 2 || mtu == 1) body(std::integral_constant<int, MT >= 2 ? 1 : 0>{});
        else body(std::integral_constant<int, MT >= 3 ? 2 : 0>{});
    };
    // coordinates and value one batch ahead, the caller index of the value two batches ahead: map[perm[.]] is a
    // dependent load, issued with the index still in flight it stalls the warp for a DRAM round trip
    double Xn = 0.0, Yn = 0.0, vn = 0.0;
    int pn = 0;
    if (start + lane < end) {
        Xn = P.px[start + lane];
        Yn = P.py[start + lane];
        vn = map[P.perm[start + lane]];
    }
    if (start + 32 + lane < end) pn = P.perm[start + 32 + lane];
    for (int batch = start; batch < end; batch += 32) {
        const int idx = batch + lane;
        const bool has = idx < end;
        const double X = Xn, Y = Yn, val = has ? vn : 0.0;
        if (idx + 32 < end) {
            Xn = P.px[idx + 32];
            Yn = P.py[idx + 32];
            vn = map[pn];
        }
        if (idx + 64 < end) pn = P.perm[idx + 64];
        // the point's value rides on the theta weights
        const int a0 = mma_publish<W, S, true>(ws, kp, lane, X, Y, val, c0);
        __syncwarp();
        const int npt = min(32, end - batch);
        int j0 = 0;
        while (j0 < npt) {
            // ---- tile: up to 8 consecutive points whose origins lie within SPAN rows of the window base ----
            const int row0 = __shfl_sync(0xffffffffu, a0, j0);
            // ---- rows below row0 are complete: flush them FG at a time (slots hold [a_lo, a_lo + S)) ----
            if (a_lo == INT_MIN) a_lo = row0 & ~(FG - 1);
            if (row0 - a_lo >= S) {
#pragma unroll 1
                for (int k = 0; k < S; k += 8) flush_group(a_lo + k, 8);
                a_lo = row0 & ~(FG - 1);
            }
#pragma unroll 1
            while (row0 - a_lo >= FG) {
                flush_aligned(a_lo);
                a_lo += FG;
            }
            const unsigned fit = __ballot_sync(0xffffffffu, has && lane >= j0 && a0 - a_lo <= SPAN);
            const int cnt = min(8, __popc(fit));
            // ---- two k-steps of 4 points each; fragments A[slot][point t], B[point t][column], point = j0 + 4 kk + t ----
#pragma unroll
            for (int kk = 0; kk < 2; ++kk) {
                if (4 * kk >= cnt) break;                          // warp-uniform
                const int jp = min(j0 + 4 * kk + t, 31);
                const int a0p = __shfl_sync(0xffffffffu, a0, jp);
                const int sp = (a0p + OFF) % S;
                const int oy = ws.oy[jp];
                const bool live = 4 * kk + t < cnt;
                const double* thp = &ws.th[live ? jp : 32][0];      // row 32 is all zero
                double a[MT], b[NT];
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    int i = 8 * mt + gq - sp;
                    if ((S & (S - 1)) == 0) i &= S - 1;
                    else if (i < 0) i += S;
                    a[mt] = thp[i];
                }
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                    const unsigned ip = (unsigned)(NT * gq + nt - oy);
                    b[nt] = (ip < (unsigned)W) ? ws.ph[jp][ip] : 0.0;
                }
#pragma unroll
                for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                    for (int nt = 0; nt < NT; ++nt) dmma_m8n8k4(acc[mt][nt][0], acc[mt][nt][1], a[mt], b[nt]);
            }
            j0 += cnt;
        }
        __syncwarp();
    }
    if (a_lo != INT_MIN) {
#pragma unroll 1
        for (int k = 0; k < S; k += 8) flush_group(a_lo + k, 8);
    }
}

template <int W>
int launch_interp_mma(const NufftParams& P, const KernelHost& h, const void* grid, void* map, cudaStream_t s) {
    const KernelPoly<double> kp = make_device_poly<double>(h);
    constexpr int NW = mma_interp_warps(W);
    k_interp_mma<W><<<(P.n_items + NW - 1) / NW, 32 * NW, 0, s>>>(P, kp, (const double*)grid, (double*)map);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}
template <int W>
int launch_spread_mma(const NufftParams& P, const KernelHost& h, const void* map, void* grid, cudaStream_t s) {
    const KernelPoly<double> kp = make_device_poly<double>(h);
    constexpr int NW = mma_spread_warps(W);
    k_spread_mma<W><<<(P.n_items + NW - 1) / NW, 32 * NW, 0, s>>>(P, kp, (const double*)map, (double*)grid);
    NUSHT_CUDA_TRY(nusht_launched());
    return NUSHT_OK;
}

int dispatch_interp_mma(int w, const NufftParams& P, const KernelHost& h, const void* grid, void* map, cudaStream_t s) {
    switch (w) {
#define NUSHT_CASE(WW) case WW: return launch_interp_mma<WW>(P, h, grid, map, s);
        NUSHT_CASE(2) NUSHT_CASE(3) NUSHT_CASE(4) NUSHT_CASE(5) NUSHT_CASE(6) NUSHT_CASE(7) NUSHT_CASE(8)
        NUSHT_CASE(9) NUSHT_CASE(10) NUSHT_CASE(11) NUSHT_CASE(12) NUSHT_CASE(13) NUSHT_CASE(14)   // sigma = 2: eps >= 1e-13 -> w <= 14
        NUSHT_CASE(15) NUSHT_CASE(16) NUSHT_CASE(17) NUSHT_CASE(18)                                // sigma = 1.25: eps >= 1e-10 -> w <= 17
#undef NUSHT_CASE
    }
    return NUSHT_ERR_UNSUPPORTED;
}
int dispatch_spread_mma(int w, const NufftParams& P, const KernelHost& h, const void* map, void* grid, cudaStream_t s) {
    switch (w) {
#define NUSHT_CASE(WW) case WW: return launch_spread_mma<WW>(P, h, map, grid, s);
        NUSHT_CASE(2) NUSHT_CASE(3) NUSHT_CASE(4) NUSHT_CASE(5) NUSHT_CASE(6) NUSHT_CASE(7) NUSHT_CASE(8)
        NUSHT_CASE(9) NUSHT_CASE(10) NUSHT_CASE(11) NUSHT_CASE(12) NUSHT_CASE(13) NUSHT_CASE(14)   // sigma = 2: eps >= 1e-13 -> w <= 14
        NUSHT_CASE(15) NUSHT_CASE(16) NUSHT_CASE(17) NUSHT_CASE(18)                                // sigma = 1.25: eps >= 1e-10 -> w <= 17
#undef NUSHT_CASE
    }
    return NUSHT_ERR_UNSUPPORTED;
}

// ---- host: Gauss-Legendre nodes (Newton on P_n), extended precision ----
void gauss_legendre(int n, std::vector<long double>& x, std::vector<long double>& wt) {
    const long double PI_L = 3.14159265358979323846264338327950288L;
    x.resize(n);
    wt.resize(n);
    for (int i = 0; i < n; ++i) {
        long double z = cosl(PI_L * (i + 0.75L) / (n + 0.5L));
        long double dp = 0;
        for (int it = 0; it < 100; ++it) {
            long double p0 = 1, p1 = z;
            for (int k = 2; k <= n; ++k) {
                long double p2 = ((2 * k - 1) * z * p1 - (k - 1) * p0) / k;
                p0 = p1;
                p1 = p2;
            }
            dp = n * (z * p1 - p0) / (z * z - 1);
            long double dz = p1 / dp;
            z -= dz;
            if (fabsl(dz) < 1e-19L) break;
        }
        x[i] = z;
        wt[i] = 2 / ((1 - z * z) * dp * dp);
    }
}

}  // namespace

// the host model of the kernel (extended-precision polynomial coefficients) hangs off the plan
static KernelHost* g_kernel_of(const nusht_plan_s* p) { return static_cast<KernelHost*>(p->kernel_host); }

int nufft_choose_kernel(nusht_plan_s* p) {
    // width / shape rule of the ES kernel (reading G8, the published rule of the paper's ref. [38]):
    // up-sampling 2:      w = ceil(log10(1/eps)) + 1,               beta = 2.30 w
    // other up-sampling:  w = ceil(-ln eps / (pi sqrt(1 - 1/sigma))), beta = 0.97 pi w (1 - 1/(2 sigma))
    int w;
    double bw;
    if (p->sigma == 2.0) {
        w = (int)ceil(log10(1.0 / p->eps)) + 1;
        if (w < 2) w = 2;
        bw = 2.30;
        if (w == 2) bw = 2.20;
        if (w == 3) bw = 2.26;
        if (w == 4) bw = 2.38;
    } else {
        const double PI_D = 3.14159265358979323846;
        w = (int)ceil(-log(p->eps) / (PI_D * sqrt(1.0 - 1.0 / p->sigma)));
        if (w < 2) w = 2;
        bw = 0.97 * PI_D * (1.0 - 0.5 / p->sigma);
    }
    if (w > NUSHT_MAX_W) return NUSHT_ERR_INVALID_ARG;
    KernelHost* h = new KernelHost();
    h->w = w;
    h->deg = poly_degree(w);
    h->beta = bw * w;
    p->beta = h->beta;
    p->ng.w = w;
    p->ng.fl = w / 2;
    p->ng.deg = h->deg;
    // strip width in footprint-origin columns: FP64 runs on the DMMA kernels (8 NT columns per strip),
    // FP32 on the register-window kernels (32 columns per strip)
    p->ng.mb = (p->dtype == NUSHT_F64) ? 8 * mma_nt(w) - w + 1 : 33 - w;
    // Chebyshev interpolation of tap i on u in [-1,1]:  z = (u + 1 - w + 2 i)/w
    const long double PI_L = 3.14159265358979323846264338327950288L;
    const int d = h->deg, nn = d + 1;
    std::vector<long double> un(nn), f(nn), cheb(nn);
    for (int k = 0; k < nn; ++k) un[k] = cosl(PI_L * (k + 0.5L) / nn);
    for (int i = 0; i < w; ++i) {
        for (int k = 0; k < nn; ++k) {
            long double z = (un[k] + 1 - w + 2 * i) / w;
            long double a = 1 - z * z;
            if (a < 0) a = 0;
            f[k] = expl((long double)h->beta * (sqrtl(a) - 1));
        }
        for (int j = 0; j < nn; ++j) {
            long double s = 0;
            for (int k = 0; k < nn; ++k) s += f[k] * cosl(PI_L * j * (k + 0.5L) / nn);
            cheb[j] = (j == 0 ? 1.0L : 2.0L) * s / nn;
        }
        // Chebyshev -> monomial: T_0 = 1, T_1 = u, T_{j+1} = 2 u T_j - T_{j-1}
        std::vector<long double> t0(nn, 0.0L), t1(nn, 0.0L), t2(nn, 0.0L), mono(nn, 0.0L);
        t0[0] = 1;
        for (int q = 0; q < nn; ++q) mono[q] += cheb[0] * t0[q];
        if (nn > 1) {
            t1[1] = 1;
            for (int q = 0; q < nn; ++q) mono[q] += cheb[1] * t1[q];
        }
        for (int j = 2; j < nn; ++j) {
            for (int q = 0; q < nn; ++q) t2[q] = (q > 0 ? 2 * t1[q - 1] : 0.0L) - t0[q];
            for (int q = 0; q < nn; ++q) mono[q] += cheb[j] * t2[q];
            t0 = t1;
            t1 = t2;
        }
        for (int q = 0; q <= NUSHT_MAX_DEG; ++q) h->c[i][q] = (q < nn) ? mono[q] : 0.0L;
    }
    // the kernel is even: make tap w-1-i exactly tap i mirrored (the fit gives this up to rounding),
    // which is what eval_taps relies on; the deconvolution factors use these same coefficients
    for (int i = 0; i < w / 2; ++i)
        for (int q = 0; q <= NUSHT_MAX_DEG; ++q) {
            const long double sgn = (q & 1) ? -1.0L : 1.0L;
            const long double v = 0.5L * (h->c[i][q] + sgn * h->c[w - 1 - i][q]);
            h->c[i][q] = v;
            h->c[w - 1 - i][q] = sgn * v;
        }
    if (w & 1)
        for (int q = 1; q <= NUSHT_MAX_DEG; q += 2) h->c[w / 2][q] = 0.0L;
    p->kernel_host = h;
    return NUSHT_OK;
}

// Fourier transform of the piecewise-polynomial kernel on a grid of n cells:
//   psihat(k) = int psi(x) cos(2 pi k x/n) dx,  x = xi - w/2 + i on tap interval i, xi in [0,1)
double nufft_kernel_ft(const nusht_plan_s* p, double k, int n) {
    const KernelHost* h = g_kernel_of(p);
    static std::vector<long double> xg, wg;
    static std::once_flag once;
    std::call_once(once, [] { gauss_legendre(32, xg, wg); });
    const long double PI_L = 3.14159265358979323846264338327950288L;
    long double tot = 0;
    for (int i = 0; i < h->w; ++i) {
        for (size_t q = 0; q < xg.size(); ++q) {
            const long double u = xg[q];
            long double v = h->c[i][h->deg];
            for (int d = h->deg - 1; d >= 0; --d) v = v * u + h->c[i][d];
            const long double x = 0.5L * (u + 1) - 0.5L * h->w + i;
            tot += 0.5L * wg[q] * v * cosl(2 * PI_L * (long double)k * x / n);
        }
    }
    return (double)tot;
}

template <typename T>
static int nu_alloc(T** ptr, size_t count, nusht_plan_s* p) {
    size_t bytes = count * sizeof(T);
    if (bytes == 0) bytes = sizeof(T);
    NUSHT_CUDA_TRY(cudaMalloc((void**)ptr, bytes));
    p->workspace_bytes += (int64_t)bytes;
    return NUSHT_OK;
}

// the point tables are accounted for separately, so that nusht_set_points can replace them
static int sort_points_impl(nusht_plan_s* p, const double* theta, const double* phi);
int nufft_sort_points(nusht_plan_s* p, const double* theta, const double* phi) {
    const int64_t before = p->workspace_bytes;
    const int st = sort_points_impl(p, theta, phi);
    p->points_bytes += p->workspace_bytes - before;
    return st;
}

static int sort_points_impl(nusht_plan_s* p, const double* theta, const double* phi) {
    NufftGeom& g = p->ng;
    g.nstrip = (g.nph + 1 + g.mb - 1) / g.mb;   // origins cb = 0..nph inclusive
    g.nseg = (g.nth / 2 + 2 + NUSHT_SEG_ROWS - 1) / NUSHT_SEG_ROWS;
    g.inv_hth = (double)g.nth / TWO_PI;
    g.inv_hph = (double)g.nph / TWO_PI;
    p->n_items = g.nseg * g.nstrip;
    const int64_t nbins64 = (int64_t)p->n_items * NUSHT_SEG_ROWS;
    if (nbins64 + 1 >= (int64_t)1 << 31) return NUSHT_ERR_UNSUPPORTED;
    const int nbins = (int)nbins64;
    const int64_t n = p->npts;
    if (!p->d_px) {     // (nusht_set_points with an unchanged point count keeps the tables and overwrites them)
        NUSHT_TRY(nu_alloc(&p->d_px, (size_t)n, p));
        NUSHT_TRY(nu_alloc(&p->d_py, (size_t)n, p));
        NUSHT_TRY(nu_alloc(&p->d_perm, (size_t)n, p));
        NUSHT_TRY(nu_alloc(&p->d_item_off, (size_t)p->n_items + 1, p));
    }

    SortGeom sg;
    sg.nth = g.nth; sg.nph = g.nph; sg.w = g.w; sg.fl = g.fl; sg.mb = g.mb; sg.nstrip = g.nstrip; sg.nseg = g.nseg;
    sg.inv_hth = g.inv_hth; sg.inv_hph = g.inv_hph; sg.half_w = 0.5 * g.w;

    int *d_keys = nullptr, *d_ranks = nullptr, *d_hist = nullptr, *d_off = nullptr, *d_tot = nullptr, *d_bad = nullptr;
    PointRec* d_rec = nullptr;
    cudaEvent_t ev_sort[2] = {nullptr, nullptr};
    const int ntiles = (nbins + 1 + SCAN_TILE - 1) / SCAN_TILE;
    int status = NUSHT_OK;
    auto cleanup = [&]() {
        cudaFree(d_keys); cudaFree(d_ranks); cudaFree(d_hist); cudaFree(d_off); cudaFree(d_tot); cudaFree(d_bad);
        cudaFree(d_rec);
        d_rec = nullptr;
        d_ranks = nullptr;
        if (ev_sort[0]) cudaEventDestroy(ev_sort[0]);
        if (ev_sort[1]) cudaEventDestroy(ev_sort[1]);
        ev_sort[0] = ev_sort[1] = nullptr;
    };
#define SORT_TRY(expr)                                                              \
    do {                                                                            \
        cudaError_t _e = (expr);                                                    \
        if (_e != cudaSuccess) {                                                    \
            nusht_note_cuda_error(_e, #expr, __FILE__, __LINE__);                   \
            cleanup();                                                              \
            return (_e == cudaErrorMemoryAllocation) ? NUSHT_ERR_ALLOC : NUSHT_ERR_CUDA; \
        }                                                                           \
    } while (0)
    SORT_TRY(cudaMalloc((void**)&d_keys, sizeof(int) * (size_t)(n > 0 ? n : 1)));
    SORT_TRY(cudaMalloc((void**)&d_ranks, sizeof(int) * (size_t)(n > 0 ? n : 1)));
    SORT_TRY(cudaMalloc((void**)&d_hist, sizeof(int) * ((size_t)nbins + 1)));
    SORT_TRY(cudaMalloc((void**)&d_off, sizeof(int) * ((size_t)nbins + 1)));
    SORT_TRY(cudaMalloc((void**)&d_tot, sizeof(int) * (size_t)ntiles));
    SORT_TRY(cudaMalloc((void**)&d_bad, sizeof(int)));
    SORT_TRY(cudaMalloc((void**)&d_rec, sizeof(PointRec) * (size_t)(n > 0 ? n : 1)));   // plan-time scratch, freed below
    SORT_TRY(cudaMemset(d_hist, 0, sizeof(int) * ((size_t)nbins + 1)));
    SORT_TRY(cudaMemset(d_bad, 0, sizeof(int)));
    SORT_TRY(cudaEventCreate(&ev_sort[0]));
    SORT_TRY(cudaEventCreate(&ev_sort[1]));
    SORT_TRY(cudaEventRecord(ev_sort[0], 0));
    if (n > 0) {
        const int threads = 256;
        const unsigned blocks = (unsigned)((n + threads - 1) / threads);
        k_point_keys<<<blocks, threads>>>(sg, n, theta, phi, d_keys, d_ranks, d_hist, d_bad);
        SORT_TRY(nusht_launched());
    }
    k_scan_tiles<<<ntiles, SCAN_BLOCK>>>(d_hist, d_off, d_tot, nbins + 1);
    SORT_TRY(nusht_launched());
    k_scan_totals<<<1, 1024>>>(d_tot, ntiles);
    SORT_TRY(nusht_launched());
    k_scan_add<<<ntiles, SCAN_BLOCK>>>(d_off, d_tot, nbins + 1);
    SORT_TRY(nusht_launched());
    k_item_offsets<<<(p->n_items + 1 + 255) / 256, 256>>>(d_off, p->d_item_off, p->n_items, (int)n);
    SORT_TRY(nusht_launched());
    if (n > 0) {
        const int threads = 256;
        const unsigned blocks = (unsigned)((n + threads - 1) / threads);
        k_point_scatter<<<blocks, threads>>>(sg, n, theta, phi, d_keys, d_ranks, d_off, d_rec);
        SORT_TRY(nusht_launched());
        k_point_unpack<<<blocks, threads>>>(n, d_rec, p->d_px, p->d_py, p->d_perm);
        SORT_TRY(nusht_launched());
    }
    SORT_TRY(cudaEventRecord(ev_sort[1], 0));
    SORT_TRY(cudaDeviceSynchronize());
    {
        float ms = 0.f;
        SORT_TRY(cudaEventElapsedTime(&ms, ev_sort[0], ev_sort[1]));
        p->sort_ms = ms;
        // the bad-point counter is read once everything is enqueued and done (a rejected point took key 0, rank 0:
        // harmless, the plan is discarded)
        int bad = 0;
        SORT_TRY(cudaMemcpy(&bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost));
        if (bad != 0) {
            cleanup();
            return NUSHT_ERR_BAD_POINTS;
        }
    }
    cleanup();
    d_keys = d_ranks = d_hist = d_off = d_tot = d_bad = nullptr;
    // L2-blocked un-permutation tables (FP32 gather interpolation; see k_unpermute)
    p->n_buckets = 1;
    int bshift = BUCKET_SHIFT;
    while (((n + ((int64_t)1 << bshift) - 1) >> bshift) > BUCKET_MAX) ++bshift;
    if (const char* ev = getenv("NUSHT_UNPERMUTE_SHIFT")) {      // tests: several buckets at small point counts
        const int v = atoi(ev);
        if (v >= 4 && v <= 30) bshift = v;
    }
    const int64_t nb64 = (n + ((int64_t)1 << bshift) - 1) >> bshift;
    if (p->dtype == NUSHT_F32 && g.w <= 8 && nb64 > 1 && nb64 <= BUCKET_MAX) {
        const int nb = (int)nb64;
        const int nchunks = (int)((n + BUCKET_CHUNK - 1) / BUCKET_CHUNK);
        const int ncnt = BUCKET_MAX * nchunks;
        const int nt = (ncnt + SCAN_TILE - 1) / SCAN_TILE;
        if (!p->d_slot) {
            NUSHT_TRY(nu_alloc(&p->d_slot, (size_t)n, p));
            NUSHT_TRY(nu_alloc(&p->d_dest, (size_t)n, p));
            float* stage = nullptr;
            NUSHT_TRY(nu_alloc(&stage, (size_t)n, p));
            p->d_stage = stage;
        }
        SORT_TRY(cudaMalloc((void**)&d_hist, sizeof(int) * (size_t)ncnt));
        SORT_TRY(cudaMalloc((void**)&d_off, sizeof(int) * (size_t)ncnt));
        SORT_TRY(cudaMalloc((void**)&d_tot, sizeof(int) * (size_t)nt));
        const int blocks = (nchunks + BUCKET_WARPS - 1) / BUCKET_WARPS;
        k_bucket_count<<<blocks, 32 * BUCKET_WARPS>>>(p->d_perm, n, bshift, nchunks, d_hist);
        SORT_TRY(nusht_launched());
        k_scan_tiles<<<nt, SCAN_BLOCK>>>(d_hist, d_off, d_tot, ncnt);
        SORT_TRY(nusht_launched());
        k_scan_totals<<<1, 1024>>>(d_tot, nt);
        SORT_TRY(nusht_launched());
        k_scan_add<<<nt, SCAN_BLOCK>>>(d_off, d_tot, ncnt);
        SORT_TRY(nusht_launched());
        k_bucket_place<<<blocks, 32 * BUCKET_WARPS>>>(p->d_perm, n, bshift, nchunks, d_off, p->d_slot, p->d_dest);
        SORT_TRY(nusht_launched());
        SORT_TRY(cudaDeviceSynchronize());
        cleanup();
        p->n_buckets = nb;
    }
#undef SORT_TRY
    return status;
}

static NufftParams make_nufft_params(const nusht_plan_s* p) {
    NufftParams P;
    P.g = p->ng;
    P.px = p->d_px;
    P.py = p->d_py;
    P.perm = p->d_perm;
    P.item_off = p->d_item_off;
    P.n_items = p->n_items;
    return P;
}

int nufft_interp(nusht_plan_s* p, const void* grid, void* map, cudaStream_t s) {
    if (p->npts == 0) return NUSHT_OK;
    const KernelHost* h = g_kernel_of(p);
    const NufftParams P = make_nufft_params(p);
    if (p->dtype == NUSHT_F64) return dispatch_interp_mma(p->ng.w, P, *h, grid, map, s);
    // FP32: thread-per-point gather up to W = 8 (eps >= 1e-7); NUSHT_INTERP_F32=window keeps the register-window
    // kernel for the tests, which compare the two
    const char* ev = getenv("NUSHT_INTERP_F32");
    const bool window = ev && strcmp(ev, "window") == 0;
    if (p->ng.w <= 8 && !window) {
        if (p->n_buckets <= 1) return dispatch_interp_gather(p->ng.w, P, *h, p->npts, grid, map, s);
        NufftParams Q = P;
        Q.perm = p->d_slot;       // results go to their bucket-major slot, then to the caller's order
        NUSHT_TRY(dispatch_interp_gather(p->ng.w, Q, *h, p->npts, grid, p->d_stage, s));
        k_unpermute<float><<<(unsigned)((p->npts + 255) / 256), 256, 0, s>>>((const float*)p->d_stage, p->d_dest,
                                                                           p->npts, (float*)map);
        NUSHT_CUDA_TRY(nusht_launched());
        return NUSHT_OK;
    }
    return dispatch_interp<float>(p->ng.w, P, *h, grid, map, s);
}

int nufft_spread(nusht_plan_s* p, const void* map, void* grid, cudaStream_t s) {
    const size_t esz = (p->dtype == NUSHT_F64) ? 8 : 4;
    NUSHT_CUDA_TRY(cudaMemsetAsync(grid, 0, (size_t)p->ng.nrow_half * (size_t)p->ng.nph * esz, s));
    if (p->npts == 0) return NUSHT_OK;
    const KernelHost* h = g_kernel_of(p);
    const NufftParams P = make_nufft_params(p);
    if (p->dtype == NUSHT_F64) return dispatch_spread_mma(p->ng.w, P, *h, map, grid, s);
    return dispatch_spread<float>(p->ng.w, P, *h, map, grid, s);
}

void nufft_free_points(nusht_plan_s* p) {
    cudaFree(p->d_px); cudaFree(p->d_py); cudaFree(p->d_perm); cudaFree(p->d_item_off);
    p->d_px = p->d_py = nullptr; p->d_perm = nullptr; p->d_item_off = nullptr;
    cudaFree(p->d_slot); cudaFree(p->d_dest); cudaFree(p->d_stage);
    p->d_slot = p->d_dest = nullptr; p->d_stage = nullptr;
    p->n_buckets = 1;
    p->workspace_bytes -= p->points_bytes;
    p->points_bytes = 0;
}

void nufft_free(nusht_plan_s* p) {
    nufft_free_points(p);
    delete static_cast<KernelHost*>(p->kernel_host);
    p->kernel_host = nullptr;
}
