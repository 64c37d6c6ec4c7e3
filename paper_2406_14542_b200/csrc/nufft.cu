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
                             const double* __restrict__ phi, int* __restrict__ keys, int* __restrict__ hist,
                             int* __restrict__ bad) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npts) return;
    double X, Y;
    int ra, cb;
    if (!point_coords(g, theta[i], phi[i], X, Y, ra, cb)) {
        atomicAdd(bad, 1);
        keys[i] = 0;
        return;
    }
    const int seg = ra / NUSHT_SEG_ROWS, strip = cb / g.mb;
    const int key = (seg * g.nstrip + strip) * NUSHT_SEG_ROWS + (ra - seg * NUSHT_SEG_ROWS);
    keys[i] = key;
    atomicAdd(&hist[key], 1);
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

__global__ void k_item_offsets(const int* __restrict__ bin_off, int* __restrict__ item_off, int n_items,
                               int npts) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_items) item_off[i] = bin_off[(int64_t)i * NUSHT_SEG_ROWS];
    if (i == n_items) item_off[i] = npts;
}

__global__ void k_point_scatter(SortGeom g, int64_t npts, const double* __restrict__ theta,
                                const double* __restrict__ phi, const int* __restrict__ keys,
                                int* __restrict__ cursor, double* __restrict__ px, double* __restrict__ py,
                                int* __restrict__ perm) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npts) return;
    double X, Y;
    int ra, cb;
    point_coords(g, theta[i], phi[i], X, Y, ra, cb);
    const int pos = atomicAdd(&cursor[keys[i]], 1);
    px[pos] = X;
    py[pos] = Y;
    perm[pos] = (int)i;
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
    int2 org[32];       // per point: (a0, lane of first footprint column)
};

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

    for (int batch = start; batch < end; batch += 32) {
        const int idx = batch + lane;
        const bool has = idx < end;
        // ---- each lane evaluates the 2W weights of its own point ----
        {
            const double X = has ? P.px[idx] : 0.0, Y = has ? P.py[idx] : 0.0;
            const double a0d = ceil(X - 0.5 * W), b0d = ceil(Y - 0.5 * W);
            const T ut = (T)(2.0 * ((a0d + 0.5 * W) - X) - 1.0);
            const T up = (T)(2.0 * ((b0d + 0.5 * W) - Y) - 1.0);
            T k[W];
            eval_taps<W, T>(kp, ut, k);
            if constexpr (sizeof(T) == 8) {
#pragma unroll
                for (int i = 0; i + 1 < W; i += 2)
                    *reinterpret_cast<double2*>(&ws.th[lane][i]) = make_double2(k[i], k[i + 1]);
                if (W & 1) *reinterpret_cast<double2*>(&ws.th[lane][W - 1]) = make_double2(k[W - 1], 0.0);
            } else {
#pragma unroll
                for (int i = 0; i < W; ++i) ws.th[lane][i] = k[i];
            }
            eval_taps<W, T>(kp, up, k);
#pragma unroll
            for (int i = 0; i < W; ++i) ws.ph[lane][i] = k[i];
            ws.org[lane] = make_int2((int)a0d, (int)b0d - c0);
        }
        __syncwarp();
        const int npt = min(32, end - batch);
        int j = 0;
        int2 org = ws.org[0];
        while (j < npt) {
            // ---- slide the register window down to row org.x (warp-uniform) ----
            if (org.x != a_base) {
                int d = (a_base == INT_MIN) ? W : org.x - a_base;
                if (d >= W) {
                    a_base = org.x;
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
            // ---- all points of the batch whose footprint starts on this row: the window is
            //      loop-invariant here, so it stays in place in registers ----
#pragma unroll 1
            do {
                // theta contraction in registers (two independent chains), phi weight per lane
                T acc0 = 0, acc1 = 0;
                if constexpr (sizeof(T) == 8) {
#pragma unroll
                    for (int i = 0; i + 1 < W; i += 2) {
                        const double2 kk = *reinterpret_cast<const double2*>(&ws.th[j][i]);
                        acc0 = fma(kk.x, win[i], acc0);
                        acc1 = fma(kk.y, win[i + 1], acc1);
                    }
                    if (W & 1) acc0 = fma(ws.th[j][W - 1], win[W - 1], acc0);
                } else {
#pragma unroll
                    for (int i = 0; i + 1 < W; i += 2) {
                        acc0 = fma(ws.th[j][i], win[i], acc0);
                        acc1 = fma(ws.th[j][i + 1], win[i + 1], acc1);
                    }
                    if (W & 1) acc0 = fma(ws.th[j][W - 1], win[W - 1], acc0);
                }
                const unsigned t = (unsigned)(lane - org.y);
                if (t < (unsigned)W) ws.part[j][t] = (acc0 + acc1) * ws.ph[j][t];
                ++j;
                if (j >= npt) break;
                org = ws.org[j];
            } while (org.x == a_base);
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
// a8: type-1 spreading (grid must be zero on entry)
// ---------------------------------------------------------------------------------------------
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

    for (int batch = start; batch < end; batch += 32) {
        const int idx = batch + lane;
        const bool has = idx < end;
        {
            const double X = has ? P.px[idx] : 0.0, Y = has ? P.py[idx] : 0.0;
            const T val = has ? map[P.perm[idx]] : (T)0;
            const double a0d = ceil(X - 0.5 * W), b0d = ceil(Y - 0.5 * W);
            const T ut = (T)(2.0 * ((a0d + 0.5 * W) - X) - 1.0);
            const T up = (T)(2.0 * ((b0d + 0.5 * W) - Y) - 1.0);
            T k[W];
            eval_taps<W, T>(kp, ut, k);
            // the point's value rides on the theta weights
            if constexpr (sizeof(T) == 8) {
#pragma unroll
                for (int i = 0; i + 1 < W; i += 2)
                    *reinterpret_cast<double2*>(&ws.th[lane][i]) = make_double2(val * k[i], val * k[i + 1]);
                if (W & 1) *reinterpret_cast<double2*>(&ws.th[lane][W - 1]) = make_double2(val * k[W - 1], 0.0);
            } else {
#pragma unroll
                for (int i = 0; i < W; ++i) ws.th[lane][i] = val * k[i];
            }
            eval_taps<W, T>(kp, up, k);
#pragma unroll
            for (int i = 0; i < W; ++i) ws.ph[lane][i] = k[i];
            ws.org[lane] = make_int2((int)a0d, (int)b0d - c0);
        }
        __syncwarp();
        const int npt = min(32, end - batch);
        int j = 0;
        int2 org = ws.org[0];
        while (j < npt) {
            if (org.x != a_base) {
                if (a_base == INT_MIN) {
                    a_base = org.x;
                } else {
                    int d = org.x - a_base;
                    if (d >= W) {
                        // flush the whole window
#pragma unroll
                        for (int i = 0; i < W; ++i) {
                            if (acc[i] != (T)0) atomicAdd(&grid[grid_index(g, a_base + i, col_n, col_m)], acc[i]);
                            acc[i] = 0;
                        }
                        a_base = org.x;
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
            // all points of the batch whose footprint starts on this row
#pragma unroll 1
            do {
                const unsigned t = (unsigned)(lane - org.y);
                const T kph = (t < (unsigned)W) ? ws.ph[j][t] : (T)0;
                if constexpr (sizeof(T) == 8) {
#pragma unroll
                    for (int i = 0; i + 1 < W; i += 2) {
                        const double2 kk = *reinterpret_cast<const double2*>(&ws.th[j][i]);
                        acc[i] = fma(kk.x, kph, acc[i]);
                        acc[i + 1] = fma(kk.y, kph, acc[i + 1]);
                    }
                    if (W & 1) acc[W - 1] = fma(ws.th[j][W - 1], kph, acc[W - 1]);
                } else {
#pragma unroll
                    for (int i = 0; i < W; ++i) acc[i] = fma(ws.th[j][i], kph, acc[i]);
                }
                ++j;
                if (j >= npt) break;
                org = ws.org[j];
            } while (org.x == a_base);
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
    NUSHT_CUDA_TRY(cudaGetLastError());
    return NUSHT_OK;
}
template <int W, typename T>
int launch_spread(const NufftParams& P, const KernelHost& h, const void* map, void* grid, cudaStream_t s) {
    const KernelPoly<T> kp = make_device_poly<T>(h);
    constexpr int NU_WARPS = nu_warps<W, T>();
    const int blocks = (P.n_items + NU_WARPS - 1) / NU_WARPS;
    k_spread<W, T><<<blocks, NU_WARPS * 32, 0, s>>>(P, kp, (const T*)map, (T*)grid);
    NUSHT_CUDA_TRY(cudaGetLastError());
    return NUSHT_OK;
}

template <typename T>
int dispatch_interp(int w, const NufftParams& P, const KernelHost& h, const void* grid, void* map, cudaStream_t s) {
    switch (w) {
#define NUSHT_CASE(WW) case WW: return launch_interp<WW, T>(P, h, grid, map, s);
        NUSHT_CASE(2) NUSHT_CASE(3) NUSHT_CASE(4) NUSHT_CASE(5) NUSHT_CASE(6) NUSHT_CASE(7) NUSHT_CASE(8)
        NUSHT_CASE(9) NUSHT_CASE(10) NUSHT_CASE(11) NUSHT_CASE(12) NUSHT_CASE(13) NUSHT_CASE(14)
        NUSHT_CASE(15) NUSHT_CASE(16)
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
        NUSHT_CASE(15) NUSHT_CASE(16)
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
    // width / shape rule of the ES kernel at up-sampling 2 (reading G8)
    int w = (int)ceil(log10(1.0 / p->eps)) + 1;
    if (w < 2) w = 2;
    if (w > NUSHT_MAX_W) return NUSHT_ERR_INVALID_ARG;
    double bw = 2.30;
    if (w == 2) bw = 2.20;
    if (w == 3) bw = 2.26;
    if (w == 4) bw = 2.38;
    KernelHost* h = new KernelHost();
    h->w = w;
    h->deg = poly_degree(w);
    h->beta = bw * w;
    p->beta = h->beta;
    p->ng.w = w;
    p->ng.fl = w / 2;
    p->ng.deg = h->deg;
    p->ng.mb = 33 - w;
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
    if (xg.empty()) gauss_legendre(32, xg, wg);
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

int nufft_sort_points(nusht_plan_s* p, const double* theta, const double* phi) {
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
    NUSHT_TRY(nu_alloc(&p->d_px, (size_t)n, p));
    NUSHT_TRY(nu_alloc(&p->d_py, (size_t)n, p));
    NUSHT_TRY(nu_alloc(&p->d_perm, (size_t)n, p));
    NUSHT_TRY(nu_alloc(&p->d_item_off, (size_t)p->n_items + 1, p));

    SortGeom sg;
    sg.nth = g.nth; sg.nph = g.nph; sg.w = g.w; sg.fl = g.fl; sg.mb = g.mb; sg.nstrip = g.nstrip; sg.nseg = g.nseg;
    sg.inv_hth = g.inv_hth; sg.inv_hph = g.inv_hph; sg.half_w = 0.5 * g.w;

    int *d_keys = nullptr, *d_hist = nullptr, *d_off = nullptr, *d_tot = nullptr, *d_bad = nullptr;
    const int ntiles = (nbins + 1 + SCAN_TILE - 1) / SCAN_TILE;
    int status = NUSHT_OK;
    auto cleanup = [&]() {
        cudaFree(d_keys); cudaFree(d_hist); cudaFree(d_off); cudaFree(d_tot); cudaFree(d_bad);
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
    SORT_TRY(cudaMalloc((void**)&d_hist, sizeof(int) * ((size_t)nbins + 1)));
    SORT_TRY(cudaMalloc((void**)&d_off, sizeof(int) * ((size_t)nbins + 1)));
    SORT_TRY(cudaMalloc((void**)&d_tot, sizeof(int) * (size_t)ntiles));
    SORT_TRY(cudaMalloc((void**)&d_bad, sizeof(int)));
    SORT_TRY(cudaMemset(d_hist, 0, sizeof(int) * ((size_t)nbins + 1)));
    SORT_TRY(cudaMemset(d_bad, 0, sizeof(int)));
    if (n > 0) {
        const int threads = 256;
        const unsigned blocks = (unsigned)((n + threads - 1) / threads);
        k_point_keys<<<blocks, threads>>>(sg, n, theta, phi, d_keys, d_hist, d_bad);
        SORT_TRY(cudaGetLastError());
        int bad = 0;
        SORT_TRY(cudaMemcpy(&bad, d_bad, sizeof(int), cudaMemcpyDeviceToHost));
        if (bad != 0) {
            cleanup();
            return NUSHT_ERR_BAD_POINTS;
        }
    }
    k_scan_tiles<<<ntiles, SCAN_BLOCK>>>(d_hist, d_off, d_tot, nbins + 1);
    SORT_TRY(cudaGetLastError());
    k_scan_totals<<<1, 1024>>>(d_tot, ntiles);
    SORT_TRY(cudaGetLastError());
    k_scan_add<<<ntiles, SCAN_BLOCK>>>(d_off, d_tot, nbins + 1);
    SORT_TRY(cudaGetLastError());
    k_item_offsets<<<(p->n_items + 1 + 255) / 256, 256>>>(d_off, p->d_item_off, p->n_items, (int)n);
    SORT_TRY(cudaGetLastError());
    if (n > 0) {
        const int threads = 256;
        const unsigned blocks = (unsigned)((n + threads - 1) / threads);
        k_point_scatter<<<blocks, threads>>>(sg, n, theta, phi, d_keys, d_off, p->d_px, p->d_py, p->d_perm);
        SORT_TRY(cudaGetLastError());
    }
    SORT_TRY(cudaDeviceSynchronize());
#undef SORT_TRY
    cleanup();
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
    if (p->dtype == NUSHT_F64) return dispatch_interp<double>(p->ng.w, P, *h, grid, map, s);
    return dispatch_interp<float>(p->ng.w, P, *h, grid, map, s);
}

int nufft_spread(nusht_plan_s* p, const void* map, void* grid, cudaStream_t s) {
    const size_t esz = (p->dtype == NUSHT_F64) ? 8 : 4;
    NUSHT_CUDA_TRY(cudaMemsetAsync(grid, 0, (size_t)p->ng.nrow_half * (size_t)p->ng.nph * esz, s));
    if (p->npts == 0) return NUSHT_OK;
    const KernelHost* h = g_kernel_of(p);
    const NufftParams P = make_nufft_params(p);
    if (p->dtype == NUSHT_F64) return dispatch_spread<double>(p->ng.w, P, *h, map, grid, s);
    return dispatch_spread<float>(p->ng.w, P, *h, map, grid, s);
}

void nufft_free(nusht_plan_s* p) {
    cudaFree(p->d_px); cudaFree(p->d_py); cudaFree(p->d_perm); cudaFree(p->d_item_off);
    p->d_px = p->d_py = nullptr; p->d_perm = nullptr; p->d_item_off = nullptr;
    delete static_cast<KernelHost*>(p->kernel_host);
    p->kernel_host = nullptr;
}
