// ls_pre.cu — per-point pre-processing kernels.
//
//   K1 stats        sum dy^-2, sum dy^-2 y per series -> W, ybar   (weights h_j: PAPER.md:22;
//                   w_j = dy_j^-2 / W, ybar weighted: north_star, reading A12)
//   K3 bin count    fine-grid cell of x1 = n df t and x2 = 2 x1 (f_k = k/2pi => rescale,
//                   PAPER.md:45; A3), histogram over bins of kBinCells cells, exclusive scan
//   K2 premultiply  cell/offset pair by a double-double product, unit phasor e^{2 pi i f_c t}
//                   (north_star "pre-multiplied by e^{2 pi i f0 t_j}"; A4), scatter into bin order
//   K2' rows        real strengths w_j and w_j (y_j - ybar) per series in bin order, and YY
//
// Coordinates and phases are ALWAYS fp64 double-double arithmetic (A9; error floor N_f eps_mach,
// PAPER.md:71): a grid coordinate is carried as (integer cell, fraction), never as one double.
#include "ls_internal.h"

namespace lsb {
namespace {

constexpr int kPreThreads = 256;
constexpr int kScanThreads = 1024;
constexpr int kScanItems = 4;
constexpr int kScanChunk = kScanThreads * kScanItems;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum over the CTA; result valid in thread 0.  `red` holds one double per warp.
__device__ __forceinline__ double block_sum(double v, double* red) {
    v = warp_sum(v);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) red[wid] = v;
    __syncthreads();
    double r = 0.0;
    if (wid == 0) {
        r = (lane < (int)(blockDim.x >> 5)) ? red[lane] : 0.0;
        r = warp_sum(r);
    }
    return r;
}

// (integer cell in [0,n), fraction in [0,1)) of the real number (A.hi + A.lo) * t  mod n.
// p = A.hi t is split exactly (p - floor p is exact), the FMA recovers the rounding error of the
// product, so the fraction is good to ~1e-16 cell even when p ~ 1e9 cells.
__device__ __forceinline__ void grid_coord(dd A, double t, double dn, int& cell, double& frac) {
    const double p = A.hi * t;
    const double e = fma(A.hi, t, -p) + A.lo * t;
    double c = floor(p);
    double f = (p - c) + e;
    if (f < 0.0) { f += 1.0; c -= 1.0; }
    if (f >= 1.0) { f -= 1.0; c += 1.0; }
    double r = fmod(c, dn);               // exact: c and dn are integers < 2^53
    if (r < 0.0) r += dn;
    cell = (int)r;
    frac = f;
}

// x2 = 2 x1 (exact doubling of cell and fraction), folded into [0, n).
__device__ __forceinline__ void grid_coord_x2(int c1, double f1, int n, int& c2, double& f2) {
    const int carry = f1 >= 0.5 ? 1 : 0;
    long long c = 2ll * c1 + carry;
    if (c >= n) c -= n;
    c2 = (int)c;
    f2 = 2.0 * f1 - (double)carry;
}

// First touched cell offset i0 = ceil(frac - w/2) and x0 = i0 - frac in [-w/2, -w/2 + 1).
__device__ __forceinline__ void support_start(double frac, int w, int& i0, double& x0) {
    const double a = ceil(frac - 0.5 * (double)w);
    i0 = (int)a;
    x0 = a - frac;
}

// opts.t_is_dtype: float times promoted exactly to double once, so every kernel below reads double times
__global__ void ls_promote_t_kernel(const float* __restrict__ tf, double* __restrict__ td, long long Nd) {
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < Nd; j += (long long)gridDim.x * blockDim.x)
        td[j] = (double)tf[j];
}

// ------------------------------------------------------------------------------ K1 stats + K3 count
// grid (point CTAs, batch), grid-stride over the points.  Every series accumulates sum dy^-2 y (and
// sum dy^-2 when it has its own dy); the CTAs of series 0 also histogram the fine-grid bins of both
// point sets.  One atomicAdd(double) per CTA and sum: the CTA count is capped by the launcher.
template <typename T>
__global__ void __launch_bounds__(kPreThreads)
ls_stats_count_kernel(const double* __restrict__ t, const T* __restrict__ y, const T* __restrict__ dy,
                      double* __restrict__ sums, long long Nd, int dy_per_series, dd ndf, int n,
                      int* __restrict__ hist1, int* __restrict__ hist2) {
    __shared__ double red[kPreThreads / 32];
    const int s = blockIdx.y;
    const T* ys = y + (long long)s * Nd;
    const T* ds = dy + (dy_per_series ? (long long)s * Nd : 0);
    const double dn = (double)n;
    const bool need_w = dy_per_series || s == 0;
    double a = 0.0, b = 0.0;
    for (long long j = (long long)blockIdx.x * kPreThreads + threadIdx.x; j < Nd;
         j += (long long)gridDim.x * kPreThreads) {
        const double d = (double)ds[j];
        const double iv = 1.0 / (d * d);
        a += iv;
        b += iv * (double)ys[j];
        if (s == 0) {
            int c1, c2;
            double f1, f2;
            grid_coord(ndf, t[j], dn, c1, f1);
            grid_coord_x2(c1, f1, n, c2, f2);
            atomicAdd(&hist1[c1 / kBinCells], 1);
            atomicAdd(&hist2[c2 / kBinCells], 1);
        }
    }
    b = block_sum(b, red);
    if (threadIdx.x == 0) atomicAdd(&sums[4 * s + 1], b);
    if (need_w) {
        a = block_sum(a, red);
        if (threadIdx.x == 0) atomicAdd(&sums[4 * s + 0], a);
    }
}

// ------------------------------------------------------------------------------ K3 scan
// Exclusive scan of one chunk of kScanChunk counts held 4 per thread; returns the thread's
// exclusive prefix within the chunk and the chunk total (all threads).
__device__ __forceinline__ int chunk_exclusive_scan(int v[kScanItems], int* warp_tot, int& total) {
    int tsum = 0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) tsum += v[i];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int inc = tsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int u = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += u;
    }
    __syncthreads();
    if (lane == 31) warp_tot[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int wv = warp_tot[lane];
        int winc = wv;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int u = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += u;
        }
        warp_tot[lane] = winc - wv;                 // exclusive prefix of warp totals
        if (lane == 31) warp_tot[32] = winc;        // chunk total
    }
    __syncthreads();
    total = warp_tot[32];
    return warp_tot[wid] + inc - tsum;
}

// Phase A: per-chunk totals; the last CTA to finish turns them into exclusive chunk offsets.
// tmp layout per point set: [nchunks] totals/offsets, then one ticket counter.
__global__ void __launch_bounds__(kScanThreads)
ls_bin_scan_totals_kernel(const int* __restrict__ hist1, const int* __restrict__ hist2, int nbins,
                          int nchunks, int* __restrict__ tmp) {
    __shared__ int warp_tot[33];
    __shared__ int is_last;
    const int psi = blockIdx.y;
    const int* hist = psi ? hist2 : hist1;
    int* tot = tmp + psi * (nchunks + 1);
    int* ticket = tot + nchunks;
    const int b0 = blockIdx.x * kScanChunk + threadIdx.x * kScanItems;
    int v[kScanItems];
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) v[i] = (b0 + i < nbins) ? hist[b0 + i] : 0;
    int total;
    chunk_exclusive_scan(v, warp_tot, total);
    if (threadIdx.x == 0) {
        tot[blockIdx.x] = total;
        __threadfence();
        is_last = (atomicAdd(ticket, 1) == nchunks - 1);
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        // serial-in-chunks scan of the nchunks totals by this CTA (nchunks <= a few thousand)
        int carry = 0;
        for (int c0 = 0; c0 < nchunks; c0 += kScanChunk) {
            const int i0 = c0 + threadIdx.x * kScanItems;
            int u[kScanItems];
#pragma unroll
            for (int i = 0; i < kScanItems; ++i) u[i] = (i0 + i < nchunks) ? __ldcg(&tot[i0 + i]) : 0;
            int ctot;
            int ex = chunk_exclusive_scan(u, warp_tot, ctot) + carry;
#pragma unroll
            for (int i = 0; i < kScanItems; ++i) {
                if (i0 + i < nchunks) tot[i0 + i] = ex;
                ex += u[i];
            }
            carry += ctot;
            __syncthreads();
        }
        if (threadIdx.x == 0) *ticket = 0;          // ready for the next execute
    }
}

// Phase B: exclusive scan inside each chunk + chunk offset -> bin_start and the scatter cursors
// (written over the counts).
__global__ void __launch_bounds__(kScanThreads)
ls_bin_scan_apply_kernel(int* __restrict__ hist1, int* __restrict__ hist2, int* __restrict__ start1,
                         int* __restrict__ start2, int nbins, int nchunks, const int* __restrict__ tmp,
                         int Nd) {
    __shared__ int warp_tot[33];
    const int psi = blockIdx.y;
    int* hist = psi ? hist2 : hist1;
    int* start = psi ? start2 : start1;
    const int offset = tmp[psi * (nchunks + 1) + blockIdx.x];
    const int b0 = blockIdx.x * kScanChunk + threadIdx.x * kScanItems;
    int v[kScanItems];
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) v[i] = (b0 + i < nbins) ? hist[b0 + i] : 0;
    int total;
    int ex = chunk_exclusive_scan(v, warp_tot, total) + offset;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        if (b0 + i < nbins) {
            start[b0 + i] = ex;
            hist[b0 + i] = ex;
        }
        ex += v[i];
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) start[nbins] = Nd;
}

// Small grids (all bins of a point set fit one chunk): both phases in one launch.
__global__ void __launch_bounds__(kScanThreads)
ls_bin_scan_single_kernel(int* __restrict__ hist1, int* __restrict__ hist2, int* __restrict__ start1,
                          int* __restrict__ start2, int nbins, int Nd) {
    __shared__ int warp_tot[33];
    int* hist = blockIdx.y ? hist2 : hist1;
    int* start = blockIdx.y ? start2 : start1;
    const int b0 = threadIdx.x * kScanItems;
    int v[kScanItems];
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) v[i] = (b0 + i < nbins) ? hist[b0 + i] : 0;
    int total;
    int ex = chunk_exclusive_scan(v, warp_tot, total);
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        if (b0 + i < nbins) {
            start[b0 + i] = ex;
            hist[b0 + i] = ex;                   // the counts become the scatter cursors
        }
        ex += v[i];
    }
    if (threadIdx.x == 0) start[nbins] = Nd;
}

// ------------------------------------------------------------------------------ K2 premultiply
template <typename T>
struct RecOf;
template <>
struct RecOf<double> { using type = Rec64; };
template <>
struct RecOf<float> { using type = Rec32; };

// One whole-record store: 32 bytes (STG.256) for fp64, 16 bytes for fp32.
__device__ __forceinline__ void store_rec(Rec64* dst, double eta, int l0, double qx, double qy) {
    const long long mid = (long long)(unsigned)l0;
    asm volatile("st.global.v4.b64 [%0], {%1, %2, %3, %4};" ::"l"(dst), "l"(__double_as_longlong(eta)), "l"(mid),
                 "l"(__double_as_longlong(qx)), "l"(__double_as_longlong(qy))
                 : "memory");
}
__device__ __forceinline__ void store_rec(Rec32* dst, double eta, int l0, double qx, double qy) {
    float4 v;
    v.x = (float)eta;
    v.y = __int_as_float(l0);
    v.z = (float)qx;
    v.w = (float)qy;
    *reinterpret_cast<float4*>(dst) = v;
}

// grid-stride over the points.
// FOLD_W (dy shared by the batch): the record's phasor is w_j e^{2 pi i f_c t_j}, not the unit phasor, so
//   the w transforms need no strength row at all (strength 1) and an h transform's strength is just
//   y_j - ybar: one scattered 8-byte store per point instead of three (they were half of this kernel's time).
// FUSE_ROWS (batch == 1): that one strength row of the single series is scattered here too and YY is
//   reduced, so no separate rows kernel runs.  Otherwise the sorted slot -> input index map `perm` is
//   written for the gathering rows kernel.
template <typename T, bool FUSE_ROWS, bool FOLD_W>
__global__ void __launch_bounds__(kPreThreads)
ls_premultiply_kernel(const double* __restrict__ t, const T* __restrict__ y, const T* __restrict__ dy,
                      double* __restrict__ sums, long long Nd, dd ndf, dd fc, int n, int w,
                      int* __restrict__ cur1, int* __restrict__ cur2, int* __restrict__ perm1,
                      int* __restrict__ perm2, typename RecOf<T>::type* __restrict__ rec1,
                      typename RecOf<T>::type* __restrict__ rec2, T* __restrict__ R1, T* __restrict__ R2) {
    __shared__ double red[kPreThreads / 32];
    const double dn = (double)n;
    double W = 1.0, ybar = 0.0, yy = 0.0;
    if (FUSE_ROWS || FOLD_W) {
        W = sums[0];
        ybar = sums[1] / W;
    }
    const double invW = 1.0 / W;
    for (long long j = (long long)blockIdx.x * kPreThreads + threadIdx.x; j < Nd;
         j += (long long)gridDim.x * kPreThreads) {
        // all three loads first, the two slot atomics as soon as the cells are known: their latencies
        // overlap each other and the phase arithmetic instead of lining up behind it
        const double tj = t[j];
        double yj = 0.0, dj = 1.0;
        if (FUSE_ROWS) yj = (double)y[j];
        if (FOLD_W) dj = (double)dy[j];
        int c1, c2, i1, i2;
        double f1, f2, xa, xb;
        grid_coord(ndf, tj, dn, c1, f1);
        grid_coord_x2(c1, f1, n, c2, f2);
        const int s1 = atomicAdd(&cur1[c1 / kBinCells], 1);
        const int s2 = atomicAdd(&cur2[c2 / kBinCells], 1);
        support_start(f1, w, i1, xa);
        support_start(f2, w, i2, xb);
        // phase of f_c t in cycles, reduced to [-0.5, 0.5] (double-double product)
        const double p = fc.hi * tj;
        const double e = fma(fc.hi, tj, -p) + fc.lo * tj;
        double ph = (p - rint(p)) + e;
        ph -= rint(ph);
        double sn, cs;
        sincospi(2.0 * ph, &sn, &cs);
        const double wj = FOLD_W ? invW / (dj * dj) : 1.0;
        // eta = 2 (x0 + w/2) - 1 in [-1, 1): argument of the piecewise-polynomial kernel
        store_rec(&rec1[s1], 2.0 * xa + (double)(w - 1), c1 + i1, wj * cs, wj * sn);
        store_rec(&rec2[s2], 2.0 * xb + (double)(w - 1), c2 + i2, wj * (cs * cs - sn * sn), wj * (2.0 * sn * cs));
        if (FUSE_ROWS) {
            const double yc = yj - ybar;
            R1[s1] = (T)yc;                     // the only stored row of x1: h / w = y - ybar
            yy += wj * yc * yc;
        } else {
            perm1[s1] = (int)j;
            if (!FOLD_W) perm2[s2] = (int)j;
        }
    }
    if (FUSE_ROWS) {
        yy = block_sum(yy, red);
        if (threadIdx.x == 0) atomicAdd(&sums[2], yy);
    }
}

// ------------------------------------------------------------------------------ K2' rows + YY
// batch > 1.  grid (slot CTAs, batch), grid-stride over SORTED slots: coalesced row writes, gathers
// of y and dy through perm (one series is Nd reals: L1/L2-resident).  Row layout: DESIGN.md §4.
template <typename T>
__global__ void __launch_bounds__(kPreThreads)
ls_rows_kernel(const T* __restrict__ y, const T* __restrict__ dy, double* __restrict__ sums,
               long long Nd, int dy_per_series, int no_w_row, const int* __restrict__ perm1,
               const int* __restrict__ perm2, T* __restrict__ R1, T* __restrict__ R2) {
    __shared__ double red[kPreThreads / 32];
    const int s = blockIdx.y;
    const T* ys = y + (long long)s * Nd;
    const T* ds = dy + (dy_per_series ? (long long)s * Nd : 0);
    const double W = sums[dy_per_series ? 4 * s : 0];
    const double ybar = sums[4 * s + 1] / W;
    const double invW = 1.0 / W;
    // per-series dy: R1 = [w_0, h_0, w_1, h_1, ...], R2 = [w_0, w_1, ...], h_s = w_s (y_s - ybar_s);
    // shared dy (weights folded into the records' phasors): R1 = [y_0 - ybar_0, y_1 - ybar_1, ...], no R2
    // (fixed mean, no_w_row: the w transform at x1 does not exist and its row is not stored: R1 = [h_0, h_1, ...])
    T* rowh = R1 + (long long)((dy_per_series && !no_w_row) ? 2 * s + 1 : s) * Nd;
    T* roww1 = R1 + (long long)(2 * s) * Nd;
    T* roww2 = R2 + (long long)s * Nd;
    double yy = 0.0;
    for (long long q = (long long)blockIdx.x * kPreThreads + threadIdx.x; q < Nd;
         q += (long long)gridDim.x * kPreThreads) {
        const int j = perm1[q];
        const double d = (double)ds[j];
        const double wj = invW / (d * d);
        const double yc = (double)ys[j] - ybar;
        yy += wj * yc * yc;
        if (dy_per_series) {
            rowh[q] = (T)(wj * yc);
            if (!no_w_row) roww1[q] = (T)wj;
            const double d2 = (double)ds[perm2[q]];
            roww2[q] = (T)(invW / (d2 * d2));
        } else {
            rowh[q] = (T)yc;
        }
    }
    yy = block_sum(yy, red);
    if (threadIdx.x == 0) atomicAdd(&sums[4 * s + 2], yy);
}

// CTAs along the points: enough to fill the machine, few enough that the one-per-CTA double atomics
// on the per-series sums stay cheap.
inline int point_blocks(long long Nd, int batch) {
    const long long want = (Nd + kPreThreads - 1) / kPreThreads;
    const long long cap = std::max<long long>(2, (148 * 16 + batch - 1) / batch);   // ~2400 CTAs over the whole batch
    return (int)(want < cap ? want : cap);
}

}  // namespace

cudaError_t launch_promote_t(ls_plan_s* p, const void* t_f32, cudaStream_t s) {
    ls_promote_t_kernel<<<point_blocks(p->Nd, 1), kPreThreads, 0, s>>>((const float*)t_f32, p->t64, p->Nd);
    return cudaGetLastError();
}

cudaError_t launch_stats_count(ls_plan_s* p, const double* t, const void* y, const void* dy, cudaStream_t s) {
    dim3 grid(point_blocks(p->Nd, p->batch), p->batch);
    if (p->dtype == LS_F64)
        ls_stats_count_kernel<double><<<grid, kPreThreads, 0, s>>>(t, (const double*)y, (const double*)dy, p->sums,
                                                                   p->Nd, p->opts.dy_per_series, p->ndf, (int)p->n,
                                                                   p->ps[0].hist, p->ps[1].hist);
    else
        ls_stats_count_kernel<float><<<grid, kPreThreads, 0, s>>>(t, (const float*)y, (const float*)dy, p->sums,
                                                                  p->Nd, p->opts.dy_per_series, p->ndf, (int)p->n,
                                                                  p->ps[0].hist, p->ps[1].hist);
    return cudaGetLastError();
}

cudaError_t launch_bin_scan(ls_plan_s* p, cudaStream_t s) {
    const int nchunks = (p->nbins + kScanChunk - 1) / kScanChunk;
    dim3 grid(nchunks, 2);
    if (nchunks == 1) {
        ls_bin_scan_single_kernel<<<grid, kScanThreads, 0, s>>>(p->ps[0].hist, p->ps[1].hist, p->ps[0].bin_start,
                                                               p->ps[1].bin_start, p->nbins, (int)p->Nd);
        return cudaGetLastError();
    }
    ls_bin_scan_totals_kernel<<<grid, kScanThreads, 0, s>>>(p->ps[0].hist, p->ps[1].hist, p->nbins, nchunks,
                                                            p->scan_tmp);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    ls_bin_scan_apply_kernel<<<grid, kScanThreads, 0, s>>>(p->ps[0].hist, p->ps[1].hist, p->ps[0].bin_start,
                                                           p->ps[1].bin_start, p->nbins, nchunks, p->scan_tmp,
                                                           (int)p->Nd);
    return cudaGetLastError();
}

template <typename T>
static cudaError_t premultiply_t(ls_plan_s* p, const double* t, const void* y, const void* dy, cudaStream_t s) {
    using R = typename RecOf<T>::type;
    const int nb = point_blocks(p->Nd, 1);
    PointSet& a = p->ps[0];
    PointSet& b = p->ps[1];
#define LS_PREMUL_ARGS                                                                                              \
    t, (const T*)y, (const T*)dy, p->sums, p->Nd, p->ndf, p->fc, (int)p->n, p->w, a.hist, b.hist, a.perm, b.perm,   \
        (R*)a.rec, (R*)b.rec, (T*)a.rows, (T*)b.rows
    if (p->opts.dy_per_series) ls_premultiply_kernel<T, false, false><<<nb, kPreThreads, 0, s>>>(LS_PREMUL_ARGS);
    else if (p->batch == 1) ls_premultiply_kernel<T, true, true><<<nb, kPreThreads, 0, s>>>(LS_PREMUL_ARGS);
    else ls_premultiply_kernel<T, false, true><<<nb, kPreThreads, 0, s>>>(LS_PREMUL_ARGS);
#undef LS_PREMUL_ARGS
    return cudaGetLastError();
}

cudaError_t launch_premultiply(ls_plan_s* p, const double* t, const void* y, const void* dy, cudaStream_t s) {
    return p->dtype == LS_F64 ? premultiply_t<double>(p, t, y, dy, s) : premultiply_t<float>(p, t, y, dy, s);
}

cudaError_t launch_rows(ls_plan_s* p, const void* y, const void* dy, cudaStream_t s) {
    dim3 grid(point_blocks(p->Nd, p->batch), p->batch);
    if (p->dtype == LS_F64)
        ls_rows_kernel<double><<<grid, kPreThreads, 0, s>>>((const double*)y, (const double*)dy, p->sums, p->Nd,
                                                            p->opts.dy_per_series, p->opts.no_floating_mean, p->ps[0].perm,
                                                            p->ps[1].perm, (double*)p->ps[0].rows, (double*)p->ps[1].rows);
    else
        ls_rows_kernel<float><<<grid, kPreThreads, 0, s>>>((const float*)y, (const float*)dy, p->sums, p->Nd,
                                                           p->opts.dy_per_series, p->opts.no_floating_mean, p->ps[0].perm,
                                                           p->ps[1].perm, (float*)p->ps[0].rows, (float*)p->ps[1].rows);
    return cudaGetLastError();
}

}  // namespace lsb
