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
constexpr int kPreItems = 4;                       // points per thread in the 1-D point kernels
constexpr int kPreChunk = kPreThreads * kPreItems;
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

// ------------------------------------------------------------------------------ K1 stats
template <typename T>
__global__ void __launch_bounds__(kPreThreads)
ls_stats_kernel(const T* __restrict__ y, const T* __restrict__ dy, double* __restrict__ sums,
                long long Nd, int dy_per_series) {
    __shared__ double red[kPreThreads / 32];
    const int s = blockIdx.y;
    const long long base = (long long)blockIdx.x * kPreChunk;
    const T* ys = y + (long long)s * Nd;
    const T* ds = dy + (dy_per_series ? (long long)s * Nd : 0);
    double a = 0.0, b = 0.0;
#pragma unroll
    for (int i = 0; i < kPreItems; ++i) {
        const long long j = base + threadIdx.x + (long long)i * kPreThreads;
        if (j < Nd) {
            const double d = (double)ds[j];
            const double iv = 1.0 / (d * d);
            a += iv;
            b += iv * (double)ys[j];
        }
    }
    b = block_sum(b, red);
    if (threadIdx.x == 0) atomicAdd(&sums[4 * s + 1], b);
    if (dy_per_series || s == 0) {
        a = block_sum(a, red);
        if (threadIdx.x == 0) atomicAdd(&sums[4 * s + 0], a);
    }
}

// ------------------------------------------------------------------------------ K3 bin count
__global__ void __launch_bounds__(kPreThreads)
ls_bin_count_kernel(const double* __restrict__ t, long long Nd, dd ndf, int n,
                    int* __restrict__ hist1, int* __restrict__ hist2) {
    const long long base = (long long)blockIdx.x * kPreChunk;
    const double dn = (double)n;
#pragma unroll
    for (int i = 0; i < kPreItems; ++i) {
        const long long j = base + threadIdx.x + (long long)i * kPreThreads;
        if (j < Nd) {
            int c1, c2;
            double f1, f2;
            grid_coord(ndf, t[j], dn, c1, f1);
            grid_coord_x2(c1, f1, n, c2, f2);
            atomicAdd(&hist1[c1 / kBinCells], 1);
            atomicAdd(&hist2[c2 / kBinCells], 1);
        }
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

// ------------------------------------------------------------------------------ K2 premultiply
template <typename T>
struct Cplx;
template <>
struct Cplx<double> { using type = double2; };
template <>
struct Cplx<float> { using type = float2; };

template <typename T>
__global__ void __launch_bounds__(kPreThreads)
ls_premultiply_kernel(const double* __restrict__ t, long long Nd, dd ndf, dd fc, int n, int w,
                      int* __restrict__ cur1, int* __restrict__ cur2,
                      int* __restrict__ pos1, int* __restrict__ pos2,
                      int* __restrict__ l01, int* __restrict__ l02,
                      T* __restrict__ x01, T* __restrict__ x02,
                      typename Cplx<T>::type* __restrict__ q1, typename Cplx<T>::type* __restrict__ q2) {
    using T2 = typename Cplx<T>::type;
    const long long base = (long long)blockIdx.x * kPreChunk;
    const double dn = (double)n;
#pragma unroll
    for (int i = 0; i < kPreItems; ++i) {
        const long long j = base + threadIdx.x + (long long)i * kPreThreads;
        if (j >= Nd) continue;
        const double tj = t[j];
        int c1, c2, i1, i2;
        double f1, f2, xa, xb;
        grid_coord(ndf, tj, dn, c1, f1);
        grid_coord_x2(c1, f1, n, c2, f2);
        support_start(f1, w, i1, xa);
        support_start(f2, w, i2, xb);
        // phase of f_c t in cycles, reduced to [-0.5, 0.5] (double-double product)
        const double p = fc.hi * tj;
        const double e = fma(fc.hi, tj, -p) + fc.lo * tj;
        double ph = (p - rint(p)) + e;
        ph -= rint(ph);
        double sn, cs;
        sincospi(2.0 * ph, &sn, &cs);
        const int s1 = atomicAdd(&cur1[c1 / kBinCells], 1);
        const int s2 = atomicAdd(&cur2[c2 / kBinCells], 1);
        pos1[j] = s1;
        pos2[j] = s2;
        l01[s1] = c1 + i1;
        l02[s2] = c2 + i2;
        x01[s1] = (T)xa;
        x02[s2] = (T)xb;
        T2 a, b;
        a.x = (T)cs;
        a.y = (T)sn;
        b.x = (T)(cs * cs - sn * sn);
        b.y = (T)(2.0 * sn * cs);
        q1[s1] = a;
        q2[s2] = b;
    }
}

// ------------------------------------------------------------------------------ K2' rows + YY
// grid (point chunks, batch).  Row layout:
//   shared dy:      R1 = [w ; h_0 .. h_{B-1}],  R2 = [w]
//   per-series dy:  R1 = [w_0, h_0, w_1, h_1, ...],  R2 = [w_0, w_1, ...]
template <typename T>
__global__ void __launch_bounds__(kPreThreads)
ls_rows_kernel(const T* __restrict__ y, const T* __restrict__ dy, double* __restrict__ sums,
               long long Nd, int dy_per_series, const int* __restrict__ pos1,
               const int* __restrict__ pos2, T* __restrict__ R1, T* __restrict__ R2) {
    __shared__ double red[kPreThreads / 32];
    const int s = blockIdx.y;
    const long long base = (long long)blockIdx.x * kPreChunk;
    const T* ys = y + (long long)s * Nd;
    const T* ds = dy + (dy_per_series ? (long long)s * Nd : 0);
    const double W = sums[dy_per_series ? 4 * s : 0];
    const double ybar = sums[4 * s + 1] / W;
    const double invW = 1.0 / W;
    T* rowh = R1 + (long long)(dy_per_series ? 2 * s + 1 : 1 + s) * Nd;
    T* roww1 = R1 + (long long)(dy_per_series ? 2 * s : 0) * Nd;
    T* roww2 = R2 + (long long)(dy_per_series ? s : 0) * Nd;
    const bool write_w = dy_per_series || s == 0;
    double yy = 0.0;
#pragma unroll
    for (int i = 0; i < kPreItems; ++i) {
        const long long j = base + threadIdx.x + (long long)i * kPreThreads;
        if (j < Nd) {
            const double d = (double)ds[j];
            const double wj = invW / (d * d);
            const double yc = (double)ys[j] - ybar;
            const int s1 = pos1[j];
            rowh[s1] = (T)(wj * yc);
            yy += wj * yc * yc;
            if (write_w) {
                roww1[s1] = (T)wj;
                roww2[pos2[j]] = (T)wj;
            }
        }
    }
    yy = block_sum(yy, red);
    if (threadIdx.x == 0) atomicAdd(&sums[4 * s + 2], yy);
}

inline int point_blocks(long long Nd) { return (int)((Nd + kPreChunk - 1) / kPreChunk); }

}  // namespace

cudaError_t launch_stats(ls_plan_s* p, const double*, const void* y, const void* dy, cudaStream_t s) {
    dim3 grid(point_blocks(p->Nd), p->batch);
    if (p->dtype == LS_F64)
        ls_stats_kernel<double><<<grid, kPreThreads, 0, s>>>((const double*)y, (const double*)dy, p->sums, p->Nd,
                                                             p->opts.dy_per_series);
    else
        ls_stats_kernel<float><<<grid, kPreThreads, 0, s>>>((const float*)y, (const float*)dy, p->sums, p->Nd,
                                                            p->opts.dy_per_series);
    return cudaGetLastError();
}

cudaError_t launch_bin_count(ls_plan_s* p, const double* t, cudaStream_t s) {
    ls_bin_count_kernel<<<point_blocks(p->Nd), kPreThreads, 0, s>>>(t, p->Nd, p->ndf, (int)p->n, p->ps[0].hist,
                                                                    p->ps[1].hist);
    return cudaGetLastError();
}

cudaError_t launch_bin_scan(ls_plan_s* p, cudaStream_t s) {
    const int nchunks = (p->nbins + kScanChunk - 1) / kScanChunk;
    dim3 grid(nchunks, 2);
    ls_bin_scan_totals_kernel<<<grid, kScanThreads, 0, s>>>(p->ps[0].hist, p->ps[1].hist, p->nbins, nchunks,
                                                            p->scan_tmp);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    ls_bin_scan_apply_kernel<<<grid, kScanThreads, 0, s>>>(p->ps[0].hist, p->ps[1].hist, p->ps[0].bin_start,
                                                           p->ps[1].bin_start, p->nbins, nchunks, p->scan_tmp,
                                                           (int)p->Nd);
    return cudaGetLastError();
}

cudaError_t launch_premultiply(ls_plan_s* p, const double* t, cudaStream_t s) {
    const int nb = point_blocks(p->Nd);
    if (p->dtype == LS_F64)
        ls_premultiply_kernel<double><<<nb, kPreThreads, 0, s>>>(
            t, p->Nd, p->ndf, p->fc, (int)p->n, p->w, p->ps[0].hist, p->ps[1].hist, p->ps[0].pos, p->ps[1].pos,
            p->ps[0].l0, p->ps[1].l0, (double*)p->ps[0].x0, (double*)p->ps[1].x0, (double2*)p->ps[0].q,
            (double2*)p->ps[1].q);
    else
        ls_premultiply_kernel<float><<<nb, kPreThreads, 0, s>>>(
            t, p->Nd, p->ndf, p->fc, (int)p->n, p->w, p->ps[0].hist, p->ps[1].hist, p->ps[0].pos, p->ps[1].pos,
            p->ps[0].l0, p->ps[1].l0, (float*)p->ps[0].x0, (float*)p->ps[1].x0, (float2*)p->ps[0].q,
            (float2*)p->ps[1].q);
    return cudaGetLastError();
}

cudaError_t launch_rows(ls_plan_s* p, const void* y, const void* dy, cudaStream_t s) {
    dim3 grid(point_blocks(p->Nd), p->batch);
    if (p->dtype == LS_F64)
        ls_rows_kernel<double><<<grid, kPreThreads, 0, s>>>((const double*)y, (const double*)dy, p->sums, p->Nd,
                                                            p->opts.dy_per_series, p->ps[0].pos, p->ps[1].pos,
                                                            (double*)p->ps[0].rows, (double*)p->ps[1].rows);
    else
        ls_rows_kernel<float><<<grid, kPreThreads, 0, s>>>((const float*)y, (const float*)dy, p->sums, p->Nd,
                                                           p->opts.dy_per_series, p->ps[0].pos, p->ps[1].pos,
                                                           (float*)p->ps[0].rows, (float*)p->ps[1].rows);
    return cudaGetLastError();
}

}  // namespace lsb
