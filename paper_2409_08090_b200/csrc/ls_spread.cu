// ls_spread.cu — K4, tile-owner spreading ("upsample the data to
// a fine grid"; spreading kernel = "exponential of semicircle" phi(z) = exp(beta (sqrt(1-z^2) - 1)),
// PAPER.md:47, formula from the cited Barnett et al. 2019).
//
//   b_l = sum_j c_j psi(l - u_j),  psi(s) = phi(2 s / w),  l taken mod n,
//   c_j = q_j r_{m,j}: one unit phasor q_j per point, one REAL strength per (transform m, point).
//
// Design (differs from the paper's cuFINUFFT prior art): every CTA OWNS one tile of
// L consecutive fine-grid cells of up to NS transforms and GATHERS the points whose support
// overlaps it (its own sort bins plus one halo bin each side, periodic images included).  The
// candidates are counting-sorted by first-touched cell in shared memory, then each thread
// accumulates the cells it owns in REGISTERS and writes them once with coalesced 16-byte stores —
// zeros included, so there is no memset pass, no global or shared floating-point atomic, and each
// grid cell is written exactly once.  Tiles without points reduce to a pure streaming store.
#include "ls_internal.h"

namespace lsb {
namespace {

constexpr int kCellsPerThreadMax = 4;                 // L <= kSpreadThreads * 4
constexpr int kChunkPts = 1024;                       // candidates staged per pass through smem
constexpr int kPtsPerThread = kChunkPts / kSpreadThreads;

template <typename T>
struct V2;
template <>
struct V2<double> { using type = double2; };
template <>
struct V2<float> { using type = float2; };

__device__ __forceinline__ double es_kernel(double z, double beta) {
    const double a = fmax(0.0, 1.0 - z * z);
    return exp(beta * (sqrt(a) - 1.0));
}
__device__ __forceinline__ float es_kernel(float z, float beta) {
    const float a = fmaxf(0.0f, 1.0f - z * z);
    return __expf(beta * (sqrtf(a) - 1.0f));
}

template <typename T>
struct SpreadArgs {
    int n, L, nbins, w, H;          // H = ceil(w/2): candidate halo in cells
    int ntiles, tile_stride;        // CTA b owns tile (b * tile_stride) mod ntiles (stride coprime to ntiles)
    T beta, two_over_w;
    const int* bin_start;
    const int* l0;
    const T* x0;
    const typename V2<T>::type* q;
    const T* rows;                   // first row of this launch
    long long Nd;
    int nrows;
    typename V2<T>::type* grid;      // first slot of this launch, [nrows][n]
};

// Block-wide exclusive scan of `cnt[0..len)` (len <= kSpreadThreads * 5) into `start[0..len]`.
__device__ __forceinline__ void block_scan_counts(const int* cnt, int* start, int len, int* warp_tot) {
    constexpr int PER = 5;
    const int b = threadIdx.x * PER;
    int v[PER], tsum = 0;
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        v[i] = (b + i < len) ? cnt[b + i] : 0;
        tsum += v[i];
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int inc = tsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int u = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += u;
    }
    if (lane == 31) warp_tot[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        int wv = (lane < kSpreadThreads / 32) ? warp_tot[lane] : 0;
        int winc = wv;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int u = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += u;
        }
        if (lane < kSpreadThreads / 32) warp_tot[lane] = winc - wv;
    }
    __syncthreads();
    int ex = warp_tot[wid] + inc - tsum;
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        if (b + i <= len) start[b + i] = ex;
        ex += v[i];
    }
}

template <typename T, int NS>
__global__ void __launch_bounds__(kSpreadThreads)
ls_spread_tile_kernel(const SpreadArgs<T> a) {
    using T2 = typename V2<T>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // shared layout: q[kChunkPts] T2 | x0[kChunkPts] T | r[NS][kChunkPts] T | rel[kChunkPts] int |
    //                cnt[HN] int | start[HN+1] int | warp_tot[8] int
    T2* sq = reinterpret_cast<T2*>(smem_raw);
    T* sx = reinterpret_cast<T*>(sq + kChunkPts);
    T* sr = sx + kChunkPts;
    int* srel = reinterpret_cast<int*>(sr + NS * kChunkPts);
    const int HN = a.L + a.w;                       // keys rel + (w-1) in [0, L + w - 1)
    int* cnt = srel + kChunkPts;
    int* start = cnt + HN;
    int* warp_tot = start + HN + 1;

    // Occupied tiles (compute/latency-bound) and empty tiles (pure streaming stores) are interleaved in
    // launch order by a multiplicative permutation, so the two kinds of work overlap on every SM.
    const int tile = (int)(((long long)blockIdx.x * a.tile_stride) % a.ntiles);
    const int row0 = blockIdx.y * NS;
    const int tile_lo = tile * a.L;
    const int Lt = min(a.L, a.n - tile_lo);
    const int w = a.w;

    // Candidate pieces: cells [lo, hi) = [tile_lo - H, tile_lo + Lt + H); the parts below 0 / at or
    // above n are the periodic images (shift -n / +n applied to the point's cell).
    const int lo = tile_lo - a.H, hi = tile_lo + Lt + a.H;
    int pbeg[3], pcnt[3], pshift[3];
    {
        // main piece
        const int mlo = max(lo, 0), mhi = min(hi, a.n);
        pbeg[0] = a.bin_start[mlo / kBinCells];
        pcnt[0] = a.bin_start[(mhi - 1) / kBinCells + 1] - pbeg[0];
        pshift[0] = 0;
        // left image: cells [n + lo, n) shifted by -n
        if (lo < 0) {
            const int c0 = max(a.n + lo, 0);
            pbeg[1] = a.bin_start[c0 / kBinCells];
            pcnt[1] = a.bin_start[a.nbins] - pbeg[1];
        } else { pbeg[1] = 0; pcnt[1] = 0; }
        pshift[1] = -a.n;
        // right image: cells [0, hi - n) shifted by +n
        if (hi > a.n) {
            const int c1 = min(hi - a.n, a.n);
            pbeg[2] = 0;
            pcnt[2] = a.bin_start[(c1 - 1) / kBinCells + 1];
        } else { pbeg[2] = 0; pcnt[2] = 0; }
        pshift[2] = a.n;
    }
    const int total = pcnt[0] + pcnt[1] + pcnt[2];

    T2 acc[kCellsPerThreadMax][NS];
#pragma unroll
    for (int c = 0; c < kCellsPerThreadMax; ++c)
#pragma unroll
        for (int s = 0; s < NS; ++s) acc[c][s].x = acc[c][s].y = (T)0;

    for (int base = 0; base < total; base += kChunkPts) {
        // ---- 1. count candidates of this chunk per first-touched cell
        for (int i = threadIdx.x; i < HN; i += kSpreadThreads) cnt[i] = 0;
        __syncthreads();
        int g[kPtsPerThread], key[kPtsPerThread];
#pragma unroll
        for (int i = 0; i < kPtsPerThread; ++i) {
            int ci = base + threadIdx.x + i * kSpreadThreads;
            key[i] = -1;
            g[i] = 0;
            if (ci < total) {
                int pc = 0;
                if (ci >= pcnt[0]) { ci -= pcnt[0]; pc = 1; if (ci >= pcnt[1]) { ci -= pcnt[1]; pc = 2; } }
                g[i] = pbeg[pc] + ci;
                const int rel = a.l0[g[i]] + pshift[pc] - tile_lo;     // first touched cell, tile-relative
                if (rel + w > 0 && rel < Lt) {
                    key[i] = rel + w - 1;
                    atomicAdd(&cnt[key[i]], 1);
                }
            }
        }
        __syncthreads();
        // ---- 2. exclusive scan -> start[]; cnt[] becomes the scatter cursor
        block_scan_counts(cnt, start, HN, warp_tot);
        __syncthreads();
        for (int i = threadIdx.x; i < HN; i += kSpreadThreads) cnt[i] = start[i];
        __syncthreads();
        // ---- 3. scatter the candidates into cell order
#pragma unroll
        for (int i = 0; i < kPtsPerThread; ++i) {
            if (key[i] >= 0) {
                const int slot = atomicAdd(&cnt[key[i]], 1);
                sq[slot] = a.q[g[i]];
                sx[slot] = a.x0[g[i]];
                srel[slot] = key[i] - (w - 1);
#pragma unroll
                for (int s = 0; s < NS; ++s)
                    sr[s * kChunkPts + slot] = (row0 + s < a.nrows) ? a.rows[(long long)(row0 + s) * a.Nd + g[i]] : (T)0;
            }
        }
        __syncthreads();
        // ---- 4. gather: cell l receives every point with rel in [l - w + 1, l], i.e. key in [l, l + w)
#pragma unroll
        for (int c = 0; c < kCellsPerThreadMax; ++c) {
            const int l = threadIdx.x + c * kSpreadThreads;
            if (l < Lt) {
                const int pe = start[l + w];
                for (int pt = start[l]; pt < pe; ++pt) {
                    const T z = (sx[pt] + (T)(l - srel[pt])) * a.two_over_w;
                    const T k = es_kernel(z, a.beta);
                    const T2 qq = sq[pt];
                    const T kx = k * qq.x, ky = k * qq.y;
#pragma unroll
                    for (int s = 0; s < NS; ++s) {
                        const T r = sr[s * kChunkPts + pt];
                        acc[c][s].x = fma(kx, r, acc[c][s].x);
                        acc[c][s].y = fma(ky, r, acc[c][s].y);
                    }
                }
            }
        }
        __syncthreads();
    }

    // ---- 5. the tile is written exactly once (zeros included)
#pragma unroll
    for (int s = 0; s < NS; ++s) {
        if (row0 + s < a.nrows) {
            T2* out = a.grid + (long long)(row0 + s) * a.n + tile_lo;
#pragma unroll
            for (int c = 0; c < kCellsPerThreadMax; ++c) {
                const int l = threadIdx.x + c * kSpreadThreads;
                if (l < Lt) out[l] = acc[c][s];
            }
        }
    }
}

template <typename T, int NS>
size_t spread_smem_bytes(int L, int w) {
    const int HN = L + w;
    return sizeof(typename V2<T>::type) * kChunkPts + sizeof(T) * kChunkPts * (1 + NS) + sizeof(int) * kChunkPts +
           sizeof(int) * (HN + HN + 1 + 8);
}

template <typename T, int NS>
cudaError_t launch_ns(ls_plan_s* p, const SpreadArgs<T>& a, cudaStream_t s) {
    static bool configured = false;
    const size_t smem = spread_smem_bytes<T, NS>(p->L, p->w);
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(ls_spread_tile_kernel<T, NS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)spread_smem_bytes<T, NS>(kSpreadThreads * kCellsPerThreadMax, kMaxWidth));
        if (e != cudaSuccess) return e;
        configured = true;
    }
    dim3 grid(p->ntiles, (a.nrows + NS - 1) / NS);
    ls_spread_tile_kernel<T, NS><<<grid, kSpreadThreads, smem, s>>>(a);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_t(ls_plan_s* p, int pointset, int row0, int nrows, int slot0, cudaStream_t s) {
    using T2 = typename V2<T>::type;
    const PointSet& ps = p->ps[pointset];
    SpreadArgs<T> a;
    a.n = (int)p->n;
    a.L = p->L;
    a.nbins = p->nbins;
    a.ntiles = p->ntiles;
    a.tile_stride = p->tile_stride;
    a.w = p->w;
    a.H = (p->w + 1) / 2;
    a.beta = (T)p->beta;
    a.two_over_w = (T)(2.0 / p->w);
    a.bin_start = ps.bin_start;
    a.l0 = ps.l0;
    a.x0 = (const T*)ps.x0;
    a.q = (const T2*)ps.q;
    a.rows = (const T*)ps.rows + (long long)row0 * p->Nd;
    a.Nd = p->Nd;
    a.nrows = nrows;
    a.grid = (T2*)p->grids + (long long)slot0 * p->n;
    if (nrows == 1) return launch_ns<T, 1>(p, a, s);
    if (nrows == 2) return launch_ns<T, 2>(p, a, s);
    return launch_ns<T, 4>(p, a, s);
}

}  // namespace

cudaError_t launch_spread(ls_plan_s* p, int pointset, int row0, int nrows, int slot0, cudaStream_t s) {
    if (nrows <= 0) return cudaSuccess;
    return p->dtype == LS_F64 ? launch_t<double>(p, pointset, row0, nrows, slot0, s)
                              : launch_t<float>(p, pointset, row0, nrows, slot0, s);
}

}  // namespace lsb
