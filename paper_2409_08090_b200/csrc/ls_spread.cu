// ls_spread.cu — K4, tile-owner spreading ("upsample the data to
// a fine grid"; spreading kernel = "exponential of semicircle" phi(z) = exp(beta (sqrt(1-z^2) - 1)),
// PAPER.md:47, formula from the cited Barnett et al. 2019, evaluated as a piecewise polynomial
// ("piecewise polynomial kernel approximation") fitted at plan time).
//
//   b_l = sum_j c_j psi(l - u_j),  psi(s) = phi(2 s / w),  l taken mod n,
//   c_j = q_j r_{m,j}: one unit phasor q_j per point, one REAL strength per (transform m, point).
//
// Design (differs from the paper's cuFINUFFT prior art): every CTA OWNS one tile of
// L consecutive fine-grid cells of up to NS transforms and GATHERS the points whose support
// overlaps it (its own sort bins plus one halo bin each side, periodic images included):
//   1. each thread takes one candidate (one 32-byte record load), keys it by first-touched cell and
//      ranks it with an integer shared-memory atomic;
//   2. a block scan of the per-cell counts gives every candidate its slot in cell order;
//   3. the candidate's thread evaluates its w kernel values by Horner (coefficients are warp-uniform
//      kernel parameters; even/odd symmetry gives two values per evaluation) and stores them, with
//      the NS complex strengths, at its slot;
//   4. every thread then owns CPT consecutive cells, accumulates them in REGISTERS from the
//      slot-ordered staging area and writes them once with 32-byte stores.
// There is no memset pass and no global or shared floating-point atomic; each grid cell is written at
// most once.  A tile without points is a pure streaming store of zeros when cuFFT follows; with the
// library's own FFT it is not written at all (its liveness bit stays unset).  One launch covers both point
// sets (blockIdx.y) and the tiles are visited in a permuted order so that compute-bound occupied
// tiles and store-bound empty tiles overlap on every SM.
#include "ls_internal.h"

namespace lsb {
namespace {

constexpr int kScanPer = 5;                           // counts per thread in the block scan
constexpr int kValStride = kChunkPts + 1;             // odd: conflict-free kernel-value staging

template <typename T>
struct V2;
template <>
struct V2<double> { using type = double2; };
template <>
struct V2<float> { using type = float2; };
template <typename T>
struct RecOf;
template <>
struct RecOf<double> { using type = Rec64; };
template <>
struct RecOf<float> { using type = Rec32; };

template <typename T>
struct SpreadSeg {
    const int* bin_start;
    const typename RecOf<T>::type* rec;
    const T* rows;                   // stored strength rows of this point set (physical row 0)
    int first_row;                   // logical index of the launch's first row within the point set
    typename V2<T>::type* grid;      // first slot of this segment, [nrows][n]
    int nrows, ngroups;
};

template <typename T>
struct SpreadArgs {
    int n, L, nbins, w, H;           // H = ceil(w/2): candidate halo in cells
    int ntiles, tile_stride;         // CTA b owns tile (b * tile_stride) mod ntiles
    int tile_mask;                   // ntiles - 1 when ntiles is a power of two, else -1
    int half;                        // ceil(w/2) stored polynomial pieces
    int skip_empty;                  // own FFT: tiles without points are flagged, not zero-filled
    unsigned* row_masks;             // own FFT: liveness bits of the written tiles (layout: ls_fft.cu FftArgs)
    int ncoltiles, coltile_shift;    // tiles per FFT pass-1 row (65536 / L) and its log2
    int fft_rb;                      // pass-1 radix / 16: row = fft_rb * i + j
    const int* tile_list;            // own FFT: [2][ntiles] tiles that hold points, per point set (x2, x1)
    const int* tile_counts;          // own FFT: [2] lengths of the two lists
    int w_implicit;                  // shared dy: logical row 0 (the w transform) has strength 1 (the weights are
                                     // folded into the records' phasors) and is not stored; stored row = logical - 1
    long long Nd;
    SpreadSeg<T> seg[2];             // blockIdx.y < seg[0].ngroups: x2 rows, else x1 rows
    T c[kHalfMax][kMaxDeg + 1];      // only degrees <= PolyDeg<T> are read
};

__device__ __forceinline__ void load_rec(const Rec64* p, double& eta, int& l0, double& qx, double& qy) {
    long long a, b, c, d;
    asm volatile("ld.global.nc.v4.b64 {%0, %1, %2, %3}, [%4];" : "=l"(a), "=l"(b), "=l"(c), "=l"(d) : "l"(p));
    eta = __longlong_as_double(a);
    l0 = (int)(unsigned)(unsigned long long)b;
    qx = __longlong_as_double(c);
    qy = __longlong_as_double(d);
}
__device__ __forceinline__ void load_rec(const Rec32* p, float& eta, int& l0, float& qx, float& qy) {
    const float4 v = __ldg(reinterpret_cast<const float4*>(p));
    eta = v.x;
    l0 = __float_as_int(v.y);
    qx = v.z;
    qy = v.w;
}

// CPT consecutive complex cells of one thread, written with the widest stores available.
template <int CPT>
__device__ __forceinline__ void store_cells(double2* dst, const double2 (&v)[CPT]) {
    if constexpr (CPT % 2 == 0) {
#pragma unroll
        for (int c = 0; c < CPT; c += 2)
            asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(dst + c), "d"(v[c].x), "d"(v[c].y),
                         "d"(v[c + 1].x), "d"(v[c + 1].y)
                         : "memory");
    } else {
#pragma unroll
        for (int c = 0; c < CPT; ++c) dst[c] = v[c];
    }
}
template <int CPT>
__device__ __forceinline__ void store_cells(float2* dst, const float2 (&v)[CPT]) {
    if constexpr (CPT % 4 == 0) {
#pragma unroll
        for (int c = 0; c < CPT; c += 4)
            asm volatile("st.global.v8.f32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(dst + c), "f"(v[c].x),
                         "f"(v[c].y), "f"(v[c + 1].x), "f"(v[c + 1].y), "f"(v[c + 2].x), "f"(v[c + 2].y),
                         "f"(v[c + 3].x), "f"(v[c + 3].y)
                         : "memory");
    } else if constexpr (CPT % 2 == 0) {
#pragma unroll
        for (int c = 0; c < CPT; c += 2)
            *reinterpret_cast<float4*>(dst + c) = make_float4(v[c].x, v[c].y, v[c + 1].x, v[c + 1].y);
    } else {
#pragma unroll
        for (int c = 0; c < CPT; ++c) dst[c] = v[c];
    }
}

// Block-wide exclusive scan of cnt[0..len) (len <= kSpreadThreads * kScanPer) into start[0..len];
// cnt is left zeroed.
__device__ __forceinline__ void block_scan_counts(int* cnt, int* start, int len, int* warp_tot) {
    const int b = threadIdx.x * kScanPer;
    int v[kScanPer], tsum = 0;
#pragma unroll
    for (int i = 0; i < kScanPer; ++i) {
        v[i] = 0;
        if (b + i < len) {
            v[i] = cnt[b + i];
            cnt[b + i] = 0;                          // ready for the next chunk of candidates
        }
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
        const int wv = (lane < kSpreadThreads / 32) ? warp_tot[lane] : 0;
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
    for (int i = 0; i < kScanPer; ++i) {
        if (b + i <= len) start[b + i] = ex;
        ex += v[i];
    }
}

// Polynomial degree the kernels unroll to (coefficients above the fitted degree are zero):
// 12 reaches the sqrt-singularity floor of the ES kernel (<= 7e-13) for every fp64 width, 8 is
// below 1e-7 for every fp32 width (measured at plan time, KernelPoly::max_err).
template <typename T>
struct PolyDeg;
template <>
struct PolyDeg<double> { static constexpr int value = 12; };
template <>
struct PolyDeg<float> { static constexpr int value = 8; };

// Cells [lbase, lbase + CPT) of one thread += the staged candidates [pb, pe) (cell order); NR <= NS
// rows are live.
template <typename T, int NR, int NS, int CPT>
__device__ __forceinline__ void gather_cells(typename V2<T>::type (&acc)[NS][CPT], const typename V2<T>::type* sc,
                                             const T* sval, const int* srel, int pb, int pe, int lbase, int w) {
    using T2 = typename V2<T>::type;
    for (int pt = pb; pt < pe; ++pt) {
        const int i0 = lbase - srel[pt];
        T2 cs[NR];
#pragma unroll
        for (int s = 0; s < NR; ++s) cs[s] = sc[s * kChunkPts + pt];
#pragma unroll
        for (int c = 0; c < CPT; ++c) {
            const int i = i0 + c;
            if ((unsigned)i < (unsigned)w) {
                const T k = sval[i * kValStride + pt];
#pragma unroll
                for (int s = 0; s < NR; ++s) {
                    acc[s][c].x = fma(k, cs[s].x, acc[s][c].x);
                    acc[s][c].y = fma(k, cs[s].y, acc[s][c].y);
                }
            }
        }
    }
}

// Candidates of the tile [tile_lo, tile_lo + Lt): the points of the sort bins overlapping cells
// [lo, hi) = [tile_lo - H, tile_lo + Lt + H).  Main piece = the part inside [0, n); the parts below 0 / at
// or above n are periodic images (pieces 1 and 2, cell shift -n / +n).  Returns the total count.
__device__ __forceinline__ int tile_candidates(const int* __restrict__ bin_start, int n, int nbins, int H, int tile_lo,
                                               int Lt, int& pbeg0, int& pcnt0, int& pbeg1, int& pcnt1, int& pcnt2) {
    const int lo = tile_lo - H, hi = tile_lo + Lt + H;
    pbeg1 = 0; pcnt1 = 0; pcnt2 = 0;
    if (lo >= 0 && hi <= n) {                        // interior tile: two loads, no images
        pbeg0 = __ldg(&bin_start[(unsigned)lo / kBinCells]);
        pcnt0 = __ldg(&bin_start[(unsigned)(hi - 1) / kBinCells + 1]) - pbeg0;
    } else {
        const int mlo = max(lo, 0), mhi = min(hi, n);
        pbeg0 = __ldg(&bin_start[mlo / kBinCells]);
        pcnt0 = __ldg(&bin_start[(mhi - 1) / kBinCells + 1]) - pbeg0;
        if (lo < 0) {                                // left image: cells [n + lo, n) shifted by -n
            pbeg1 = __ldg(&bin_start[max(n + lo, 0) / kBinCells]);
            pcnt1 = __ldg(&bin_start[nbins]) - pbeg1;
        }
        if (hi > n)                                  // right image: cells [0, hi - n) shifted by +n
            pcnt2 = __ldg(&bin_start[(min(hi - n, n) - 1) / kBinCells + 1]);
    }
    return pcnt0 + pcnt1 + pcnt2;
}

// Own-FFT path: the tiles that hold points, listed per point set (so that the spreading kernel launches
// work for them only), and their liveness bits for the first FFT pass.  One thread per (set, tile).
__global__ void ls_tile_list_kernel(const int* __restrict__ bin_start_x2, const int* __restrict__ bin_start_x1, int n,
                                    int nbins, int H, int L, int ntiles, int* __restrict__ list, int* __restrict__ counts,
                                    unsigned* __restrict__ row_masks, int ncoltiles, int coltile_shift, int fft_rb) {
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 2 * ntiles) return;
    const int set = idx >= ntiles ? 1 : 0, tile = idx - set * ntiles;
    const int tile_lo = tile * L;
    int b0, c0, b1, c1, c2;
    if (tile_candidates(set ? bin_start_x1 : bin_start_x2, n, nbins, H, tile_lo, min(L, n - tile_lo), b0, c0, b1, c1, c2) == 0)
        return;
    const int row = tile >> coltile_shift, ct = tile & (ncoltiles - 1);
    atomicOr(&row_masks[(set * ncoltiles + ct) * fft_rb + (row % fft_rb)], 1u << (row / fft_rb));
    // one counter atomic per warp and set, not per tile (thousands of same-address atomics serialise)
    const unsigned peers = __match_any_sync(__activemask(), set);
    const int leader = __ffs(peers) - 1, lane = threadIdx.x & 31;
    int base = 0;
    if (lane == leader) base = atomicAdd(&counts[set], __popc(peers));
    base = __shfl_sync(peers, base, leader);
    list[set * ntiles + base + __popc(peers & ((1u << lane) - 1))] = tile;
}

// cuFFT path: the library FFT reads every cell, so tiles without points must hold zeros — but writing them with one
// CTA per (tile, row group) is latency-bound when nearly all tiles are empty (config 5: 96 % of 307 000 tiles, 1.5 ms for
// 3.8 GB of zeros).  This kernel does both jobs in one persistent sweep: every thread tests one (set, tile) pair of a
// chunk of 256, occupied tiles go to the per-set lists the spreading kernel then walks (as on the own-FFT path), and the
// CTA streams zeros over the chunk's empty tiles for all rows of the pass with 16-byte stores.  build_list = 0 on later
// passes of a batch (the lists do not change, the grids are reused).
template <typename T2>
__global__ void __launch_bounds__(256)
ls_tile_zero_list_kernel(const int* __restrict__ bin_start_x2, const int* __restrict__ bin_start_x1, int n, int nbins, int H, int L,
                         int ntiles, int* __restrict__ list, int* __restrict__ counts, int build_list, T2* __restrict__ grid_x2,
                         int nrows_x2, T2* __restrict__ grid_x1, int nrows_x1) {
    __shared__ unsigned char empty[256];
    const int total = 2 * ntiles, nchunks = (total + 255) / 256;
    for (int chunk = blockIdx.x; chunk < nchunks; chunk += gridDim.x) {
        const int idx = chunk * 256 + threadIdx.x;
        bool occupied = false;
        int set = 0, tile = 0;
        if (idx < total) {
            set = idx >= ntiles ? 1 : 0;
            tile = idx - set * ntiles;
            const int tile_lo = tile * L;
            int b0, c0, b1, c1, c2;
            occupied = tile_candidates(set ? bin_start_x1 : bin_start_x2, n, nbins, H, tile_lo, min(L, n - tile_lo), b0, c0, b1, c1, c2) != 0;
        }
        if (build_list && occupied && blockIdx.y == 0) {
            const unsigned peers = __match_any_sync(__activemask(), set);
            const int leader = __ffs(peers) - 1, lane = threadIdx.x & 31;
            int base = 0;
            if (lane == leader) base = atomicAdd(&counts[set], __popc(peers));
            base = __shfl_sync(peers, base, leader);
            list[set * ntiles + base + __popc(peers & ((1u << lane) - 1))] = tile;
        }
        empty[threadIdx.x] = idx < total && !occupied;
        __syncthreads();
        for (int e = 0; e < 256; ++e) {
            if (!empty[e]) continue;                                   // CTA-uniform
            const int ix = chunk * 256 + e;
            const int st = ix >= ntiles ? 1 : 0, tl = ix - st * ntiles;
            const int rows = st ? nrows_x1 : nrows_x2;
            T2* g = (st ? grid_x1 : grid_x2) + (long long)tl * L;
            const int bytes = min(L, n - tl * L) * (int)sizeof(T2);
            for (int r = blockIdx.y; r < rows; r += gridDim.y) {         // a batch: the rows are shared out over blockIdx.y
                char* dst = reinterpret_cast<char*>(g + (long long)r * n);
                for (int off = threadIdx.x * 16; off < bytes; off += 256 * 16)
                    *reinterpret_cast<float4*>(dst + off) = make_float4(0.f, 0.f, 0.f, 0.f);
            }
        }
        __syncthreads();
    }
}

template <typename T, int NS, int CPT>
__global__ void __launch_bounds__(kSpreadThreads, (NS * CPT <= 8) ? 4 : 3)
ls_spread_tile_kernel(const __grid_constant__ SpreadArgs<T> a) {
    using T2 = typename V2<T>::type;
    constexpr int DEG = PolyDeg<T>::value;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // shared layout: sc[NS][kChunkPts] T2 | sval[w][kValStride] T | srel[kChunkPts] int |
    //                cnt[HN] int | start[HN+1] int | warp_tot[8] int
    const int w = a.w;
    T2* sc = reinterpret_cast<T2*>(smem_raw);
    T* sval = reinterpret_cast<T*>(sc + NS * kChunkPts);
    int* srel = reinterpret_cast<int*>(sval + w * kValStride);
    const int HN = a.L + w;                         // keys rel + (w-1) in [0, L + w - 1)
    int* cnt = srel + kChunkPts;
    int* start = cnt + HN;
    int* warp_tot = start + HN + 1;

    // Work items.  cuFFT path: one CTA per (tile, row group), tiles visited in a permuted order so that occupied
    // tiles (compute/latency-bound) and empty tiles (pure streaming stores of zeros) interleave on every SM.
    // Own-FFT path: empty tiles do not exist; a persistent grid walks the (listed tile, row group) pairs.
    // Persistent order: the x1 items first (two transforms and, at the same point density, twice the
    // candidates per tile: longest first shortens the tail), then the x2 items.
    int n1 = 0, nitems = 1;
    if (a.skip_empty) {
        n1 = __ldg(&a.tile_counts[1]) * a.seg[1].ngroups;
        nitems = n1 + __ldg(&a.tile_counts[0]) * a.seg[0].ngroups;
    }
    const int lbase = threadIdx.x * CPT;             // first owned cell, tile-relative
    // Two-deep prefetch down the item list: the tile id of item i + 2G and the candidate ranges of item
    // i + G are requested while item i is processed, so neither dependent load sits on the critical path.
    auto item_tile = [&](int it) -> int {
        if (it >= nitems) return 0;
        const int s_ = it < n1 ? 1 : 0, e = s_ ? it : it - n1;
        return __ldg(&a.tile_list[s_ * a.ntiles + e / a.seg[s_].ngroups]);
    };
    struct Cand { int pbeg0, pcnt0, pbeg1, pcnt1, pcnt2, total; };
    auto item_cand = [&](int it, int tl) -> Cand {
        Cand c{0, 0, 0, 0, 0, 0};
        if (it < nitems) {
            const int tlo = tl * a.L;
            c.total = tile_candidates(a.seg[it < n1 ? 1 : 0].bin_start, a.n, a.nbins, a.H, tlo, min(a.L, a.n - tlo),
                                      c.pbeg0, c.pcnt0, c.pbeg1, c.pcnt1, c.pcnt2);
        }
        return c;
    };
    int tile_cur = 0, tile_nx = 0;
    bool cnt_clean = false;
    Cand cand_cur{0, 0, 0, 0, 0, 0};
    if (a.skip_empty) {
        tile_cur = item_tile(blockIdx.x);
        tile_nx = item_tile(blockIdx.x + gridDim.x);
        cand_cur = item_cand(blockIdx.x, tile_cur);
    }
    for (int item = blockIdx.x; item < nitems || !a.skip_empty; item += gridDim.x) {
    int tile, si, grp;
    int pbeg0, pcnt0, pbeg1, pcnt1, pcnt2, total;
    int tile_nx2 = 0;
    Cand cand_nx{0, 0, 0, 0, 0, 0};
    if (a.skip_empty) {
        si = item < n1 ? 1 : 0;
        grp = (si ? item : item - n1) % a.seg[si].ngroups;
        tile = tile_cur;
        pbeg0 = cand_cur.pbeg0; pcnt0 = cand_cur.pcnt0; pbeg1 = cand_cur.pbeg1; pcnt1 = cand_cur.pcnt1;
        pcnt2 = cand_cur.pcnt2; total = cand_cur.total;
        tile_nx2 = item_tile(item + 2 * gridDim.x);
        cand_nx = item_cand(item + gridDim.x, tile_nx);
    } else {
        if (item != (int)blockIdx.x) break;          // one item per CTA
        if (a.tile_mask >= 0) tile = (int)((blockIdx.x * (unsigned)a.tile_stride) & (unsigned)a.tile_mask);
        else if (a.ntiles <= 65535) tile = (int)((blockIdx.x * (unsigned)a.tile_stride) % (unsigned)a.ntiles);
        else tile = (int)(((long long)blockIdx.x * a.tile_stride) % a.ntiles);
        si = (int)blockIdx.y < a.seg[0].ngroups ? 0 : 1;
        grp = (int)blockIdx.y - (si ? a.seg[0].ngroups : 0);
        const int tlo = tile * a.L;
        total = tile_candidates(a.seg[si].bin_start, a.n, a.nbins, a.H, tlo, min(a.L, a.n - tlo), pbeg0, pcnt0, pbeg1,
                                pcnt1, pcnt2);
    }
    const SpreadSeg<T>& sg = a.seg[si];
    const int row0 = grp * NS;
    const int nr = min(NS, sg.nrows - row0);
    const int tile_lo = tile * a.L;
    const int Lt = min(a.L, a.n - tile_lo);

    T2 acc[NS][CPT];
#pragma unroll
    for (int s = 0; s < NS; ++s)
#pragma unroll
        for (int c = 0; c < CPT; ++c) acc[s][c].x = acc[s][c].y = (T)0;

    for (int base = 0; base < total; base += kChunkPts) {
        // ---- 1. one candidate per thread: its record and strengths (loads issued before the barrier)
        bool have = false;
        int rel = 0;
        T eta = (T)0, qx = (T)0, qy = (T)0, r[NS];
#pragma unroll
        for (int s = 0; s < NS; ++s) r[s] = (T)0;
        {
            int ci = base + threadIdx.x;
            if (ci < total) {
                int g = pbeg0 + ci, shift = 0;
                if (ci >= pcnt0) {
                    ci -= pcnt0;
                    if (ci < pcnt1) { g = pbeg1 + ci; shift = -a.n; }
                    else { g = ci - pcnt1; shift = a.n; }
                }
                int l0;
                load_rec(sg.rec + g, eta, l0, qx, qy);
                // strengths are fetched with the record, not after it: one global round trip, not two
#pragma unroll
                for (int s = 0; s < NS; ++s)
                    if (s < nr) {
                        const int lr = sg.first_row + row0 + s;
                        r[s] = (a.w_implicit && lr == 0) ? (T)1 : __ldg(&sg.rows[(long long)(lr - a.w_implicit) * a.Nd + g]);
                    }
                rel = l0 + shift - tile_lo;          // first touched cell, tile-relative
                have = rel + w > 0 && rel < Lt;
            }
        }
        if (!cnt_clean) {                            // later chunks, and later tiles of a persistent CTA, find cnt
            for (int i = threadIdx.x; i < HN; i += kSpreadThreads) cnt[i] = 0;   // re-zeroed by the scan
            __syncthreads();
            cnt_clean = true;
        }
        // key = first-touched cell + (w - 1); rank = arrival order among equal keys
        const int key = rel + w - 1;
        int rank = 0;
        if (have) rank = atomicAdd(&cnt[key], 1);
        __syncthreads();
        // ---- 2. exclusive scan of the per-cell counts (re-zeroes cnt for the next chunk)
        block_scan_counts(cnt, start, HN, warp_tot);
        __syncthreads();
        // ---- 3. stage the candidate at its cell-ordered slot: strengths and w kernel values
        if (have) {
            const int slot = start[key] + rank;
            srel[slot] = rel;
#pragma unroll
            for (int s = 0; s < NS; ++s) {
                T2 cc;
                cc.x = qx * r[s];
                cc.y = qy * r[s];
                sc[s * kChunkPts + slot] = cc;
            }
            const T z2 = eta * eta;
#pragma unroll
            for (int i = 0; i < kHalfMax; ++i) {
                if (i < a.half) {                    // warp-uniform; coefficients are constant-bank operands
                    T e = a.c[i][DEG], o = a.c[i][DEG - 1];
#pragma unroll
                    for (int d = DEG - 2; d >= 2; d -= 2) {
                        e = fma(e, z2, a.c[i][d]);
                        o = fma(o, z2, a.c[i][d - 1]);
                    }
                    e = fma(e, z2, a.c[i][0]);
                    o *= eta;
                    sval[i * kValStride + slot] = e + o;             // psi at cell l0 + i
                    sval[(w - 1 - i) * kValStride + slot] = e - o;   // psi at cell l0 + w-1-i (even symmetry)
                }
            }
        }
        __syncthreads();
        // ---- 4. gather: cell l receives every point with rel in [l - w + 1, l], i.e. key in [l, l + w)
        if (lbase < Lt) {
            const int pb = start[lbase], pe = start[lbase + CPT - 1 + w];
            // the x2 group of a single series carries one live row: skip the dead half of the FMAs
            if (NS > 1 && nr == 1) gather_cells<T, 1, NS, CPT>(acc, sc, sval, srel, pb, pe, lbase, w);
            else gather_cells<T, NS, NS, CPT>(acc, sc, sval, srel, pb, pe, lbase, w);
        }
        if (base + kChunkPts < total) __syncthreads();   // staging area is reused by the next chunk
    }

    // ---- 5. the tile is written exactly once
    if (lbase < Lt) {
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            if (s < nr) {
                T2* out = sg.grid + (long long)(row0 + s) * a.n + tile_lo + lbase;
                if (lbase + CPT <= Lt) {
                    store_cells<CPT>(out, acc[s]);
                } else {
#pragma unroll
                    for (int c = 0; c < CPT; ++c)
                        if (lbase + c < Lt) out[c] = acc[s][c];
                }
            }
        }
    }
    tile_cur = tile_nx;
    tile_nx = tile_nx2;
    cand_cur = cand_nx;
    }   // work items (the next item's first barrier orders its shared-memory writes after this item's reads)
}

template <typename T, int NS>
size_t spread_smem_bytes(int L, int w) {
    const int HN = L + w;
    return sizeof(typename V2<T>::type) * NS * kChunkPts + sizeof(T) * (size_t)w * kValStride + sizeof(int) * kChunkPts +
           sizeof(int) * (HN + HN + 1 + 8);
}

template <typename T, int NS, int CPT>
cudaError_t launch_inst(ls_plan_s* p, const SpreadArgs<T>& a, cudaStream_t s) {
    static bool configured[64] = {false};          // per device: the attribute belongs to the device's function
    const int dev = p->opts.device & 63;
    if (!configured[dev]) {
        cudaError_t e = cudaFuncSetAttribute(ls_spread_tile_kernel<T, NS, CPT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)spread_smem_bytes<T, NS>(kSpreadThreads * CPT, kMaxWidth));
        if (e != cudaSuccess) return e;
        configured[dev] = true;
    }
    dim3 grid(p->ntiles, a.seg[0].ngroups + a.seg[1].ngroups);
    if (a.skip_empty) {                              // persistent: as many CTAs as fit, never more than the work
        const long long items = (long long)p->ntiles * (a.seg[0].ngroups + a.seg[1].ngroups);
        grid = dim3((unsigned)std::min<long long>(items, (long long)p->num_sms * ((NS * CPT <= 8) ? 4 : 3)));
    }
    ls_spread_tile_kernel<T, NS, CPT><<<grid, kSpreadThreads, spread_smem_bytes<T, NS>(p->L, p->w), s>>>(a);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_t(ls_plan_s* p, int row0_x2, int nrows_x2, int slot0_x2, int row0_x1, int nrows_x1, int slot0_x1,
                     cudaStream_t s) {
    using T2 = typename V2<T>::type;
    using R = typename RecOf<T>::type;
    const int NS = spread_rows_per_group(p);
    SpreadArgs<T> a;
    a.n = (int)p->n;
    a.L = p->L;
    a.nbins = p->nbins;
    a.w = p->w;
    a.H = (p->w + 1) / 2;
    a.ntiles = p->ntiles;
    a.tile_stride = p->tile_stride;
    a.tile_mask = (p->ntiles & (p->ntiles - 1)) == 0 ? p->ntiles - 1 : -1;
    a.half = p->poly.half;
    a.skip_empty = (p->fft_prune || p->list_tiles) ? 1 : 0;
    a.row_masks = p->row_masks;
    a.tile_list = p->tile_list;
    a.w_implicit = p->opts.dy_per_series ? 0 : 1;
    a.tile_counts = p->tile_counts;
    a.ncoltiles = own_fft_ncoltiles(p);
    a.fft_rb = p->fft_prune ? own_fft_rb(p) : 1;
    a.coltile_shift = 0;
    while ((1 << a.coltile_shift) < a.ncoltiles) ++a.coltile_shift;
    a.Nd = p->Nd;
    for (int i = 0; i < kHalfMax; ++i)
        for (int d = 0; d <= kMaxDeg; ++d) a.c[i][d] = (T)p->poly.c[i][d];
    const int row0[2] = {row0_x2, row0_x1}, nrows[2] = {nrows_x2, nrows_x1}, slot0[2] = {slot0_x2, slot0_x1};
    for (int g = 0; g < 2; ++g) {
        const PointSet& ps = p->ps[g == 0 ? 1 : 0];
        a.seg[g].bin_start = ps.bin_start;
        a.seg[g].rec = (const R*)ps.rec;
        a.seg[g].rows = (const T*)ps.rows;
        a.seg[g].first_row = row0[g];
        a.seg[g].grid = (T2*)p->grids + (long long)slot0[g] * p->n;
        a.seg[g].nrows = nrows[g];
        a.seg[g].ngroups = (nrows[g] + NS - 1) / NS;
    }
    const int cpt = p->L / kSpreadThreads;
    if (NS == 2) {
        if (cpt == 4) return launch_inst<T, 2, 4>(p, a, s);
        if (cpt == 2) return launch_inst<T, 2, 2>(p, a, s);
        return launch_inst<T, 2, 1>(p, a, s);
    }
    if (cpt == 2) return launch_inst<T, 4, 2>(p, a, s);
    return launch_inst<T, 4, 1>(p, a, s);
}

}  // namespace

// Own-FFT path, once per execute after the bin scan: occupied-tile lists and liveness masks of both point sets.
cudaError_t launch_tile_list(ls_plan_s* p, cudaStream_t s) {
    const int ncol = own_fft_ncoltiles(p);
    int shift = 0;
    while ((1 << shift) < ncol) ++shift;
    const int total = 2 * p->ntiles;
    ls_tile_list_kernel<<<(total + 255) / 256, 256, 0, s>>>(p->ps[1].bin_start, p->ps[0].bin_start, (int)p->n, p->nbins,
                                                           (p->w + 1) / 2, p->L, p->ntiles, p->tile_list, p->tile_counts,
                                                           p->row_masks, ncol, shift, own_fft_rb(p));
    return cudaGetLastError();
}

// cuFFT path, before every spreading launch: zeros into the tiles without points, occupied tiles into the lists.
cudaError_t launch_zero_list(ls_plan_s* p, int nrows_x2, int slot0_x2, int nrows_x1, int slot0_x1, int build_list, cudaStream_t s) {
    const int nchunks = (2 * p->ntiles + 255) / 256;
    const int nbx = std::min(nchunks, 8 * p->num_sms);
    const int rows = std::max(nrows_x2, nrows_x1);
    const dim3 nblk(nbx, (unsigned)std::max(1, std::min(rows, (8 * p->num_sms + nbx - 1) / nbx)));
    const int H = (p->w + 1) / 2;
    if (p->dtype == LS_F64) {
        double2* g = (double2*)p->grids;
        ls_tile_zero_list_kernel<double2><<<nblk, 256, 0, s>>>(p->ps[1].bin_start, p->ps[0].bin_start, (int)p->n, p->nbins, H, p->L,
                                                               p->ntiles, p->tile_list, p->tile_counts, build_list,
                                                               g + (long long)slot0_x2 * p->n, nrows_x2, g + (long long)slot0_x1 * p->n, nrows_x1);
    } else {
        float2* g = (float2*)p->grids;
        ls_tile_zero_list_kernel<float2><<<nblk, 256, 0, s>>>(p->ps[1].bin_start, p->ps[0].bin_start, (int)p->n, p->nbins, H, p->L,
                                                              p->ntiles, p->tile_list, p->tile_counts, build_list,
                                                              g + (long long)slot0_x2 * p->n, nrows_x2, g + (long long)slot0_x1 * p->n, nrows_x1);
    }
    return cudaGetLastError();
}

// Transforms accumulated per CTA: 2 for a single series ({w, h} at x1), 4 for a batch.
int spread_rows_per_group(const ls_plan_s* p) { return p->batch == 1 ? 2 : 4; }

cudaError_t launch_spread(ls_plan_s* p, int row0_x2, int nrows_x2, int slot0_x2, int row0_x1, int nrows_x1,
                          int slot0_x1, cudaStream_t s) {
    if (nrows_x2 <= 0 && nrows_x1 <= 0) return cudaSuccess;
    return p->dtype == LS_F64 ? launch_t<double>(p, row0_x2, nrows_x2, slot0_x2, row0_x1, nrows_x1, slot0_x1, s)
                              : launch_t<float>(p, row0_x2, nrows_x2, slot0_x2, row0_x1, nrows_x1, slot0_x1, s);
}

}  // namespace lsb
