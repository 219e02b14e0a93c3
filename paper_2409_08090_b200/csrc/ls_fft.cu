// ls_fft.cu — the library's own fine-grid FFT for complex128 grids of n = 2^12 .. 2^24 cells (
// PAPER.md:47 "use an equispaced FFT", :73 "the FFT time dominates").
//
//   B_k = sum_l b_l e^{+2 pi i k l / n}     (reading A7: the unnormalised inverse transform)
//
// Three passes over n = R1 R2 R3, R2 = R3 = 256, R1 = n / 2^16 = 2 .. 256 (256^3 at the headline size; two passes
// R1 x 256 for n <= 2^16), decimation in frequency:
//   l = l1 R2 R3 + l2 R3 + l3,   k = k1 + R1 k2 + R1 R2 k3
//   pass 1: FFT over l1 -> k1, times w_n^{k1 (l2 R3 + l3)};   in place, layout [k1][l2][l3]
//   pass 2: FFT over l2 -> k2, times w_n^{R1 k2 l3};          in place, layout [k1][k2][l3]
//   pass 3: FFT over l3 -> k3; the kept modes k' = k - floor(Nf/2) in [-floor(Nf/2), ceil(Nf/2)) go to a
//           compact [M][Nf] array in frequency order (coalesced: 16 consecutive k1 per store)
// This is the pass structure cuFFT itself uses at this size (three regular_fft_factor<256> launches,
// profiles/r1c_cfg3.md); what the own version adds is what a library cannot know:
//   * pass 1 skips the loads of tiles the spreading kernel flagged empty (60-80 % of every grid at
//     df = 1/(5T)), and the spreading kernel no longer has to write those zeros;
//   * pass 3 writes only the N_f kept modes, already centred, so the assembly reads a dense array.
//
// One CTA = 256 threads = one tile of 256 (transform dimension) x 16 (other dimension) points (pass 1 and the fused
// passes 2 + 3: 128 threads, 256 x 8):
// 16-point FFTs in registers (radix 4 x 4), one shared-memory exchange (conflict-free layouts),
// 256-byte global segments on both sides.  Twiddles: w_256 from a shared table, w_n^e from two
// 4096-entry tables (e = 4096 e_hi + e_lo) and a base/step recurrence along the thread's 16 outputs.
#include <cuda.h>            // CUtensorMap (types only: the encoder is fetched through the runtime, no libcuda link)

#include "ls_internal.h"
#include "ls_power.cuh"

namespace lsb {
namespace {

constexpr int kC = 16;                   // columns (passes 1, 2) / rows (pass 3) of a CTA's tile
constexpr int kFftThreads = 16 * kC;
constexpr double kC1 = 0.92387953251128675613;   // cos(pi/8)
constexpr double kS1 = 0.38268343236508977173;   // sin(pi/8)
constexpr double kR2 = 0.70710678118654752440;   // sqrt(1/2)

__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 cmul(double2 a, double2 w) {
    return make_double2(fma(a.x, w.x, -a.y * w.y), fma(a.x, w.y, a.y * w.x));
}
__device__ __forceinline__ double2 cmuli(double2 a) { return make_double2(-a.y, a.x); }   // a * i

// X_k = sum_l x_l e^{+2 pi i k l / 4}, in place (a,b,c,d) -> (X0,X1,X2,X3)
__device__ __forceinline__ void fft4(double2& a, double2& b, double2& c, double2& d) {
    const double2 t0 = cadd(a, c), t1 = csub(a, c), t2 = cadd(b, d), t3 = cmuli(csub(b, d));
    a = cadd(t0, t2);
    b = cadd(t1, t3);
    c = csub(t0, t2);
    d = csub(t1, t3);
}

// 16-point transform X_k = sum_l x_l e^{+2 pi i k l / 16}, in place; X_k ends at position
// pos16(k) = 4 (k & 3) + (k >> 2).
__device__ __forceinline__ constexpr int pos16(int k) { return 4 * (k & 3) + (k >> 2); }
__device__ __forceinline__ void fft16(double2 (&x)[16]) {
#pragma unroll
    for (int b = 0; b < 4; ++b) fft4(x[b], x[4 + b], x[8 + b], x[12 + b]);     // over a: x[4 ka + b] = z[b][ka]
    // twiddle w_16^{b ka}
    x[5] = cmul(x[5], make_double2(kC1, kS1));       // b=1, ka=1: m=1
    x[6] = cmul(x[6], make_double2(kR2, kR2));       // b=2, ka=1: m=2
    x[7] = cmul(x[7], make_double2(kS1, kC1));       // b=3, ka=1: m=3
    x[9] = cmul(x[9], make_double2(kR2, kR2));       // b=1, ka=2: m=2
    x[10] = cmuli(x[10]);                            // b=2, ka=2: m=4
    x[11] = cmul(x[11], make_double2(-kR2, kR2));    // b=3, ka=2: m=6
    x[13] = cmul(x[13], make_double2(kS1, kC1));     // b=1, ka=3: m=3
    x[14] = cmul(x[14], make_double2(-kR2, kR2));    // b=2, ka=3: m=6
    x[15] = cmul(x[15], make_double2(-kC1, -kS1));   // b=3, ka=3: m=9
#pragma unroll
    for (int ka = 0; ka < 4; ++ka) fft4(x[4 * ka], x[4 * ka + 1], x[4 * ka + 2], x[4 * ka + 3]);
}

// 8-point transform (two fft4 on the even / odd samples, then a radix-2 layer); X_k ends at position
// pos8(k) = 2 (k & 3) + (k >> 2).
__device__ __forceinline__ void fft8(double2 (&x)[8]) {
    fft4(x[0], x[2], x[4], x[6]);
    fft4(x[1], x[3], x[5], x[7]);
    x[3] = cmul(x[3], make_double2(kR2, kR2));       // w_8^1
    x[5] = cmuli(x[5]);                              // w_8^2
    x[7] = cmul(x[7], make_double2(-kR2, kR2));      // w_8^3
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const double2 e = x[2 * k], o = x[2 * k + 1];
        x[2 * k] = cadd(e, o);
        x[2 * k + 1] = csub(e, o);
    }
}
// RB-point transform, RB in {1, 2, 4, 8, 16}: in place, X_k at position fft_pos<RB>(k).
template <int RB>
__device__ __forceinline__ constexpr int fft_pos(int k) {
    return RB == 16 ? 4 * (k & 3) + (k >> 2) : RB == 8 ? 2 * (k & 3) + (k >> 2) : k;
}
template <int RB>
__device__ __forceinline__ void fft_small(double2 (&x)[RB]) {
    if constexpr (RB == 16) fft16(x);
    else if constexpr (RB == 8) fft8(x);
    else if constexpr (RB == 4) fft4(x[0], x[1], x[2], x[3]);
    else if constexpr (RB == 2) {
        const double2 a = x[0], b = x[1];
        x[0] = cadd(a, b);
        x[1] = csub(a, b);
    }
}

struct FftArgs {
    double2* grids;            // [ntrans][n] in place
    long long n;
    int R1, R2, R3;            // n = R1 R2 R3; R3 = 256; R2 = 256 (three passes) or 1 (two passes); R1 a power of two
    int R1_shift;              // log2(R1)
    const double2* wlo;        // w_n^x, x < 4096
    const double2* whi;        // w_n^{4096 y}, y < n / 4096
    // pass 1 pruning (see PointSet-independent `row_masks` in ls_internal.h): for point set s, spreading-tile
    // column ct = (m >> tile_shift) and j = row % RB (RB = R1/16), bit i of row_masks[(s * ncoltiles + ct) * RB + j]
    // says that row RB i + j of that column holds data; unset = never written by the spreading kernel = zeros.
    const unsigned* row_masks;
    int ncoltiles;
    int set_of_trans_first;    // transforms [0, set_of_trans_first) belong to set 0 (x2), the rest to set 1 (x1)
    int tile_shift;            // log2(spreading tile length)
    // pass 3 output
    double2* modes;            // [ntrans][Nf]
    long long Nf, half;
    // pass 3 fused with deconvolution + assembly (K5 + K6): transform i of the launch is h of series
    // series0 + i; the (w, w2) modes are read from the compact array
    const double2* w_modes;    // [Nf] modes of w at x1
    const double2* w2_modes;   // [Nf] modes of w at x2
    const double2* ftab;       // [Nf][2] per-frequency terms of the fused assembly: (d Cw, d Sw), (1/CC, 1/SS)
    const double* dinv;        // 1 / psihat(|k'|)
    const double* sums;        // [batch][4]: YY at [4 s + 2]
    double* power;             // [batch][Nf]
    int series0;
    int no_float, norm;        // opts.no_floating_mean, opts.normalization
};

__device__ __forceinline__ double2 twiddle_n(const FftArgs& a, unsigned e) {
    const double2 lo = __ldg(&a.wlo[e & 4095u]);
    const double2 hi = __ldg(&a.whi[(e & (unsigned)(a.n - 1)) >> 12]);
    return cmul(lo, hi);
}

// Second-stage outputs k_r = ka + 16 kb, kb < NOUT, times the inter-pass twiddle tw st^kb, stored `stride` cells apart.
// For NOUT = 16 the twiddles come from TWO interleaved recurrences (even / odd kb, step st^2): these kernels are latency-bound, and
// a single chain of NOUT dependent complex products is what the stores end up waiting for (fused passes 2 + 3 at
// config 3: 0.416 -> 0.407 ms; four chains spill at the 128-register cap: 0.425 ms).
template <int NOUT, typename Get>
__device__ __forceinline__ void store_twiddled(double2* base, long long stride, int ka, double2 tw, double2 st, Get get) {
    if constexpr (NOUT == 16) {                              // shorter chains keep the single recurrence
        double2 tw1 = cmul(tw, st);
        const double2 st2 = cmul(st, st);
#pragma unroll
        for (int kb = 0; kb < NOUT; kb += 2) {
            base[(long long)(ka + 16 * kb) * stride] = cmul(get(kb), tw);
            base[(long long)(ka + 16 * kb + 16) * stride] = cmul(get(kb + 1), tw1);
            if (kb + 2 < NOUT) {
                tw = cmul(tw, st2);
                tw1 = cmul(tw1, st2);
            }
        }
    } else {
#pragma unroll
        for (int kb = 0; kb < NOUT; ++kb) {
            base[(long long)(ka + 16 * kb) * stride] = cmul(get(kb), tw);
            tw = cmul(tw, st);
        }
    }
}

// Exchange twiddles in shared memory, stored as [ka][j] = w_256^{j ka} (j, ka < 16) rather than as a w_256^m table:
// the threads of a warp that differ in j read consecutive entries (no bank conflicts; with an m-indexed table the
// lookups of ka = 8 were 16-way conflicts in pass 3), threads that share j read the same entry (broadcast).
// Passes 2 + 3 at config 3: 0.441 -> 0.430 ms.
__device__ __forceinline__ void fill_w256(double2* w256, int nthreads = kFftThreads) {
    for (int i = threadIdx.x; i < 256; i += nthreads) {
        double s, c;
        sincospi((double)((i >> 4) * (i & 15)) / 128.0, &s, &c);
        w256[i] = make_double2(c, s);
    }
}
// the plain table w_256^m, m < 256 (pass 1: two values of j per warp, nothing to gain from the layout above; measured
// 2 % slower with it)
__device__ __forceinline__ void fill_w256_linear(double2* w256, int nthreads) {
    for (int i = threadIdx.x; i < 256; i += nthreads) {
        double s, c;
        sincospi((double)i / 128.0, &s, &c);
        w256[i] = make_double2(c, s);
    }
}

// Passes 1 and 2: the transform dimension is strided (stride = inner), 16 consecutive columns per CTA.
// Data viewed as [outer][256][inner]; in place.  Inter-pass twiddle w_n^{k_r * m * outer}.
__global__ void __launch_bounds__(kFftThreads, 512 / kFftThreads)
ls_fft_cols_kernel(const FftArgs a, int outer, long long inner) {
    extern __shared__ __align__(16) unsigned char fsm[];
    double2* Y = reinterpret_cast<double2*>(fsm);            // [ka][j][c]
    double2* w256 = Y + 256 * kC;
    fill_w256(w256);
    const int c = threadIdx.x % kC, hi4 = threadIdx.x / kC;
    const long long m = (long long)blockIdx.x * kC + c;      // column
    const int o = blockIdx.y, tr = blockIdx.z;
    double2* base = a.grids + (long long)tr * a.n + (long long)o * 256 * inner + m;

    double2 x[16];
    {
        const int j = hi4;
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = base[(long long)(16 * i + j) * inner];
        fft16(x);
        __syncthreads();                                     // w256 ready
#pragma unroll
        for (int ka = 0; ka < 16; ++ka) Y[(ka * 16 + j) * kC + c] = cmul(x[pos16(ka)], w256[ka * 16 + j]);
    }
    __syncthreads();
    {
        const int ka = hi4;
#pragma unroll
        for (int j = 0; j < 16; ++j) x[j] = Y[(ka * 16 + j) * kC + c];
        fft16(x);
        // k_r = ka + 16 kb;  twiddle exponent e = k_r * m * outer (mod n) = e0 + kb * de
        // (requesting the tables before the exchange, as pass 1 does, costs this DRAM-bound pass registers: slower)
        const unsigned mm = (unsigned)m * (unsigned)outer;
        const double2 tw = twiddle_n(a, (unsigned)ka * mm);
        const double2 st = twiddle_n(a, 16u * mm);
        store_twiddled<16>(base, inner, ka, tw, st, [&](int kb) { return x[pos16(kb)]; });
    }
}

// Pass 1, pruned and persistent: radix R1 = 16 RB over l1 (row stride inner = 65536 cells), C = T / RB
// columns per tile, so a tile is always 16 T points (T = 128 threads: 2048 points, four CTAs per SM).  Stage 1: 16-point FFTs over i (rows
// RB i + j); stage 2: RB-point FFTs over j.  The 16-bit liveness mask of the NEXT tile is fetched while the
// current one is in flight, so it never sits on the critical path; dead rows are not loaded (never written).
template <int RB, int T>
__global__ void __launch_bounds__(T, 512 / T)
ls_fft_pass1_kernel(const FftArgs a, long long inner, int tiles_per_trans, int ntiles_total) {
    constexpr int C = T / RB, NI = 16 / RB, TWS = 16 / RB;     // TWS: stride of w_{R1} in the w_256 table
    extern __shared__ __align__(16) unsigned char fsm[];
    double2* Y = reinterpret_cast<double2*>(fsm);            // [ka][j][c]
    double2* w256 = Y + 16 * T;
    fill_w256_linear(w256, T);
    const int c = threadIdx.x % C, hi = threadIdx.x / C;     // hi: j in stage 1, item group in stage 2
    auto mask_of = [&](int tile) -> unsigned {
        if (tile >= ntiles_total) return 0u;
        if (a.row_masks == nullptr) return 0xffffu;          // unpruned: every row was written
        const int tr = tile / tiles_per_trans;
        const long long m0 = (long long)(tile - tr * tiles_per_trans) * C;
        const int set = tr < a.set_of_trans_first ? 0 : 1;
        return __ldg(&a.row_masks[((long long)set * a.ncoltiles + (m0 >> a.tile_shift)) * RB + hi]);
    };
    int tile = blockIdx.x;
    unsigned live = mask_of(tile);
    __syncthreads();                                         // w256 ready
    for (; tile < ntiles_total; tile += gridDim.x) {
        const int tr = tile / tiles_per_trans;
        const long long m = (long long)(tile - tr * tiles_per_trans) * C + c;
        double2* base = a.grids + (long long)tr * a.n + m;
        // the table loads of the inter-pass twiddles are requested with the data, not after the exchange
        const unsigned mm = (unsigned)m;
        const double2 st = twiddle_n(a, 16u * mm);
        const double2 tw0 = twiddle_n(a, (unsigned)(hi * NI) * mm);
        {
            const int j = hi;
            double2 x[16];
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                x[i] = make_double2(0.0, 0.0);
                if (live >> i & 1u) x[i] = base[(long long)(RB * i + j) * inner];
            }
            live = mask_of(tile + gridDim.x);                // prefetch: lands during this tile's work
            fft16(x);
#pragma unroll
            for (int ka = 0; ka < 16; ++ka)
                Y[(ka * RB + j) * C + c] = cmul(x[pos16(ka)], w256[(j * ka * TWS) & 255]);
        }
        __syncthreads();
        {
#pragma unroll
            for (int q = 0; q < NI; ++q) {
                const int ka = hi * NI + q;
                double2 y[RB];
#pragma unroll
                for (int j = 0; j < RB; ++j) y[j] = Y[(ka * RB + j) * C + c];
                fft_small<RB>(y);
                // k1 = ka + 16 kb;  twiddle exponent k1 * m = ka m + kb (16 m)
                const double2 tw = q == 0 ? tw0 : twiddle_n(a, (unsigned)ka * mm);
                store_twiddled<RB>(base, inner, ka, tw, st, [&](int kb) { return y[fft_pos<RB>(kb)]; });
            }
        }
        __syncthreads();                                     // Y is reused by the next tile
    }
}

// First pass for n = 2^17 .. 2^19 (R1 = 2, 4, 8 rows of 65536 cells): one thread per column, R1-point FFT in
// registers, times w_n^{k1 m}; in place.  Memory-bound by construction.
template <int R>
__global__ void __launch_bounds__(256)
ls_fft_pass1_small_kernel(const FftArgs a, long long inner) {
    const int tr = blockIdx.y;
    double2* base = a.grids + (long long)tr * a.n;
    for (long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x; m < inner; m += (long long)gridDim.x * blockDim.x) {
        double2 x[R];
#pragma unroll
        for (int i = 0; i < R; ++i) x[i] = base[(long long)i * inner + m];
        fft_small<R>(x);
#pragma unroll
        for (int k1 = 0; k1 < R; ++k1) {
            double2 v = x[fft_pos<R>(k1)];
            if (k1 > 0) v = cmul(v, twiddle_n(a, (unsigned)k1 * (unsigned)m));
            base[(long long)k1 * inner + m] = v;
        }
    }
}

// First pass for n = 5 * 2^k cells, two passes R1 x 256 with R1 = 80 RM rows (RM = 2, 4, 8, 16: n = 40 960 .. 327 680):
// the sizes that sit halfway between the powers of two (sigma = n / Nf in [1.25, 1.77) where the power of two has
// [1.77, 2.5): a batch of small grids moves 1.6 x fewer bytes).  R1 = 16 x RM x 5, decimation in frequency, J = 5 RM:
//   l1 = J i + j,  j = 5 p + q          (i < 16, p < RM, q < 5)
//   k1 = ka + 16 (kp + RM kq)           (ka < 16, kp < RM, kq < 5)
//   stage 1: 16-point FFTs over i -> ka, times w_R1^{ka j};      one per thread (J threads per column)
//   stage 2: RM-point FFTs over p -> kp, times w_R1^{16 kp q};   80 per column
//   stage 3: 5-point FFTs over q -> kq, times the inter-pass twiddle w_n^{k1 m};  16 RM per column
// The column tile (R1 rows x 8 columns) lives in shared memory between the stages ([ka][j][c], 128-byte rows: every
// access of a quarter warp is one row, conflict-free); 128-byte global segments on both sides, in place.
constexpr int kC5 = 8;                   // columns per CTA
constexpr double kCos5a = 0.30901699437494742410;    // cos(2 pi / 5)
constexpr double kCos5b = -0.80901699437494742410;   // cos(4 pi / 5)
constexpr double kSin5a = 0.95105651629515357212;    // sin(2 pi / 5)
constexpr double kSin5b = 0.58778525229247312917;    // sin(4 pi / 5)
// X_k = sum_l x_l e^{+2 pi i k l / 5}, in place, natural order
__device__ __forceinline__ void fft5(double2 (&x)[5]) {
    const double2 t1 = cadd(x[1], x[4]), t2 = cadd(x[2], x[3]), t3 = csub(x[1], x[4]), t4 = csub(x[2], x[3]);
    const double2 a1 = make_double2(x[0].x + kCos5a * t1.x + kCos5b * t2.x, x[0].y + kCos5a * t1.y + kCos5b * t2.y);
    const double2 a2 = make_double2(x[0].x + kCos5b * t1.x + kCos5a * t2.x, x[0].y + kCos5b * t1.y + kCos5a * t2.y);
    const double2 b1 = make_double2(kSin5a * t3.x + kSin5b * t4.x, kSin5a * t3.y + kSin5b * t4.y);
    const double2 b2 = make_double2(kSin5b * t3.x - kSin5a * t4.x, kSin5b * t3.y - kSin5a * t4.y);
    x[0] = make_double2(x[0].x + t1.x + t2.x, x[0].y + t1.y + t2.y);
    x[1] = make_double2(a1.x - b1.y, a1.y + b1.x);      // a1 + i b1
    x[4] = make_double2(a1.x + b1.y, a1.y - b1.x);      // a1 - i b1
    x[2] = make_double2(a2.x - b2.y, a2.y + b2.x);
    x[3] = make_double2(a2.x + b2.y, a2.y - b2.x);
}
// Stage-2 twiddles w_{5 RM}^{kp q}: kp is unrolled and q = b >> 4 is the same for the 32 threads of a warp (b = tj + J r,
// four consecutive tj per warp, aligned to four), so they are warp-uniform constant-bank reads — no load/store unit
// work in a kernel that is bound by it.  [log2 RM - 1][q][kp], filled by own_fft_init.
__constant__ double2 cTw5[4][5][16];
template <int RM>
constexpr size_t cols5_smem() { return sizeof(double2) * ((size_t)(80 * RM) * (kC5 + 1) + 2 * kC5); }   // tile + w_R1 table + column steps
template <int RM>
__global__ void __launch_bounds__(5 * RM * kC5, 16 / RM)      // 640 threads per SM: two CTAs at RM = 8 need <= 102 registers
ls_fft_cols5_kernel(const FftArgs a) {
    constexpr int J = 5 * RM, R1 = 16 * J;
    extern __shared__ __align__(16) unsigned char fsm[];
    double2* S = reinterpret_cast<double2*>(fsm);            // [ka][j][c]
    double2* wr = S + R1 * kC5;                              // w_R1^x, x < R1
    for (int x = threadIdx.x; x < R1; x += J * kC5) {
        double sn, cs;
        sincospi(2.0 * (double)x / (double)R1, &sn, &cs);
        wr[x] = make_double2(cs, sn);
    }
    double2* colw = wr + R1;                                 // [2][kC5]: w_n^{J m}, w_n^{16 RM m} of the CTA's columns
    if (threadIdx.x < 2 * kC5) {
        const unsigned e = (unsigned)(threadIdx.x < kC5 ? J : 16 * RM) * (unsigned)(blockIdx.x * kC5 + threadIdx.x % kC5);
        colw[threadIdx.x] = cmul(__ldg(&a.wlo[e & 4095u]), __ldg(&a.whi[e >> 12]));
    }
    const int c = threadIdx.x % kC5, tj = threadIdx.x / kC5;
    const int m = blockIdx.x * kC5 + c, tr = blockIdx.y;
    double2* base = a.grids + (long long)tr * a.n + m;
    {
        const int j = tj;
        double2 x[16];
        // rows of tiles the spreading kernel never wrote are zeros that are not in memory: one liveness bit per tile
        const unsigned* masks = a.row_masks ? a.row_masks + (tr < a.set_of_trans_first ? 0 : 32) : nullptr;
        const int rshift = a.tile_shift - 8;                 // rows (256 cells) per spreading tile, log2
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const int row = J * i + j, tile = row >> rshift;
            x[i] = make_double2(0.0, 0.0);
            if (!masks || ((__ldg(&masks[tile & 31]) >> (tile >> 5)) & 1u)) x[i] = base[(long long)row * 256];
        }
        fft16(x);
        __syncthreads();                                     // table ready
#pragma unroll
        for (int ka = 0; ka < 16; ++ka) S[(ka * J + j) * kC5 + c] = cmul(x[pos16(ka)], wr[ka * j]);
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 80 / J; ++r) {                       // stage 2: butterfly (ka, q), elements S[ka][5 p + q]
        const int b = tj + J * r, ka = b & 15, q = b >> 4;
        double2 y[RM];
#pragma unroll
        for (int p = 0; p < RM; ++p) y[p] = S[(ka * J + 5 * p + q) * kC5 + c];
        fft_small<RM>(y);
#pragma unroll
        for (int kp = 0; kp < RM; ++kp)
            S[(ka * J + 5 * kp + q) * kC5 + c] = cmul(y[fft_pos<RM>(kp)], cTw5[RM == 2 ? 0 : RM == 4 ? 1 : RM == 8 ? 2 : 3][q][kp]);
    }
    __syncthreads();
    // stage 3: butterfly b = ka + 16 kp = tj + J r (elements S[ka][5 kp + q]), outputs k1 = b + 16 RM kq times the inter-pass
    // twiddle w_n^{k1 m} = w_n^{b m} (w_n^{16 RM m})^kq.  One table lookup per thread (w_n^{tj m}) instead of two per round: the
    // step over r, w_n^{J m}, and the step over kq depend on the column only and come from shared memory (colw).
    double2 twb = cmul(__ldg(&a.wlo[((unsigned)tj * (unsigned)m) & 4095u]), __ldg(&a.whi[((unsigned)tj * (unsigned)m) >> 12]));
    const double2 stb = colw[c], st = colw[kC5 + c];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int b = tj + J * r;
        if (b < 16 * RM) {
            const int ka = b & 15, kp = b >> 4;
            double2 z[5];
#pragma unroll
            for (int q = 0; q < 5; ++q) z[q] = S[(ka * J + 5 * kp + q) * kC5 + c];
            fft5(z);
            double2 tw = twb;
#pragma unroll
            for (int kq = 0; kq < 5; ++kq) {
                base[(long long)(b + 16 * RM * kq) * 256] = cmul(z[kq], tw);
                tw = cmul(tw, st);
            }
        }
        twb = cmul(twb, stb);
    }
}

// Pass 3: the transform dimension (l3) is contiguous; the CTA takes 16 consecutive k1 at one k2, so that the
// kept modes leave in runs of 16 consecutive frequencies.  Output: modes[tr][k], k = (kk + half) mod n < Nf,
// kk = k1 + R1 k2 + R1 R2 k3 the stored mode index (= k' mod n).
// VARIANT: opts.no_floating_mean / opts.normalization in effect (kept out of the default instantiation: the extra
// branches cost the fused kernel 20 us at config 3).
template <bool FUSED, bool VARIANT = false>
__global__ void __launch_bounds__(kFftThreads, 512 / kFftThreads)
ls_fft_rows_kernel(const FftArgs a) {
    extern __shared__ __align__(16) unsigned char fsm[];
    double2* Y = reinterpret_cast<double2*>(fsm);            // [ka][j][17] (padded: conflict-free both ways)
    double2* w256 = Y + 256 * (kC + 1);
    fill_w256(w256);
    // rows are numbered rho = k1 + R1 k2 (the low part of the output index): 16 consecutive rho per CTA
    const int rho_b = blockIdx.x * kC, tr = blockIdx.z;
    const double2* src = a.grids + (long long)tr * a.n;
    double2 x[16];
    {
        const int j = threadIdx.x & 15, c = threadIdx.x >> 4;
        const int rho = rho_b + c;
        const int k1 = a.R2 == 1 ? rho : (rho & (a.R1 - 1)), k2 = a.R2 == 1 ? 0 : (rho >> a.R1_shift);   // two passes: R1 need not be 2^k
        const double2* row = src + ((long long)k1 * a.R2 + k2) * a.R3;
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = row[16 * i + j];
        fft16(x);
        __syncthreads();
#pragma unroll
        for (int ka = 0; ka < 16; ++ka) Y[(ka * 16 + j) * (kC + 1) + c] = cmul(x[pos16(ka)], w256[ka * 16 + j]);
    }
    __syncthreads();
    {
        const int c = threadIdx.x % kC, ka = threadIdx.x / kC;
#pragma unroll
        for (int j = 0; j < 16; ++j) x[j] = Y[(ka * 16 + j) * (kC + 1) + c];
        fft16(x);
        double2* out = a.modes + (long long)tr * a.Nf;
        const long long kk0 = rho_b + c;
        const long long r12 = (long long)a.R1 * a.R2;
        const int ser = a.series0 + tr;
        const double YYs = FUSED ? a.sums[4 * ser + 2] : 1.0;
        const double inv_YY = 1.0 / YYs;
        if (FUSED) {
            // K5 + K6 with the per-frequency part (1/psihat, the tau rotation, 1/CC, 1/SS: functions of the weights only)
            // read from the table ls_freq_table_kernel made of the (w, w2) modes: what is left per series is the rotation
            // of its h mode and two squares.  Four frequencies at a time: their loads are in flight together.
#pragma unroll
            for (int g = 0; g < 16; g += 4) {
                long long k[4];
                double2 fr[4], fi[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    k[q] = kk0 + r12 * (ka + 16 * (g + q)) + a.half;
                    if (k[q] >= a.n) k[q] -= a.n;
                    fr[q] = fi[q] = make_double2(0.0, 0.0);
                    if (k[q] < a.Nf)                   // one 32-byte load per frequency
                        asm volatile("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];"
                                     : "=d"(fr[q].x), "=d"(fr[q].y), "=d"(fi[q].x), "=d"(fi[q].y) : "l"(a.ftab + 2 * k[q]));
                }
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    if (k[q] < a.Nf) {
                        const double2 gh = x[pos16(g + q)];                          // (Ch, Sh) / d
                        const double YC = gh.x * fr[q].x + gh.y * fr[q].y, YS = gh.y * fr[q].x - gh.x * fr[q].y;
                        double P = (YC * YC * fi[q].x + YS * YS * fi[q].y) * inv_YY;
                        if (VARIANT) P = apply_normalization(P, a.norm, YYs, a.sums[0]);
                        a.power[(long long)ser * a.Nf + k[q]] = P;
                    }
                }
            }
        } else {
#pragma unroll
            for (int kb = 0; kb < 16; ++kb) {
                long long k = kk0 + r12 * (ka + 16 * kb) + a.half;
                if (k >= a.n) k -= a.n;
                if (k < a.Nf) out[k] = x[pos16(kb)];
            }
        }
    }
}

// Passes 2 + 3 as ONE persistent kernel that keeps the intermediate in L2 (n >= 2^20, unfused assembly).
// After pass 1 the problem is R1 independent 65536-point transforms (row k1 = 1 MB, contiguous).  A SLAB is the C = 8
// rows k1 = C g .. C g + C - 1 of one transform (8 MB): pass 2 on it is 256 tiles (C rows x 256 / C column tiles),
// pass 3 on it is 256 tiles (one per k2, C consecutive k1 each — the unit that stores runs of C consecutive
// frequencies, 128 bytes).  CTAs (128 threads, four per SM) draw tiles from an ordered queue
//   [pass 2 of slab b][pass 3 of slab b - lag],  b = 0, 1, ...
// and a pass-3 tile first waits until all 256 pass-2 tiles of its slab have been signalled done.  Every tile a CTA
// can wait for was drawn earlier, by a CTA that is running and never waits before it signals, so the queue cannot
// deadlock.  What a slab's pass 2 writes is read back by its pass 3 a few microseconds later out of the 126 MB L2
// (ncu: 0.02 % of pass 3's input comes from DRAM), and once read the lines are dead: `discard.global.L2` drops them
// before they are ever written back.  DRAM traffic of the two passes: 3.0 GB -> 1.48 GB at config 3
// (profiles/r1g_fft_l2_fusion.md).  lag = 3 (measured: lag 1 0.59 ms, 2 0.3965, 3 0.393, 4 0.395, 6 0.435 — one slab
// is less than half a wave of the 592 resident CTAs, so a short lag makes pass-3 tiles wait and a long one pushes
// slabs out of L2).
// After the kernel the fine grids hold indeterminate values; nothing reads them again (the next execute's spreading
// kernel rewrites every tile that pass 1 will load).
// queue: [0] next item, [1] CTAs that left, [2 + s] pass-2 tiles of slab s done.  The last CTA to leave zeroes it.
constexpr int kC23 = 8;                  // tile width of the fused kernel
constexpr int kLag23 = 3;
__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
constexpr int kPrefetch23 = 512;             // queue distance of the L2 prefetch: the same tile of the next slab
template <int C>                                          // C columns (pass 2) / rows (pass 3) per tile, 16 C threads
__global__ void __launch_bounds__(16 * C, 512 / (16 * C))
ls_fft_pass23_kernel(const FftArgs a, int nslabs, int* __restrict__ queue) {
    constexpr int lag = kLag23;
    constexpr int T = 16 * C, CT = 256 / C;                  // threads; column tiles per row
    extern __shared__ __align__(16) unsigned char fsm[];
    double2* Y = reinterpret_cast<double2*>(fsm);            // pass 2: [ka][j][C]; pass 3: [ka][j][C + 1]
    double2* w256 = Y + 256 * (C + 1);
    __shared__ int s_item[2];                                // the CTA's current / next queue item (double-buffered)
    fill_w256(w256, T);
    // w_256^{16 j} = e^{2 pi i j / 16} for this thread's j in a pass-2 tile (j = tid / C) and in a pass-3 tile (j = tid % 16)
    double2 c16_p2, c16_p3;
    sincospi((double)(threadIdx.x / C) / 8.0, &c16_p2.y, &c16_p2.x);
    sincospi((double)(threadIdx.x & 15) / 8.0, &c16_p3.y, &c16_p3.x);
    const int groups = a.R1 / C;                             // slabs per transform
    const int total = (nslabs + lag) * 512;
    if (threadIdx.x == 0) s_item[0] = atomicAdd(&queue[0], 1);
    __syncthreads();                                         // s_item[0], w256 ready
    // Barriers per tile: the exchange and ONE more that frees Y, publishes the next item (written by thread 0 into the
    // other half of s_item just before it) and, for a pass-2 tile, certifies that every thread's stores are issued.
    for (int par = 0;; par ^= 1) {
        const int item = s_item[par];
        if (item >= total) break;
        // the next draw is requested now and parked in a register: its latency hides behind this tile
        int next_item = 0;
        if (threadIdx.x == 0) next_item = atomicAdd(&queue[0], 1);
        const int b = item >> 9, slot = item & 255;
        double2 x[16];
        if ((item & 256) == 0) {
            // ---- pass 2 tile: row k1 = C g + slot / CT, columns C (slot % CT) ..
            if (b >= nslabs) goto next;
            const int tr = b / groups, g = b - tr * groups;
            const int k1 = C * g + slot / CT;
            const int c = threadIdx.x % C, hi4 = threadIdx.x / C;
            const long long m = (long long)(slot % CT) * C + c;
            double2* base = a.grids + (long long)tr * a.n + (long long)k1 * 65536 + m;
            {
                const int j = hi4;
#pragma unroll
                for (int i = 0; i < 16; ++i) x[i] = base[(long long)(16 * i + j) * 256];
                {
                    // pull the pass-2 tile one slab further down the queue (some CTA draws it about a wave from now)
                    // from HBM into L2: its loads then wait for L2, not for DRAM (0.450 -> 0.441 ms at config 3)
                    const int it = item + kPrefetch23;
                    const int pb = it >> 9, ps = it & 255;
                    if (pb < nslabs) {
                        const int ptr = pb / groups, pg = pb - ptr * groups;
                        const double2* pbase = a.grids + (long long)ptr * a.n + (long long)(C * pg + ps / CT) * 65536 +
                                               (long long)(ps % CT) * C;
                        for (int r = threadIdx.x; r < 256; r += T)      // one 128-byte line per row of the tile
                            asm volatile("prefetch.global.L2 [%0];" ::"l"(pbase + (long long)r * 256));
                    }
                }
                fft16(x);
#pragma unroll
                for (int ka = 0; ka <= 8; ++ka) {
                    // w^{j ka} from the table for ka <= 8; w^{j (16 - ka)} = w^{16 j} conj(w^{j ka}) (one multiplication
                    // by a per-thread constant instead of a shared-memory lookup: the kernel is LSU-bound)
                    if (ka == 0) { Y[j * C + c] = x[0]; continue; }
                    const double2 t = w256[ka * 16 + j];
                    Y[(ka * 16 + j) * C + c] = cmul(x[pos16(ka)], t);
                    if (ka < 8) Y[((16 - ka) * 16 + j) * C + c] = cmul(cmul(x[pos16(16 - ka)], c16_p2), make_double2(t.x, -t.y));
                }
            }
            __syncthreads();
            {
                const int ka = hi4;
#pragma unroll
                for (int j = 0; j < 16; ++j) x[j] = Y[(ka * 16 + j) * C + c];
                fft16(x);
                const unsigned mm = (unsigned)m * (unsigned)a.R1;
                const double2 tw = twiddle_n(a, (unsigned)ka * mm);
                const double2 st = twiddle_n(a, 16u * mm);
                store_twiddled<16>(base, 256, ka, tw, st, [&](int kb) { return x[pos16(kb)]; });
            }
            if (threadIdx.x == 0) s_item[par ^ 1] = next_item;
            __syncthreads();                                 // every thread's stores are issued ...
            if (threadIdx.x == 0) {
                // ... and ordered before the signal, device-wide: a release reduction (MEMBAR.ALL.GPU) instead of
                // __threadfence() + atomicAdd (MEMBAR.SC.GPU): 0.4005 -> 0.396 ms
                asm volatile("red.release.gpu.global.add.s32 [%0], 1;" ::"l"(queue + 2 + b) : "memory");
            }
            continue;
        } else {
            // ---- pass 3 tile: k2 = slot, k1 = C g .. C g + C - 1
            const int sl = b - lag;
            if (sl < 0) goto next;
            const int tr = sl / groups, g = sl - tr * groups;
            if (threadIdx.x == 0) {
                // acquire load, not volatile load + __threadfence(): the fence would also wait for this thread's own
                // stores of the previous tile to drain, with the whole CTA parked at the barrier below (0.406 -> 0.4005 ms)
                const int* done = queue + 2 + sl;
                while (ld_acquire_gpu(done) < 256) __nanosleep(40);
            }
            __syncthreads();
            const int rho_b = slot * a.R1 + C * g;
            const double2* src = a.grids + (long long)tr * a.n;
            {
                const int j = threadIdx.x & 15, c = threadIdx.x >> 4;
                const double2* row = src + ((long long)(C * g + c) * 256 + slot) * 256;
#pragma unroll
                for (int i = 0; i < 16; ++i) x[i] = __ldcg(&row[16 * i + j]);    // written by other SMs: read at L2
                fft16(x);
#pragma unroll
                for (int ka = 0; ka <= 8; ++ka) {
                    if (ka == 0) { Y[j * (C + 1) + c] = x[0]; continue; }
                    const double2 t = w256[ka * 16 + j];
                    Y[(ka * 16 + j) * (C + 1) + c] = cmul(x[pos16(ka)], t);
                    if (ka < 8) Y[((16 - ka) * 16 + j) * (C + 1) + c] = cmul(cmul(x[pos16(16 - ka)], c16_p3), make_double2(t.x, -t.y));
                }
            }
            __syncthreads();
            {
                // the slab is dead once read: drop its dirty lines from L2 instead of writing them back to HBM
                // (thread (c, j) drops lines 2 j and 2 j + 1 of row c's 4 KB chunk; all its loads have landed)
                const int j = threadIdx.x & 15, c = threadIdx.x >> 4;
                const double2* row = src + ((long long)(C * g + c) * 256 + slot) * 256 + 16 * j;
                asm volatile("discard.global.L2 [%0], 128;" ::"l"(row) : "memory");
                asm volatile("discard.global.L2 [%0], 128;" ::"l"(row + 8) : "memory");
            }
            {
                const int c = threadIdx.x % C, ka = threadIdx.x / C;
#pragma unroll
                for (int j = 0; j < 16; ++j) x[j] = Y[(ka * 16 + j) * (C + 1) + c];
                if (threadIdx.x == 0) s_item[par ^ 1] = next_item;
                __syncthreads();                             // Y is free
                fft16(x);
                double2* out = a.modes + (long long)tr * a.Nf;
                const long long kk0 = rho_b + c;
                const long long r12 = (long long)a.R1 * 256;
#pragma unroll
                for (int kb = 0; kb < 16; ++kb) {
                    long long k = kk0 + r12 * (ka + 16 * kb) + a.half;
                    if (k >= a.n) k -= a.n;
                    if (k < a.Nf) __stcs(&out[k], x[pos16(kb)]);     // read once, by the assembly, after 600 MB more
                }
            }
            continue;
        }
    next:                                                    // items past either end of the slab sequence: nothing to do
        if (threadIdx.x == 0) s_item[par ^ 1] = next_item;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        if (atomicAdd(&queue[1], 1) == (int)gridDim.x - 1) {  // last CTA out: nobody draws or waits any more
            for (int i = 0; i < nslabs + 2; ++i) queue[i] = 0;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Passes 2 + 3, bulk-asynchronous version (the default for n >= 2^20): the same ordered tile queue, slab signals, L2
// residency and discard as ls_fft_pass23_kernel above, but the tiles are MOVED by the TMA unit instead of by the
// threads that compute on them.  One persistent CTA per SM = one producer warp + k23Groups consumer groups of 128
// threads, a ring of k23Stages shared-memory tile buffers, one full / empty mbarrier pair per buffer:
//   producer (one elected thread): draws the next queue item, waits for the buffer to be free, waits (pass-3 tiles) for
//     the slab's pass-2 signal, then issues the tile load — pass-2 tile (256 rows x 128 bytes, rows 4 KB apart): ONE
//     cp.async.bulk.tensor.3d through a tensor map over [k1][l2][l3]; pass-3 tile (8 rows of 4 KB, 1 MB apart): eight
//     cp.async.bulk copies into rows padded by one cell (conflict-free second stage) — with complete_tx on the buffer's
//     full barrier, and prefetches the pass-2 tile one slab ahead into L2 (cp.async.bulk.prefetch.tensor);
//   consumers: wait on the full barrier, run the first 16-point stage out of shared memory IN PLACE (a thread writes
//     back exactly the 16 cells it read), one named barrier of their own 128 threads, second stage out of shared memory,
//     release the buffer (mbarrier arrive) as soon as their operands are in registers, twiddle and store.
// The 16 data registers x 2 of a thread are therefore never parked on a global load: the loads of the next k23Stages -
// k23Groups tiles are in flight while every consumer warp computes.
constexpr int k23Stages = 6;                          // tile buffers in the ring
constexpr int kLagTma = 3;                            // slabs between a slab's pass 2 and its pass 3 in the queue
constexpr int k23Batch = 4;                           // consecutive queue items per draw
__host__ __device__ constexpr int k23threads(int groups) { return (groups * 4 + 1) * 32; }   // consumer groups of 128 threads + the producer warp
constexpr int k23RowBytes = 4096 + 16;                // a pass-3 tile row (256 cells) padded by one cell
constexpr int k23BufBytes = 8 * k23RowBytes;          // 32896 >= 32768 (pass-2 tile, dense); a multiple of 128
constexpr size_t k23TmaSmem = (size_t)k23Stages * k23BufBytes + sizeof(double2) * 3 * 256 + 16 * k23Stages + 4 * k23Stages + 64;

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    unsigned ok;
    do {                                                     // try_wait suspends the thread in hardware for a while
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}"
            : "=r"(ok)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!ok);
}
__device__ __forceinline__ void tma_load_3d(unsigned dst, const CUtensorMap* map, unsigned bar, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(dst),
        "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_3d(const CUtensorMap* map, int c0, int c1, int c2) {
    asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global.tile [%0, {%1, %2, %3}];" ::"l"(map), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
__device__ __forceinline__ void bulk_load(unsigned dst, const void* src, unsigned bytes, unsigned bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void group_barrier(int id) { asm volatile("bar.sync %0, 128;" ::"r"(id) : "memory"); }

template <int k23Groups>                                 // consumer groups (128 threads, one tile at a time each)
__global__ void __launch_bounds__(k23threads(k23Groups), 1)
ls_fft_pass23_tma_kernel(const FftArgs a, const __grid_constant__ CUtensorMap tmap, int row0, int nslabs, int lag,
                         int* __restrict__ queue) {
    constexpr int C = 8, CT = 256 / C, k23Threads = k23threads(k23Groups);
    extern __shared__ __align__(128) unsigned char tsm[];
    unsigned char* bufs = tsm;
    double2* w256 = reinterpret_cast<double2*>(tsm + (size_t)k23Stages * k23BufBytes);
    // inter-pass twiddles of pass 2, w_n^{R1 k2 l3} = w_65536^x with x = k2 l3 < 65536, from two 256-entry tables in
    // shared memory: w_65536^x = wcoarse[x >> 8] wfine[x & 255].  (The 2 x 64 KB global tables of twiddle_n do not fit
    // the 20 KB of L1 this kernel leaves: their misses sat in front of every tile's stores.)
    double2* wcoarse = w256 + 256;
    double2* wfine = wcoarse + 256;
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(wfine + 256);   // full[k23Stages], empty[k23Stages]
    int* sitem = reinterpret_cast<int*>(bars + 2 * k23Stages);
    const unsigned full0 = smem_u32(bars), empty0 = smem_u32(bars + k23Stages);
    const int warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) {
        for (int b = 0; b < k23Stages; ++b) {
            mbar_init(full0 + 8 * b, 1);               // the producer's arrive.expect_tx (+ the bytes of the tile)
            mbar_init(empty0 + 8 * b, 128);            // every thread of the consumer group
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    fill_w256(w256, k23Threads);
    for (int i = threadIdx.x; i < 256; i += k23Threads) {
        double sn, cs;
        sincospi((double)i / 128.0, &sn, &cs);
        wcoarse[i] = make_double2(cs, sn);
        sincospi((double)i / 32768.0, &sn, &cs);
        wfine[i] = make_double2(cs, sn);
    }
    __syncthreads();
    const int groups = a.R1 / C;                             // slabs per transform
    const int total = (nslabs + lag) * 512;

    if (warp == k23Groups * 4) {
        // ------------------------------------------------------------------------------------------ producer
        if ((threadIdx.x & 31) == 0) {
            int filled = 0, terminators = 0;
            int ready_slabs = 0;                             // slabs [0, ready_slabs) are known to be complete
            // Items are drawn from the shared counter k23Batch at a time, the next draw always in flight.  One address takes
            // an atomic with return every ~16 cycles chip-wide (measured: 49 152 single-item draws took 0.39 - 0.44 ms,
            // whatever the kernel did otherwise — the first version of this kernel AND the per-thread-load kernel above were
            // both bound by their own work counter), so the draws must be few.
            int cur = atomicAdd(&queue[0], k23Batch), nxt = atomicAdd(&queue[0], k23Batch), sub = 0;
            while (terminators < k23Groups) {
                int item = total;
                if (terminators == 0) {
                    item = cur + sub;
                    if (++sub == k23Batch) {
                        sub = 0;
                        cur = nxt;
                        nxt = cur < total ? atomicAdd(&queue[0], k23Batch) : total;
                    }
                }
                const int buf = filled % k23Stages;
                const unsigned fb = full0 + 8 * buf, eb = empty0 + 8 * buf;
                const unsigned dst = smem_u32(bufs + (size_t)buf * k23BufBytes);
                if (item >= total) {                         // one terminator per consumer group (consecutive ring slots)
                    mbar_wait(eb, ((filled / k23Stages) & 1) ^ 1);
                    sitem[buf] = -1;
                    mbar_arrive(fb);
                    ++terminators;
                    ++filled;
                    continue;
                }
                const int b = item >> 9, slot = item & 255;
                if ((item & 256) == 0) {
                    // ---- pass-2 tile: row k1 = C g + slot / CT of transform tr, columns C (slot % CT) ..
                    {
                        const int it = item + kPrefetch23;   // the same tile of the next slab: HBM -> L2 ahead of its load
                        const int pb = it >> 9, ps = it & 255;
                        if (pb < nslabs) {
                            const int ptr = pb / groups, pg = pb - ptr * groups;
                            tma_prefetch_3d(&tmap, 2 * C * (ps % CT), 0, row0 + ptr * a.R1 + C * pg + ps / CT);
                        }
                    }
                    if (b >= nslabs) continue;
                    const int tr = b / groups, g = b - tr * groups;
                    mbar_wait(eb, ((filled / k23Stages) & 1) ^ 1);
                    sitem[buf] = item;
                    mbar_expect_tx(fb, 256 * C * 16);
                    tma_load_3d(dst, &tmap, fb, 2 * C * (slot % CT), 0, row0 + tr * a.R1 + C * g + slot / CT);
                } else {
                    // ---- pass-3 tile: k2 = slot, rows k1 = C g .. C g + C - 1 of the slab drawn `lag` slabs ago
                    const int sl = b - lag;
                    if (sl < 0) continue;
                    const int tr = sl / groups, g = sl - tr * groups;
                    mbar_wait(eb, ((filled / k23Stages) & 1) ^ 1);
                    if (sl >= ready_slabs) {                 // slabs complete in queue order (nearly): ask once per slab
                        const int* done = queue + 2 + sl;
                        while (ld_acquire_gpu(done) < 256) __nanosleep(40);
                        asm volatile("fence.proxy.async.global;" ::: "memory");   // the slab was written through the generic proxy
                        ready_slabs = sl + 1;
                    }
                    sitem[buf] = item;
                    mbar_expect_tx(fb, 256 * C * 16);
                    const double2* src = a.grids + (long long)tr * a.n + ((long long)(C * g) * 256 + slot) * 256;
#pragma unroll
                    for (int c = 0; c < C; ++c) bulk_load(dst + c * k23RowBytes, src + (long long)c * 65536, 4096, fb);
                }
                ++filled;
            }
        }
    } else {
        // ------------------------------------------------------------------------------------------ consumers
        const int grp = warp >> 2, t = threadIdx.x & 127;
        // w_256^{16 j} = e^{2 pi i j / 16} for this thread's j in a pass-2 tile (j = t / C) and in a pass-3 tile (j = t % 16)
        double2 c16_p2, c16_p3;
        sincospi((double)(t / C) / 8.0, &c16_p2.y, &c16_p2.x);
        sincospi((double)(t & 15) / 8.0, &c16_p3.y, &c16_p3.x);
        for (int seq = grp;; seq += k23Groups) {
            const int buf = seq % k23Stages;
            mbar_wait(full0 + 8 * buf, (seq / k23Stages) & 1);
            const int item = sitem[buf];
            if (item < 0) break;
            unsigned char* tile = bufs + (size_t)buf * k23BufBytes;
            const int b = item >> 9, slot = item & 255;
            double2 x[16];
            if ((item & 256) == 0) {
                // ---- pass 2: transform over l2 (the 256 rows of the tile), C columns
                const int tr = b / groups, g = b - tr * groups;
                const int k1 = C * g + slot / CT;
                const int c = t % C, hi4 = t / C;
                const long long m = (long long)(slot % CT) * C + c;
                double2* T = reinterpret_cast<double2*>(tile);
                {
                    const int j = hi4;
#pragma unroll
                    for (int i = 0; i < 16; ++i) x[i] = T[(16 * i + j) * C + c];
                    fft16(x);
#pragma unroll
                    for (int ka = 0; ka <= 8; ++ka) {
                        if (ka == 0) { T[j * C + c] = x[0]; continue; }
                        const double2 tw = w256[ka * 16 + j];
                        T[(ka * 16 + j) * C + c] = cmul(x[pos16(ka)], tw);
                        if (ka < 8) T[((16 - ka) * 16 + j) * C + c] = cmul(cmul(x[pos16(16 - ka)], c16_p2), make_double2(tw.x, -tw.y));
                    }
                }
                group_barrier(1 + grp);
                {
                    const int ka = hi4;
#pragma unroll
                    for (int j = 0; j < 16; ++j) x[j] = T[(ka * 16 + j) * C + c];
                    mbar_arrive(empty0 + 8 * buf);           // operands are in registers: the buffer can be refilled
                    const unsigned x0 = (unsigned)ka * (unsigned)m, x1 = 16u * (unsigned)m;      // k2 = ka + 16 kb
                    const double2 tw = cmul(wcoarse[x0 >> 8], wfine[x0 & 255u]);
                    const double2 st = cmul(wcoarse[x1 >> 8], wfine[x1 & 255u]);
                    fft16(x);
                    double2* base = a.grids + (long long)tr * a.n + (long long)k1 * 65536 + m;
                    store_twiddled<16>(base, 256, ka, tw, st, [&](int kb) { return x[pos16(kb)]; });
                }
                group_barrier(1 + grp);                      // every thread's stores are issued ...
                if (t == 0) {
                    // ... and ordered before the signal, device-wide, for the generic and the async proxy
                    asm volatile("fence.proxy.async.global;" ::: "memory");
                    asm volatile("red.release.gpu.global.add.s32 [%0], 1;" ::"l"(queue + 2 + b) : "memory");
                }
            } else {
                // ---- pass 3: transform over l3 (contiguous), C rows k1 = C g .. at k2 = slot
                const int sl = b - lag;
                const int tr = sl / groups, g = sl - tr * groups;
                const int rho_b = slot * a.R1 + C * g;
                {
                    const int j = t & 15, c = t >> 4;
                    double2* row = reinterpret_cast<double2*>(tile + c * k23RowBytes);
#pragma unroll
                    for (int i = 0; i < 16; ++i) x[i] = row[16 * i + j];
                    {
                        // the slab is dead once it sits in shared memory: drop its dirty lines from L2 instead of writing
                        // them back to HBM (thread (c, j) drops lines 2 j and 2 j + 1 of row c's 4 KB chunk)
                        const double2* grow = a.grids + (long long)tr * a.n + ((long long)(C * g + c) * 256 + slot) * 256 + 16 * j;
                        asm volatile("discard.global.L2 [%0], 128;" ::"l"(grow) : "memory");
                        asm volatile("discard.global.L2 [%0], 128;" ::"l"(grow + 8) : "memory");
                    }
                    fft16(x);
#pragma unroll
                    for (int ka = 0; ka <= 8; ++ka) {
                        if (ka == 0) { row[j] = x[0]; continue; }
                        const double2 tw = w256[ka * 16 + j];
                        row[ka * 16 + j] = cmul(x[pos16(ka)], tw);
                        if (ka < 8) row[(16 - ka) * 16 + j] = cmul(cmul(x[pos16(16 - ka)], c16_p3), make_double2(tw.x, -tw.y));
                    }
                }
                group_barrier(1 + grp);
                {
                    const int c = t % C, ka = t / C;
                    const double2* row = reinterpret_cast<const double2*>(tile + c * k23RowBytes);
#pragma unroll
                    for (int j = 0; j < 16; ++j) x[j] = row[ka * 16 + j];
                    mbar_arrive(empty0 + 8 * buf);
                    fft16(x);
                    double2* out = a.modes + (long long)tr * a.Nf;
                    const long long kk0 = rho_b + c;
                    const long long r12 = (long long)a.R1 * 256;
#pragma unroll
                    for (int kb = 0; kb < 16; ++kb) {
                        long long k = kk0 + r12 * (ka + 16 * kb) + a.half;
                        if (k >= a.n) k -= a.n;
                        if (k < a.Nf) __stcs(&out[k], x[pos16(kb)]);     // read once, by the assembly, after 600 MB more
                    }
                }
            }
        }
    }
    __syncthreads();                                         // every signal of this CTA has been posted
    if (threadIdx.x == 0) {
        if (atomicAdd(&queue[1], 1) == (int)gridDim.x - 1) {  // last CTA out: nobody draws or waits any more
            for (int i = 0; i < nslabs + 2; ++i) queue[i] = 0;
        }
    }
}

// Fused assembly, shared dy: the per-frequency terms of K5 + K6 from the compact (w, w2) modes, once per execute.
__global__ void ls_freq_table_kernel(const double2* __restrict__ w_modes, const double2* __restrict__ w2_modes,
                                     const double* __restrict__ dinv, long long Nf, long long half, int no_float,
                                     double2* __restrict__ ftab) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= Nf) return;
    const long long kp = k - half;
    const double d = dinv[kp < 0 ? -kp : kp];
    const double2 gw = w_modes[k], g2 = w2_modes[k];
    const double dw = no_float ? 0.0 : d;                   // fixed mean: S = C = 0
    const FreqTerms f = freq_terms(gw.y * dw, gw.x * dw, g2.y * d, g2.x * d);
    ftab[2 * k] = make_double2(f.Cw * d, f.Sw * d);
    ftab[2 * k + 1] = make_double2(f.iCC, f.iSS);
}

__global__ void ls_fft_tables_kernel(double2* wlo, double2* whi, long long n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < 4096) {
        double s, c;
        sincospi(2.0 * (double)i / (double)n, &s, &c);
        wlo[i] = make_double2(c, s);
    }
    if ((long long)i < n / 4096) {
        double s, c;
        sincospi(2.0 * (double)i * 4096.0 / (double)n, &s, &c);
        whi[i] = make_double2(c, s);
    }
}

constexpr size_t kColsSmem = sizeof(double2) * (256 * kC + 256);
constexpr int kPass1Threads = 128;
constexpr size_t kPass1Smem = sizeof(double2) * (16 * kPass1Threads + 256);
constexpr size_t kRowsSmem = sizeof(double2) * (256 * (kC + 1) + 256);
constexpr size_t k23Smem = sizeof(double2) * (256 * (kC23 + 1) + 256);

}  // namespace

// fp64 grids of n = 2^12 .. 2^24 cells:
//   2^20 .. 2^24: three passes R1 x 256 x 256, R1 = 16 .. 256, first pass pruned by the spreading kernel's liveness
//                 masks (needs spreading tiles that divide a pass-1 row of 65536 cells);
//   2^17 .. 2^19: three passes with a small first radix R1 = 2, 4, 8 (ls_fft_pass1_small_kernel), unpruned;
//   2^12 .. 2^16: two passes R1 x 256, R1 = 16 .. 256, unpruned.
//   5 x 2^13 .. 5 x 2^16: two passes R1 x 256, R1 = 160 .. 1280 = 16 x RM x 5 (ls_fft_cols5_kernel), unpruned.
int own_fft_rm5(const ls_plan_s* p) {                     // RM of the 5 x 2^k sizes, else 0
    for (int rm = 2; rm <= 16; rm *= 2)
        if (p->n == (int64_t)80 * rm * 256) return rm;
    return 0;
}
bool own_fft_supported(const ls_plan_s* p) {
    const bool pow2 = (p->n & (p->n - 1)) == 0;
    if (p->dtype == LS_F64 && own_fft_rm5(p)) return true;
    if (own_fft_f32_rm(p)) return true;                    // fp32, 5 x 2^22 .. 5 x 2^25 cells (ls_fft_f32.cu)
    if (p->dtype != LS_F64 || !pow2 || p->n < ((int64_t)1 << 12) || p->n > ((int64_t)1 << 24)) return false;
    return p->n < ((int64_t)1 << 20) || 65536 % p->L == 0;
}
bool own_fft_prunes(const ls_plan_s* p) { return p->n >= ((int64_t)1 << 20) || own_fft_rm5(p) != 0; }
// spreading tiles per liveness-mask column: 65536 / L where the first pass works on rows of 65536 cells; 1 at the 5 x 2^k
// sizes (rows of 256 cells: the masks are then one bit per TILE, word = tile % 32, bit = tile / 32 — at most 1280 tiles)
int own_fft_ncoltiles(const ls_plan_s* p) { return own_fft_rm5(p) ? 1 : own_fft_f32_rm(p) ? 131072 / p->L : std::max(1, 65536 / p->L); }
// radix of the first pass / 16 where that pass is the 16 x RB kernel (n >= 2^20: R1 = n / 2^16; n <= 2^16: R1 = n / 2^8)
int own_fft_rb(const ls_plan_s* p) { return own_fft_rm5(p) ? 32 : own_fft_f32_rm(p) ? 5 * own_fft_f32_rm(p) / 2 : (int)(p->n >= ((int64_t)1 << 20) ? p->n >> 20 : p->n >> 12); }

cudaError_t own_fft_init(ls_plan_s* p, cudaStream_t s) {
    const int cnt = (int)std::max<long long>(4096, p->n / 4096);
    ls_fft_tables_kernel<<<(cnt + 255) / 256, 256, 0, s>>>((double2*)p->fft_wlo, (double2*)p->fft_whi, p->n);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (p->dtype == LS_F32) return own_fft_f32_init(p, s);
    if ((e = cudaFuncSetAttribute(ls_fft_pass1_kernel<16, kPass1Threads>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPass1Smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_pass1_kernel<8, kPass1Threads>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPass1Smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_pass1_kernel<4, kPass1Threads>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPass1Smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_pass1_kernel<2, kPass1Threads>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPass1Smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_pass1_kernel<1, kPass1Threads>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPass1Smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_cols_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kColsSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_cols5_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cols5_smem<2>())) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_cols5_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cols5_smem<4>())) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_cols5_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cols5_smem<8>())) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_cols5_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cols5_smem<16>())) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_pass23_kernel<kC23>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k23Smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_pass23_tma_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k23TmaSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_pass23_tma_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k23TmaSmem)) != cudaSuccess) return e;
    if (own_fft_rm5(p)) {
        double2 h[4][5][16];
        for (int v = 0; v < 4; ++v)
            for (int q = 0; q < 5; ++q)
                for (int kp = 0; kp < 16; ++kp) {
                    const double ang = 2.0 * M_PI * (double)((kp * q) % (10 << v)) / (double)(10 << v);   // 5 RM = 10, 20, 40, 80
                    h[v][q][kp] = make_double2(cos(ang), sin(ang));
                }
        if ((e = cudaMemcpyToSymbolAsync(cTw5, h, sizeof h, 0, cudaMemcpyHostToDevice, s)) != cudaSuccess) return e;
        if ((e = cudaStreamSynchronize(s)) != cudaSuccess) return e;
    }
    if ((e = own_fft_make_tmap(p)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_pass23_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRowsSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_rows_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRowsSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_fft_rows_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRowsSmem)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(ls_fft_rows_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRowsSmem);
}

static void fill_common(const ls_plan_s* p, FftArgs& a, int slot0, int n_x2) {
    a.grids = (double2*)p->grids + (long long)slot0 * p->n;
    a.n = p->n;
    a.R3 = 256;
    a.R2 = (p->n > 65536 && !own_fft_rm5(p)) ? 256 : 1;    // two passes up to 2^16 cells and at the 5 x 2^k sizes
    a.R1 = (int)(p->n / ((long long)a.R2 * a.R3));
    a.R1_shift = 0;
    while ((1 << a.R1_shift) < a.R1) ++a.R1_shift;
    a.wlo = (const double2*)p->fft_wlo;
    a.whi = (const double2*)p->fft_whi;
    a.row_masks = own_fft_prunes(p) ? p->row_masks : nullptr;
    a.ncoltiles = own_fft_ncoltiles(p);
    a.set_of_trans_first = n_x2;
    a.tile_shift = 0;
    while ((1 << a.tile_shift) < p->L) ++a.tile_shift;
    a.modes = (double2*)p->modes + (long long)slot0 * p->Nf;
    a.Nf = p->Nf;
    a.half = p->Nf / 2;
    a.w_modes = a.w2_modes = nullptr;
    a.ftab = (const double2*)p->ftab;
    a.dinv = p->dinv;
    a.sums = p->sums;
    a.power = nullptr;
    a.series0 = 0;
    a.no_float = p->opts.no_floating_mean;
    a.norm = p->opts.normalization;
}

// Pass 1 of transforms [slot0, slot0 + ntrans) of the plan's grids; the first n_x2 of them belong to the x2
// point set (which liveness masks to prune by).
cudaError_t launch_own_fft_pass1(ls_plan_s* p, int slot0, int ntrans, int n_x2, cudaStream_t s) {
    if (p->dtype == LS_F32) return launch_own_fft_f32_pass1(p, slot0, ntrans, n_x2, s);
    FftArgs a;
    fill_common(p, a, slot0, n_x2);
    const long long inner1 = (long long)a.R2 * a.R3;       // 65536 (three passes) or 256 (two passes)
    if (const int rm = own_fft_rm5(p)) {                   // n = 5 x 2^k
        const dim3 g(256 / kC5, ntrans);
        switch (rm) {
            case 2: ls_fft_cols5_kernel<2><<<g, 5 * 2 * kC5, cols5_smem<2>(), s>>>(a); break;
            case 4: ls_fft_cols5_kernel<4><<<g, 5 * 4 * kC5, cols5_smem<4>(), s>>>(a); break;
            case 8: ls_fft_cols5_kernel<8><<<g, 5 * 8 * kC5, cols5_smem<8>(), s>>>(a); break;
            default: ls_fft_cols5_kernel<16><<<g, 5 * 16 * kC5, cols5_smem<16>(), s>>>(a); break;
        }
        return cudaGetLastError();
    }
    if (a.R1 < 16) {                                       // n = 2^17 .. 2^19
        dim3 g((unsigned)std::min<long long>((inner1 + 255) / 256, 4LL * p->num_sms), ntrans);
        if (a.R1 == 8) ls_fft_pass1_small_kernel<8><<<g, 256, 0, s>>>(a, inner1);
        else if (a.R1 == 4) ls_fft_pass1_small_kernel<4><<<g, 256, 0, s>>>(a, inner1);
        else ls_fft_pass1_small_kernel<2><<<g, 256, 0, s>>>(a, inner1);
        return cudaGetLastError();
    }
    const int rb = own_fft_rb(p);
    // 128-thread CTAs (tiles of 2048 points, four CTAs per SM): a barrier then waits for four warps, not eight
    // (pass 1 at config 3: 0.215 -> 0.207 ms against 256-thread CTAs with 4096-point tiles)
    constexpr int T = kPass1Threads;
    const int tiles_per_trans = (int)(inner1 / (T / rb)), total = tiles_per_trans * ntrans;
    const int nblk = std::min(total, (512 / T) * p->num_sms);
    switch (rb) {
        case 16: ls_fft_pass1_kernel<16, T><<<nblk, T, kPass1Smem, s>>>(a, inner1, tiles_per_trans, total); break;
        case 8: ls_fft_pass1_kernel<8, T><<<nblk, T, kPass1Smem, s>>>(a, inner1, tiles_per_trans, total); break;
        case 4: ls_fft_pass1_kernel<4, T><<<nblk, T, kPass1Smem, s>>>(a, inner1, tiles_per_trans, total); break;
        case 2: ls_fft_pass1_kernel<2, T><<<nblk, T, kPass1Smem, s>>>(a, inner1, tiles_per_trans, total); break;
        default: ls_fft_pass1_kernel<1, T><<<nblk, T, kPass1Smem, s>>>(a, inner1, tiles_per_trans, total); break;
    }
    return cudaGetLastError();
}

cudaError_t launch_own_fft_pass2(ls_plan_s* p, int slot0, int ntrans, cudaStream_t s) {
    if (p->dtype == LS_F32) return launch_own_fft_f32_pass2(p, slot0, ntrans, s);
    FftArgs a;
    fill_common(p, a, slot0, 0);
    if (a.R2 == 1) return cudaSuccess;                     // two-pass sizes: nothing between pass 1 and the last pass
    dim3 g2(256 / kC, a.R1, ntrans);                       // [k1][l2][l3]: outer = R1 blocks, stride 256
    ls_fft_cols_kernel<<<g2, kFftThreads, kColsSmem, s>>>(a, a.R1, 256);
    return cudaGetLastError();
}

// Tensor map over the plan's fine grids viewed as [rows k1 of every slot][l2 = 256][l3 = 256 cells = 512 doubles]
// (n >= 2^20: a pass-1 output row k1 is 65536 cells = 1 MB), box = one pass-2 tile: 8 cells x 256 rows l2 of one k1.
// The encoder is a driver entry point fetched through the runtime (no link against libcuda).  Called at plan time and
// whenever the grids move (ls_set_workspace).
cudaError_t own_fft_make_tmap(ls_plan_s* p) {
    if (!p->fuse_pass23) return cudaSuccess;
    static_assert(sizeof(CUtensorMap) <= sizeof(p->fft_tmap), "tensor map storage");
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess) return e;
    if (qres != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
    typedef CUresult (*encode_t)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    const cuuint64_t rows = (cuuint64_t)p->slots * (cuuint64_t)(p->n / 65536);
    const cuuint64_t dims[3] = {512, 256, rows};
    const cuuint64_t strides[2] = {4096, 1048576};           // bytes: l2 -> l2 + 1, k1 -> k1 + 1
    const cuuint32_t box[3] = {2 * kC23, 256, 1}, estr[3] = {1, 1, 1};
    const CUresult r = ((encode_t)fn)(reinterpret_cast<CUtensorMap*>(p->fft_tmap), CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, p->grids,
                                      dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                      CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

// Passes 2 and 3 of transforms [slot0, slot0 + ntrans) in one persistent kernel (n >= 2^20): compact modes out,
// fine grids left indeterminate.  Default: the bulk-asynchronous (TMA + mbarrier) kernel, one CTA per SM;
// opts.reserved[0] = 1 selects the first version (per-thread loads, four 128-thread CTAs per SM), kept for comparison.
cudaError_t launch_own_fft_pass23(ls_plan_s* p, int slot0, int ntrans, cudaStream_t s) {
    FftArgs a;
    fill_common(p, a, slot0, 0);
    const int nslabs = ntrans * (a.R1 / kC23);
    if (p->opts.reserved[0] == 1) {
        const int nblk = std::min(nslabs * 256, (512 / (16 * kC23)) * p->num_sms);
        ls_fft_pass23_kernel<kC23><<<nblk, 16 * kC23, k23Smem, s>>>(a, nslabs, p->fft_queue);
        return cudaGetLastError();
    }
    const int nblk = std::min(nslabs * 256, p->num_sms);
    const CUtensorMap& tm = *reinterpret_cast<const CUtensorMap*>(p->fft_tmap);
    const int lag = p->opts.reserved[1] ? p->opts.reserved[1] : kLagTma;
    if (p->opts.reserved[0] == 2)
        ls_fft_pass23_tma_kernel<3><<<nblk, k23threads(3), k23TmaSmem, s>>>(a, tm, slot0 * a.R1, nslabs, lag, p->fft_queue);
    else
        ls_fft_pass23_tma_kernel<4><<<nblk, k23threads(4), k23TmaSmem, s>>>(a, tm, slot0 * a.R1, nslabs, lag, p->fft_queue);
    return cudaGetLastError();
}

// Pass 3 -> compact modes, transforms [slot0, slot0 + ntrans).
cudaError_t launch_own_fft_pass3(ls_plan_s* p, int slot0, int ntrans, cudaStream_t s) {
    if (ntrans <= 0) return cudaSuccess;
    if (p->dtype == LS_F32) return launch_own_fft_f32_pass3(p, slot0, ntrans, s);
    FftArgs a;
    fill_common(p, a, slot0, 0);
    dim3 g3(a.R1 * a.R2 / kC, 1, ntrans);
    ls_fft_rows_kernel<false><<<g3, kFftThreads, kRowsSmem, s>>>(a);
    return cudaGetLastError();
}

// Pass 3 of the h transforms in slots [h_slot0, h_slot0 + nseries), fused with K5 + K6: power of series
// series0 + i from its h modes (registers) and the compact (w, w2) modes in slots w_slot, w2_slot.
cudaError_t launch_own_fft_assemble(ls_plan_s* p, int h_slot0, int nseries, int series0, int w_slot, int w2_slot,
                                    void* power, cudaStream_t s) {
    FftArgs a;
    fill_common(p, a, h_slot0, 0);
    a.w_modes = (const double2*)p->modes + (long long)w_slot * p->Nf;
    a.w2_modes = (const double2*)p->modes + (long long)w2_slot * p->Nf;
    a.power = (double*)power;
    a.series0 = series0;
    if (series0 == 0) {                                    // first pass of the execute: the (w, w2) modes are new
        ls_freq_table_kernel<<<(unsigned)((p->Nf + 255) / 256), 256, 0, s>>>(a.w_modes, a.w2_modes, a.dinv, a.Nf, a.half, a.no_float,
                                                                            (double2*)p->ftab);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    dim3 g3(a.R1 * a.R2 / kC, 1, nseries);
    if (a.no_float || a.norm) ls_fft_rows_kernel<true, true><<<g3, kFftThreads, kRowsSmem, s>>>(a);
    else ls_fft_rows_kernel<true><<<g3, kFftThreads, kRowsSmem, s>>>(a);
    return cudaGetLastError();
}

}  // namespace lsb
