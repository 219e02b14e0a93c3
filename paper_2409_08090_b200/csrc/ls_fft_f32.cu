// ls_fft_f32.cu — the library's own fine-grid FFT for complex64 grids of n = 5 x 2^k cells, k = 22 .. 25
// ("the FFT time dominates"; built for config 5: N_f = 1.25e8, fp32).
//
//   B_k = sum_l b_l e^{+2 pi i k l / n}     (reading A7: the unnormalised inverse transform)
//
// The power of two above 1.25 N_f is up to 2 x too large (config 5: 2^28 against 1.56e8 wanted), so the plan used to take a
// 2,3,5-smooth size and cuFFT (five passes over the grids at n = 157 464 000).  5 x 2^25 = 167 772 160 cells is three
// passes, decimation in frequency, n = R1 x 256 x 512 with R1 = 80 RM = 16 x RM x 5 (RM = 2, 4, 8, 16):
//   l = l1 (256 x 512) + l2 512 + l3,   k = k1 + R1 k2 + R1 256 k3
//   pass 1: FFT over l1 -> k1 (row stride 131 072 cells), times w_n^{k1 (512 l2 + l3)};  layout [k1][l2][l3], in place.
//           Rows of spreading tiles that hold no points are not loaded (liveness masks of ls_tile_list_kernel): with
//           clustered sampling 95 % of the tiles are empty, and the spreading kernel never writes them either.
//   pass 2: FFT over l2 -> k2 (stride 512 cells), times w_n^{R1 k2 l3};                  layout [k1][k2][l3], in place
//   pass 3: FFT over l3 -> k3 (contiguous); the kept modes k' = k - floor(Nf/2) go to the compact [M][Nf] array in
//           frequency order (16 consecutive k1 per CTA: 128-byte runs).
// Arithmetic in fp32; every twiddle comes from a double-precision table (w_n: the plan's two 4096-entry-style tables of
// ls_fft.cu) or a double sincospi and is rounded once.  The fp64 kernels of ls_fft.cu are not touched by this file.
#include "ls_internal.h"

namespace lsb {
namespace {

constexpr long long kInner = 256LL * 512LL;      // cells per pass-1 row
constexpr int kC1 = 8;                           // columns per CTA, pass 1
constexpr int kC2 = 16;                          // columns per CTA, pass 2
constexpr int kC3 = 16;                          // rows (consecutive k1) per CTA, pass 3

struct F32Args {
    float2* grids;             // [ntrans][n], in place
    long long n;
    int R1;
    const double2* wlo;        // w_n^x, x < 4096
    const double2* whi;        // w_n^{4096 y}, y < n / 4096
    const unsigned* row_masks; // pass 1: bit (row / rb) of word [(set * ncoltiles + ct) * rb + row % rb]
    int ncoltiles, rb, tile_shift, set_of_trans_first;
    float2* modes;             // [ntrans][Nf]
    long long Nf, half;
};

// Complex arithmetic on Blackwell's packed fp32 pairs (add / sub / mul / fma .f32x2 -> FADD2, FMUL2, FFMA2): one
// instruction per complex add and two per complex product instead of two and four.  The fp32 pipe does the same flops per
// clock either way (measured: 72 - 74 TFLOP/s with FFMA and with FFMA2); what halves is the ISSUE slots, and these kernels
// are issue-bound (profiles/r2_cfg5.md).  ptxas folds the packing moves, the (-y, x) swizzle of a multiplication by i and
// the (x, x) broadcasts into operand modifiers.  Same roundings as the scalar forms.
__device__ __forceinline__ unsigned long long pk(float2 a) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y));
    return r;
}
__device__ __forceinline__ float2 upk(unsigned long long r) {
    float2 a;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a.x), "=f"(a.y) : "l"(r));
    return a;
}
__device__ __forceinline__ float2 add2(float2 a, float2 b) {
    unsigned long long d;
    asm("add.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pk(a)), "l"(pk(b)));
    return upk(d);
}
__device__ __forceinline__ float2 sub2(float2 a, float2 b) {
    unsigned long long d;
    asm("sub.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pk(a)), "l"(pk(b)));
    return upk(d);
}
__device__ __forceinline__ float2 mul2(float2 a, float2 b) {
    unsigned long long d;
    asm("mul.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pk(a)), "l"(pk(b)));
    return upk(d);
}
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(pk(a)), "l"(pk(b)), "l"(pk(c)));
    return upk(d);
}
// PK = false keeps the scalar forms: pass 2 runs at the DRAM roofline and was 5 % SLOWER with the packed ones (1.28 ms
// against 1.22: more register-pair moves), passes 1 and 3 gained 8 % and 1 %.
template <bool PK = true>
__device__ __forceinline__ float2 cadd(float2 a, float2 b) {
    if constexpr (PK) return add2(a, b);
    else return make_float2(a.x + b.x, a.y + b.y);
}
template <bool PK = true>
__device__ __forceinline__ float2 csub(float2 a, float2 b) {
    if constexpr (PK) return sub2(a, b);
    else return make_float2(a.x - b.x, a.y - b.y);
}
// (a.x w.x - a.y w.y, a.x w.y + a.y w.x) = (a.x, a.x) (w.x, w.y) + (a.y, a.y) (-w.y, w.x)
template <bool PK = true>
__device__ __forceinline__ float2 cmul(float2 a, float2 w) {
    if constexpr (PK) return fma2(make_float2(a.x, a.x), w, mul2(make_float2(a.y, a.y), make_float2(-w.y, w.x)));
    else return make_float2(fmaf(a.x, w.x, -a.y * w.y), fmaf(a.x, w.y, a.y * w.x));
}
__device__ __forceinline__ float2 cmuli(float2 a) { return make_float2(-a.y, a.x); }
__device__ __forceinline__ double2 cmuld(double2 a, double2 w) { return make_double2(fma(a.x, w.x, -a.y * w.y), fma(a.x, w.y, a.y * w.x)); }
__device__ __forceinline__ float2 to_f(double2 w) { return make_float2((float)w.x, (float)w.y); }

constexpr float kC1f = 0.92387953251128675613f, kS1f = 0.38268343236508977173f, kR2f = 0.70710678118654752440f;

template <bool PK = true>
__device__ __forceinline__ void fft4(float2& a, float2& b, float2& c, float2& d) {
    const float2 t0 = cadd<PK>(a, c), t1 = csub<PK>(a, c), t2 = cadd<PK>(b, d), t3 = cmuli(csub<PK>(b, d));
    a = cadd<PK>(t0, t2);
    b = cadd<PK>(t1, t3);
    c = csub<PK>(t0, t2);
    d = csub<PK>(t1, t3);
}
// X_k = sum_l x_l e^{+2 pi i k l / 16}, in place; X_k ends at position pos16(k)
__device__ __forceinline__ constexpr int pos16(int k) { return 4 * (k & 3) + (k >> 2); }
template <bool PK = true>
__device__ __forceinline__ void fft16(float2 (&x)[16]) {
#pragma unroll
    for (int b = 0; b < 4; ++b) fft4<PK>(x[b], x[4 + b], x[8 + b], x[12 + b]);
    x[5] = cmul<PK>(x[5], make_float2(kC1f, kS1f));
    x[6] = cmul<PK>(x[6], make_float2(kR2f, kR2f));
    x[7] = cmul<PK>(x[7], make_float2(kS1f, kC1f));
    x[9] = cmul<PK>(x[9], make_float2(kR2f, kR2f));
    x[10] = cmuli(x[10]);
    x[11] = cmul<PK>(x[11], make_float2(-kR2f, kR2f));
    x[13] = cmul<PK>(x[13], make_float2(kS1f, kC1f));
    x[14] = cmul<PK>(x[14], make_float2(-kR2f, kR2f));
    x[15] = cmul<PK>(x[15], make_float2(-kC1f, -kS1f));
#pragma unroll
    for (int ka = 0; ka < 4; ++ka) fft4<PK>(x[4 * ka], x[4 * ka + 1], x[4 * ka + 2], x[4 * ka + 3]);
}
__device__ __forceinline__ void fft8(float2 (&x)[8]) {       // X_k at position 2 (k & 3) + (k >> 2)
    fft4(x[0], x[2], x[4], x[6]);
    fft4(x[1], x[3], x[5], x[7]);
    x[3] = cmul(x[3], make_float2(kR2f, kR2f));
    x[5] = cmuli(x[5]);
    x[7] = cmul(x[7], make_float2(-kR2f, kR2f));
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float2 e = x[2 * k], o = x[2 * k + 1];
        x[2 * k] = cadd(e, o);
        x[2 * k + 1] = csub(e, o);
    }
}
template <int RB>
__device__ __forceinline__ constexpr int fft_pos(int k) {
    return RB == 16 ? 4 * (k & 3) + (k >> 2) : RB == 8 ? 2 * (k & 3) + (k >> 2) : k;
}
template <int RB>
__device__ __forceinline__ void fft_small(float2 (&x)[RB]) {
    if constexpr (RB == 16) fft16(x);
    else if constexpr (RB == 8) fft8(x);
    else if constexpr (RB == 4) fft4(x[0], x[1], x[2], x[3]);
    else {
        const float2 a = x[0], b = x[1];
        x[0] = cadd(a, b);
        x[1] = csub(a, b);
    }
}
constexpr float kCos5a = 0.30901699437494742410f, kCos5b = -0.80901699437494742410f;
constexpr float kSin5a = 0.95105651629515357212f, kSin5b = 0.58778525229247312917f;
__device__ __forceinline__ void fft5(float2 (&x)[5]) {       // natural order
    const float2 t1 = cadd(x[1], x[4]), t2 = cadd(x[2], x[3]), t3 = csub(x[1], x[4]), t4 = csub(x[2], x[3]);
    const float2 ca = make_float2(kCos5a, kCos5a), cb = make_float2(kCos5b, kCos5b);
    const float2 sa = make_float2(kSin5a, kSin5a), sb = make_float2(kSin5b, kSin5b);
    const float2 a1 = fma2(cb, t2, fma2(ca, t1, x[0]));
    const float2 a2 = fma2(ca, t2, fma2(cb, t1, x[0]));
    const float2 b1 = fma2(sb, t4, mul2(sa, t3));
    const float2 b2 = fma2(sb, t3, mul2(make_float2(-kSin5a, -kSin5a), t4));
    x[0] = cadd(x[0], cadd(t1, t2));
    x[1] = cadd(a1, cmuli(b1));                          // a1 + i b1
    x[4] = csub(a1, cmuli(b1));
    x[2] = cadd(a2, cmuli(b2));
    x[3] = csub(a2, cmuli(b2));
}

// w_n^e, e < n, in double from the two tables (e = 4096 e_hi + e_lo)
__device__ __forceinline__ double2 twiddle_n(const F32Args& a, unsigned e) {
    return cmuld(__ldg(&a.wlo[e & 4095u]), __ldg(&a.whi[e >> 12]));
}

// warp-uniform twiddles as constant-bank operands: stage 2 of pass 1, w_{5 RM}^{kp q} as [log2 RM - 1][q][kp], and the
// radix-2 layer of the 32-point transform of pass 3, w_32^k
__constant__ float2 cTw5f[4][5][16];
__constant__ float2 cW32[16];

// Pass 1: radix R1 = 16 x RM x 5 over l1 (row stride 131 072 cells), one CTA = R1 rows x 8 columns held in shared memory
// ([ka][j][c]) between the three stages, 5 RM thread rows x 4 column pairs.  l1 = J i + j (J = 5 RM), j = 5 p + q;
// k1 = ka + 16 (kp + RM kq).  Same structure as ls_fft_cols5_kernel (ls_fft.cu), in fp32 and with a long row stride.
// Liveness: row l1 of column tile ct is bit (l1 / rb) of word [(set ncoltiles + ct) rb + l1 % rb], rb = J / 2 = R1 / 32,
// so the 16 rows J i + j of a thread are bits 2 i + (j / rb) of ONE word.
template <int RM>
constexpr size_t pass1_smem() { return sizeof(float2) * ((size_t)16 * (5 * RM + 1) * kC1 + 80 * RM) + sizeof(double2) * 2 * kC1; }   // tile (padded) + table + column steps
// TWO adjacent columns per thread (5 RM x 4 threads per CTA): every shared-memory and global access is 16 bytes, the index
// arithmetic and the stage twiddles are shared by the two columns (1.65 -> 1.61 ms at config 5 against one column per
// thread; 16 columns per CTA for 128-byte row segments, one 640-thread CTA per SM: 1.70 ms).
template <int RM>
__global__ void __launch_bounds__(5 * RM * (kC1 / 2), RM == 16 ? 2 : 1)
ls_f32_pass1_kernel(const F32Args a) {
    constexpr int J = 5 * RM, R1 = 16 * J, RBW = J / 2, NT = J * (kC1 / 2);
    // rows of 8 float2 = 64 bytes, J + 1 rows per ka: a warp's consecutive ka then alternate between the two halves of the
    // 128-byte bank line (with J rows they all start at bank 0: every access of stages 2 and 3 was a 2-way conflict)
    constexpr int JP = J + 1;
    extern __shared__ __align__(16) unsigned char fsm[];
    float2* S = reinterpret_cast<float2*>(fsm);              // [ka][j (padded to JP)][c]
    float2* wr = S + 16 * JP * kC1;                          // [ka][j] = w_R1^{ka j}: a warp's lookups are consecutive entries
    for (int x = threadIdx.x; x < R1; x += NT) {
        double sn, cs;
        sincospi(2.0 * (double)((x / J) * (x % J)) / (double)R1, &sn, &cs);
        wr[x] = make_float2((float)cs, (float)sn);
    }
    double2* colw = reinterpret_cast<double2*>(wr + R1);     // [2][kC1]: w_n^{J m}, w_n^{16 RM m} of the CTA's columns
    if (threadIdx.x < 2 * kC1) {
        const long long mc = (long long)blockIdx.x * kC1 + (threadIdx.x % kC1);
        const long long e = (threadIdx.x < kC1 ? (long long)J : 16LL * RM) * mc;
        sincospi(2.0 * (double)e / (double)a.n, &colw[threadIdx.x].y, &colw[threadIdx.x].x);
    }
    const int c = 2 * (threadIdx.x % (kC1 / 2)), tj = threadIdx.x / (kC1 / 2);      // columns c, c + 1
    const long long m = (long long)blockIdx.x * kC1 + c;
    const int tr = blockIdx.y;
    float2* base = a.grids + (long long)tr * a.n + m;
    auto ld2 = [](const float2* p, float2& u, float2& v) {
        const float4 q = *reinterpret_cast<const float4*>(p);
        u = make_float2(q.x, q.y);
        v = make_float2(q.z, q.w);
    };
    auto st2 = [](float2* p, float2 u, float2 v) { *reinterpret_cast<float4*>(p) = make_float4(u.x, u.y, v.x, v.y); };
    {
        const int j = tj;
        unsigned live = 0xffffffffu;
        if (a.row_masks) {
            const int set = tr < a.set_of_trans_first ? 0 : 1;
            const int ct = (int)(m >> a.tile_shift);
            live = __ldg(&a.row_masks[((long long)set * a.ncoltiles + ct) * RBW + (j % RBW)]);
        }
        live >>= (j / RBW);
        float2 x[16], y[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            x[i] = y[i] = make_float2(0.f, 0.f);
            if ((live >> (2 * i)) & 1u) ld2(base + (long long)(J * i + j) * kInner, x[i], y[i]);
        }
        fft16(x);
        fft16(y);
        __syncthreads();                                     // table ready
#pragma unroll
        for (int ka = 0; ka < 16; ++ka) {
            const float2 t = wr[ka * J + j];
            st2(&S[(ka * JP + j) * kC1 + c], cmul(x[pos16(ka)], t), cmul(y[pos16(ka)], t));
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 80 / J; ++r) {                       // stage 2: butterfly (ka, q), elements S[ka][5 p + q]
        const int b = tj + J * r, ka = b & 15, q = b >> 4;
        float2 u[RM], v[RM];
#pragma unroll
        for (int p = 0; p < RM; ++p) ld2(&S[(ka * JP + 5 * p + q) * kC1 + c], u[p], v[p]);
        fft_small<RM>(u);
        fft_small<RM>(v);
#pragma unroll
        for (int kp = 0; kp < RM; ++kp) {
            const float2 t = cTw5f[RM == 2 ? 0 : RM == 4 ? 1 : RM == 8 ? 2 : 3][q][kp];
            st2(&S[(ka * JP + 5 * kp + q) * kC1 + c], cmul(u[fft_pos<RM>(kp)], t), cmul(v[fft_pos<RM>(kp)], t));
        }
    }
    __syncthreads();
    // stage 3: butterfly b = ka + 16 kp = tj + J r (elements S[ka][5 kp + q]), outputs k1 = b + 16 RM kq times the inter-pass
    // twiddle w_n^{k1 m} = w_n^{b m} (w_n^{16 RM m})^kq.  No table lookups: a warp's 32 gathered 16-byte entries cost the
    // load/store unit as much as sixteen of its shared-memory accesses.  Per column the base w_n^{tj m} is one double
    // sincospi; its step over r, w_n^{J m}, and the step over kq, w_n^{16 RM m}, depend on the column only and sit in shared
    // memory (colw); the five-term chain over kq runs in fp32.
    double2 twb0, twb1;
    sincospi(2.0 * (double)((long long)tj * m) / (double)a.n, &twb0.y, &twb0.x);
    sincospi(2.0 * (double)((long long)tj * (m + 1)) / (double)a.n, &twb1.y, &twb1.x);
    const double2 stb0 = colw[c], stb1 = colw[c + 1];
    const float2 sq0 = to_f(colw[kC1 + c]), sq1 = to_f(colw[kC1 + c + 1]);
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const int b = tj + J * r;
        if (b < 16 * RM) {
            const int ka = b & 15, kp = b >> 4;
            float2 z0[5], z1[5];
#pragma unroll
            for (int q = 0; q < 5; ++q) ld2(&S[(ka * JP + 5 * kp + q) * kC1 + c], z0[q], z1[q]);
            fft5(z0);
            fft5(z1);
            float2 t0 = to_f(twb0), t1 = to_f(twb1);
#pragma unroll
            for (int kq = 0; kq < 5; ++kq) {
                st2(base + (long long)(b + 16 * RM * kq) * kInner, cmul(z0[kq], t0), cmul(z1[kq], t1));
                t0 = cmul(t0, sq0);
                t1 = cmul(t1, sq1);
            }
        }
        twb0 = cmuld(twb0, stb0);
        twb1 = cmuld(twb1, stb1);
    }
}

// Pass 2: 256-point FFTs over l2 (stride 512 cells) for 16 consecutive l3 of one row k1; in place; then w_n^{R1 k2 l3}.
constexpr size_t kPass2Smem = sizeof(float2) * (256 * kC2 + 256);
__global__ void __launch_bounds__(256)
ls_f32_pass2_kernel(const F32Args a) {
    extern __shared__ __align__(16) unsigned char fsm[];
    float2* Y = reinterpret_cast<float2*>(fsm);              // [ka][j][c]
    float2* w256 = Y + 256 * kC2;                            // [ka][j] = w_256^{ka j}
    for (int i = threadIdx.x; i < 256; i += 256) {
        double sn, cs;
        sincospi((double)((i >> 4) * (i & 15)) / 128.0, &sn, &cs);
        w256[i] = make_float2((float)cs, (float)sn);
    }
    const int c = threadIdx.x % kC2, hi = threadIdx.x / kC2;
    const int m = blockIdx.x * kC2 + c;                      // l3
    const int k1 = blockIdx.y, tr = blockIdx.z;
    float2* base = a.grids + (long long)tr * a.n + (long long)k1 * kInner + m;
    float2 x[16];
    {
        const int j = hi;
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = base[(16 * i + j) * 512];
        fft16<false>(x);
        __syncthreads();
#pragma unroll
        for (int ka = 0; ka < 16; ++ka) Y[(ka * 16 + j) * kC2 + c] = cmul<false>(x[pos16(ka)], w256[ka * 16 + j]);
    }
    __syncthreads();
    {
        const int ka = hi;
#pragma unroll
        for (int j = 0; j < 16; ++j) x[j] = Y[(ka * 16 + j) * kC2 + c];
        fft16<false>(x);
        // k2 = ka + 16 kb; exponent k2 l3 R1 < n; two interleaved chains (even / odd kb) in double
        const unsigned mm = (unsigned)m * (unsigned)a.R1;
        double2 tw = twiddle_n(a, (unsigned)ka * mm);
        const double2 st = twiddle_n(a, 16u * mm);
        double2 tw1 = cmuld(tw, st);
        const double2 st2 = cmuld(st, st);
#pragma unroll
        for (int kb = 0; kb < 16; kb += 2) {
            base[(ka + 16 * kb) * 512] = cmul<false>(x[pos16(kb)], to_f(tw));
            base[(ka + 16 * kb + 16) * 512] = cmul<false>(x[pos16(kb + 1)], to_f(tw1));
            tw = cmuld(tw, st2);
            tw1 = cmuld(tw1, st2);
        }
    }
}

// Pass 3: 512-point FFTs over l3 (contiguous rows of 4 KB) of 16 consecutive k1 at one k2; 512 = 16 x 32: every thread
// does two 16-point transforms (columns jj and jj + 16 of the 16 x 32 view), one exchange, then one 32-point transform
// (two 16-point ones and a radix-2 layer).  Output: mode k = k1 + R1 k2 + 256 R1 k3, stored at (k + half) mod n if that
// is below Nf — the compact, centred layout the assembly kernel reads.
constexpr size_t kPass3Smem = sizeof(float2) * (512 * (kC3 + 1) + 512);
// measured and not kept: three CTAs per SM at 80 registers (1.70 ms against 1.61), 32 rows per CTA for 256-byte output
// runs (one 512-thread CTA per SM: 1.74 ms)
__global__ void __launch_bounds__(16 * kC3, kC3 == 16 ? 2 : 1)
ls_f32_pass3_kernel(const F32Args a) {
    extern __shared__ __align__(16) unsigned char fsm[];
    float2* S = reinterpret_cast<float2*>(fsm);              // [ka][jj][17]
    float2* w512 = S + 512 * (kC3 + 1);
    for (int i = threadIdx.x; i < 512; i += 16 * kC3) {      // [ka][h][jl] = w_512^{ka (2 jl + h)}: consecutive entries per warp
        double sn, cs;
        sincospi((double)((i >> 5) * (2 * (i & 15) + ((i >> 4) & 1))) / 256.0, &sn, &cs);
        w512[i] = make_float2((float)cs, (float)sn);
    }
    const int k1b = blockIdx.x * kC3, k2 = blockIdx.y, tr = blockIdx.z;
    const float2* src = a.grids + (long long)tr * a.n;
    __syncthreads();
    {
        const int jl = threadIdx.x & 15, c = threadIdx.x >> 4;
        const float2* row = src + ((long long)(k1b + c) * 256 + k2) * 512;
        // the thread takes the adjacent columns jj = 2 jl and 2 jl + 1 of the 16 x 32 view: sixteen 16-byte loads; column
        // jj is kept at position (jj & 1) 16 + (jj >> 1) of S, which is how the 32-point stage wants it (evens, then odds)
        float2 x0[16], x1[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const float4 v = __ldcs(reinterpret_cast<const float4*>(row) + 16 * i + jl);
            x0[i] = make_float2(v.x, v.y);
            x1[i] = make_float2(v.z, v.w);
        }
        fft16(x0);
#pragma unroll
        for (int ka = 0; ka < 16; ++ka) S[(ka * 32 + jl) * (kC3 + 1) + c] = cmul(x0[pos16(ka)], w512[ka * 32 + jl]);
        fft16(x1);
#pragma unroll
        for (int ka = 0; ka < 16; ++ka) S[(ka * 32 + jl + 16) * (kC3 + 1) + c] = cmul(x1[pos16(ka)], w512[ka * 32 + jl + 16]);
    }
    __syncthreads();
    {
        const int c = threadIdx.x % kC3, ka = threadIdx.x / kC3;
        float2 e[16], o[16];
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            e[q] = S[(ka * 32 + q) * (kC3 + 1) + c];
            o[q] = S[(ka * 32 + 16 + q) * (kC3 + 1) + c];
        }
        fft16(e);
        fft16(o);
        float2* out = a.modes + (long long)tr * a.Nf;
        const long long kk0 = (long long)(k1b + c) + (long long)a.R1 * k2;
        const long long r12 = (long long)a.R1 * 256;
#pragma unroll
        for (int kq = 0; kq < 16; ++kq) {
            const float2 E = e[pos16(kq)], O = cmul(o[pos16(kq)], cW32[kq]);
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int k3 = ka + 16 * (kq + 16 * h);
                long long k = kk0 + r12 * k3 + a.half;
                if (k >= a.n) k -= a.n;
                if (k < a.Nf) out[k] = h ? csub(E, O) : cadd(E, O);
            }
        }
    }
}

void fill_args(const ls_plan_s* p, F32Args& a, int slot0, int n_x2) {
    a.grids = (float2*)p->grids + (long long)slot0 * p->n;
    a.n = p->n;
    a.R1 = (int)(p->n / kInner);
    a.wlo = (const double2*)p->fft_wlo;
    a.whi = (const double2*)p->fft_whi;
    a.row_masks = p->fft_prune ? p->row_masks : nullptr;
    a.ncoltiles = own_fft_ncoltiles(p);
    a.rb = own_fft_rb(p);
    a.tile_shift = 0;
    while ((1 << a.tile_shift) < p->L) ++a.tile_shift;
    a.set_of_trans_first = n_x2;
    a.modes = (float2*)p->modes + (long long)slot0 * p->Nf;
    a.Nf = p->Nf;
    a.half = p->Nf / 2;
}

}  // namespace

// fp32 grids of n = 80 RM x 256 x 512 = 5 x 2^22 .. 5 x 2^25 cells: RM = 2, 4, 8, 16; else 0
int own_fft_f32_rm(const ls_plan_s* p) {
    if (p->dtype != LS_F32) return 0;
    for (int rm = 2; rm <= 16; rm *= 2)
        if (p->n == 80LL * rm * kInner) return rm;
    return 0;
}

cudaError_t own_fft_f32_init(ls_plan_s* p, cudaStream_t s) {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(ls_f32_pass1_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pass1_smem<2>())) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_f32_pass1_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pass1_smem<4>())) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_f32_pass1_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pass1_smem<8>())) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_f32_pass1_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pass1_smem<16>())) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_f32_pass2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPass2Smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(ls_f32_pass3_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPass3Smem)) != cudaSuccess) return e;
    float2 h5[4][5][16], h32[16];
    for (int v = 0; v < 4; ++v)
        for (int q = 0; q < 5; ++q)
            for (int kp = 0; kp < 16; ++kp) {
                const double ang = 2.0 * M_PI * (double)((kp * q) % (10 << v)) / (double)(10 << v);     // 5 RM = 10, 20, 40, 80
                h5[v][q][kp] = make_float2((float)cos(ang), (float)sin(ang));
            }
    for (int k = 0; k < 16; ++k) h32[k] = make_float2((float)cos(2.0 * M_PI * k / 32.0), (float)sin(2.0 * M_PI * k / 32.0));
    if ((e = cudaMemcpyToSymbolAsync(cTw5f, h5, sizeof h5, 0, cudaMemcpyHostToDevice, s)) != cudaSuccess) return e;
    if ((e = cudaMemcpyToSymbolAsync(cW32, h32, sizeof h32, 0, cudaMemcpyHostToDevice, s)) != cudaSuccess) return e;
    return cudaStreamSynchronize(s);
}

cudaError_t launch_own_fft_f32_pass1(ls_plan_s* p, int slot0, int ntrans, int n_x2, cudaStream_t s) {
    F32Args a;
    fill_args(p, a, slot0, n_x2);
    const dim3 g((unsigned)(kInner / kC1), ntrans);
    switch (own_fft_f32_rm(p)) {
        case 2: ls_f32_pass1_kernel<2><<<g, 5 * 2 * kC1 / 2, pass1_smem<2>(), s>>>(a); break;
        case 4: ls_f32_pass1_kernel<4><<<g, 5 * 4 * kC1 / 2, pass1_smem<4>(), s>>>(a); break;
        case 8: ls_f32_pass1_kernel<8><<<g, 5 * 8 * kC1 / 2, pass1_smem<8>(), s>>>(a); break;
        default: ls_f32_pass1_kernel<16><<<g, 5 * 16 * kC1 / 2, pass1_smem<16>(), s>>>(a); break;
    }
    return cudaGetLastError();
}

cudaError_t launch_own_fft_f32_pass2(ls_plan_s* p, int slot0, int ntrans, cudaStream_t s) {
    F32Args a;
    fill_args(p, a, slot0, 0);
    ls_f32_pass2_kernel<<<dim3(512 / kC2, a.R1, ntrans), 256, kPass2Smem, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_own_fft_f32_pass3(ls_plan_s* p, int slot0, int ntrans, cudaStream_t s) {
    if (ntrans <= 0) return cudaSuccess;
    F32Args a;
    fill_args(p, a, slot0, 0);
    ls_f32_pass3_kernel<<<dim3(a.R1 / kC3, 256, ntrans), 16 * kC3, kPass3Smem, s>>>(a);
    return cudaGetLastError();
}

}  // namespace lsb
