// ls_post.cu — P0 deconvolution table, and K5+K6: mode extraction, diagonal rescaling
// ("correct with a diagonal rescaling") fused with the tau / power assembly
// (north_star: "compute tan(2 omega tau), then the YY/YC/YS/CC/SS terms and the
// standard-normalised power").
//
// Mode k of the periodogram (f_k = f0 + k df) is the centred NUFFT mode k' = k - floor(Nf/2)
// (Eq. 2; readings A2, A4), stored by the FFT at index k' mod n.  Re g = C, Im g = S
// (A7).  The assembly runs in fp64 registers for both dtypes (A9).
#include "ls_internal.h"
#include "ls_power.cuh"

namespace lsb {
namespace {

constexpr int kPostThreads = 256;

// psihat(k') = (w/2) * int_{-1}^{1} phi(z) cos(pi w k' z / n) dz,  phi even -> twice the half range.
// nodes/weights: Gauss-Legendre on [0, 1].
__global__ void __launch_bounds__(kPostThreads)
ls_deconv_table_kernel(double* __restrict__ dinv, long long count, const double* __restrict__ nodes,
                       const double* __restrict__ weights, int w, double beta, double inv_n) {
    __shared__ double sz[kQuadNodes], sf[kQuadNodes];
    if (threadIdx.x < kQuadNodes) {
        const double z = nodes[threadIdx.x];
        sz[threadIdx.x] = z;
        sf[threadIdx.x] = weights[threadIdx.x] * exp(beta * (sqrt(fmax(0.0, 1.0 - z * z)) - 1.0));
    }
    __syncthreads();
    const long long k = (long long)blockIdx.x * kPostThreads + threadIdx.x;
    if (k >= count) return;
    const double a = (double)w * (double)k * inv_n;      // argument of cos(pi a z)
    double acc = 0.0;
#pragma unroll 4
    for (int i = 0; i < kQuadNodes; ++i) acc = fma(sf[i], cospi(a * sz[i]), acc);
    dinv[k] = 1.0 / ((double)w * acc);                   // (w/2) * 2 * sum
}

template <typename T>
struct V2;
template <>
struct V2<double> { using type = double2; };
template <>
struct V2<float> { using type = float2; };

struct AssembleArgs {
    const void* grids;              // fine grids after the FFT, or (compact) the own FFT's [slots][Nf] mode array
    long long n, Nf;
    long long k0, k1;               // frequencies [k0, k1) of this launch
    long long stride;               // elements between transforms: n, or Nf when compact
    int compact;                    // 1: mode k of a transform sits at index k
    int no_float;                   // opts.no_floating_mean: the (S, C) sums of the weights drop out
    int norm;                       // opts.normalization
    long long half;                 // floor(Nf/2)
    const double* dinv;
    const double* sums;
    int series0, dy_per_series;
    int h_slot, h_stride, w_slot, w_stride, w2_slot, w2_stride;
    void* power;
};

template <typename T>
__global__ void __launch_bounds__(kPostThreads)
ls_assemble_kernel(const AssembleArgs a) {
    using T2 = typename V2<T>::type;
    const long long k = a.k0 + (long long)blockIdx.x * kPostThreads + threadIdx.x;
    if (k >= a.k1) return;
    const int i = blockIdx.y;                      // series within this pass
    const int s = a.series0 + i;
    const long long kp = k - a.half;               // centred mode k'
    const long long idx = a.compact ? k : (kp < 0 ? kp + a.n : kp);
    const double d = a.dinv[kp < 0 ? -kp : kp];
    const T2* g = reinterpret_cast<const T2*>(a.grids);
    const T2 gh = __ldcs(&g[(long long)(a.h_slot + i * a.h_stride) * a.stride + idx]);
    const T2 gw = g[(long long)(a.w_slot + i * a.w_stride) * a.stride + idx];
    const T2 g2 = g[(long long)(a.w2_slot + i * a.w2_stride) * a.stride + idx];
    const double YY = a.sums[4 * s + 2], W = a.sums[a.dy_per_series ? 4 * s : 0];
    const double dw = a.no_float ? 0.0 : d;        // fixed mean: S = C = 0
    const double P = assemble_power((double)gh.y * d, (double)gh.x * d, (double)gw.y * dw, (double)gw.x * dw,
                                    (double)g2.y * d, (double)g2.x * d, 1.0 / YY);
    reinterpret_cast<T*>(a.power)[(long long)s * a.Nf + k] = (T)apply_normalization(P, a.norm, YY, W);
}

// Batch with shared dy: the (w, w2) transforms and hence FreqTerms are common to all series, so one
// thread owns a frequency, computes them once and streams kSeriesPerThread series' h-modes through.
constexpr int kSeriesPerThread = 16;
template <typename T>
__global__ void __launch_bounds__(kPostThreads)
ls_assemble_shared_kernel(const AssembleArgs a, int nseries) {
    using T2 = typename V2<T>::type;
    const long long k = a.k0 + (long long)blockIdx.x * kPostThreads + threadIdx.x;
    if (k >= a.k1) return;
    const long long kp = k - a.half;
    const long long idx = a.compact ? k : (kp < 0 ? kp + a.n : kp);
    const double d = a.dinv[kp < 0 ? -kp : kp];
    const T2* g = reinterpret_cast<const T2*>(a.grids);
    const T2 gw = g[(long long)a.w_slot * a.stride + idx];
    const T2 g2 = g[(long long)a.w2_slot * a.stride + idx];
    const double dw = a.no_float ? 0.0 : d;        // fixed mean: S = C = 0
    const FreqTerms f = freq_terms((double)gw.y * dw, (double)gw.x * dw, (double)g2.y * d, (double)g2.x * d);
    const double W = a.sums[0];
    const int i0 = blockIdx.y * kSeriesPerThread;
    const int i1 = min(i0 + kSeriesPerThread, nseries);
#pragma unroll 4
    for (int i = i0; i < i1; ++i) {
        const int s = a.series0 + i;
        const T2 gh = __ldcs(&g[(long long)(a.h_slot + i) * a.stride + idx]);
        const double YY = a.sums[4 * s + 2];
        const double P = series_power(f, (double)gh.y * d, (double)gh.x * d, 1.0 / YY);
        __stcs(&reinterpret_cast<T*>(a.power)[(long long)s * a.Nf + k], (T)apply_normalization(P, a.norm, YY, W));
    }
}

template <typename T>
__global__ void ls_debug_modes_kernel(const void* grids, long long n, long long stride, int compact, long long half, const double* dinv,
                                      int h_slot, int w_slot, int w2_slot, long long K,
                                      const long long* kidx, double* out) {
    using T2 = typename V2<T>::type;
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= K) return;
    const long long kp = kidx[q] - half;
    const long long idx = compact ? kidx[q] : (kp < 0 ? kp + n : kp);
    const double d = dinv[kp < 0 ? -kp : kp];
    const T2* g = reinterpret_cast<const T2*>(grids);
    const T2 gh = g[(long long)h_slot * stride + idx], gw = g[(long long)w_slot * stride + idx], g2 = g[(long long)w2_slot * stride + idx];
    double* o = out + 6 * q;
    o[0] = (double)gh.y * d; o[1] = (double)gh.x * d;
    o[2] = (double)gw.y * d; o[3] = (double)gw.x * d;
    o[4] = (double)g2.y * d; o[5] = (double)g2.x * d;
}

// K6 alone, on sums handed in by a test (stage pin: the oracle's exact sums in, power out)
__global__ void ls_debug_assemble_kernel(long long K, const double* __restrict__ sums, double YY, double W, int no_float,
                                         int norm, double* __restrict__ out) {
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= K) return;
    const double* g = sums + 6 * q;                  // (Sh, Ch, S, C, S2, C2)
    const double P = assemble_power(g[0], g[1], no_float ? 0.0 : g[2], no_float ? 0.0 : g[3], g[4], g[5], 1.0 / YY);
    out[q] = apply_normalization(P, norm, YY, W);
}

}  // namespace

cudaError_t launch_debug_assemble(int64_t K, const double* d_sums, double YY, double W, int no_float, int norm,
                                  double* d_out, cudaStream_t s) {
    ls_debug_assemble_kernel<<<(unsigned)((K + 127) / 128), 128, 0, s>>>(K, d_sums, YY, W, no_float, norm, d_out);
    return cudaGetLastError();
}

cudaError_t launch_deconv_table(ls_plan_s* p, const double* nodes, const double* weights, cudaStream_t s) {
    const long long count = p->Nf / 2 + 1;
    const int nb = (int)((count + kPostThreads - 1) / kPostThreads);
    ls_deconv_table_kernel<<<nb, kPostThreads, 0, s>>>(p->dinv, count, nodes, weights, p->w, p->beta,
                                                       1.0 / (double)p->n);
    return cudaGetLastError();
}

cudaError_t launch_assemble(ls_plan_s* p, int series0, int nseries, int h_slot, int h_stride, int w_slot,
                            int w_stride, int w2_slot, int w2_stride, void* power, cudaStream_t s, long long k0, long long k1) {
    AssembleArgs a;
    a.k0 = k0;
    a.k1 = k1 < 0 ? p->Nf : k1;
    a.grids = p->own_fft ? p->modes : p->grids;
    a.n = p->n;
    a.Nf = p->Nf;
    a.stride = p->own_fft ? p->Nf : p->n;
    a.compact = p->own_fft ? 1 : 0;
    a.no_float = p->opts.no_floating_mean;
    a.norm = p->opts.normalization;
    a.half = p->Nf / 2;
    a.dinv = p->dinv;
    a.sums = p->sums;
    a.series0 = series0;
    a.dy_per_series = p->opts.dy_per_series;
    a.h_slot = h_slot; a.h_stride = h_stride;
    a.w_slot = w_slot; a.w_stride = w_stride;
    a.w2_slot = w2_slot; a.w2_stride = w2_stride;
    a.power = power;
    const unsigned gx = (unsigned)((a.k1 - a.k0 + kPostThreads - 1) / kPostThreads);
    if (nseries > 1 && h_stride == 1 && w_stride == 0 && w2_stride == 0) {       // shared dy
        dim3 grid(gx, (nseries + kSeriesPerThread - 1) / kSeriesPerThread);
        if (p->dtype == LS_F64) ls_assemble_shared_kernel<double><<<grid, kPostThreads, 0, s>>>(a, nseries);
        else ls_assemble_shared_kernel<float><<<grid, kPostThreads, 0, s>>>(a, nseries);
    } else {
        dim3 grid(gx, nseries);
        if (p->dtype == LS_F64) ls_assemble_kernel<double><<<grid, kPostThreads, 0, s>>>(a);
        else ls_assemble_kernel<float><<<grid, kPostThreads, 0, s>>>(a);
    }
    return cudaGetLastError();
}

cudaError_t launch_debug_modes(ls_plan_s* p, int h_slot, int w_slot, int w2_slot, int64_t K,
                               const int64_t* d_kidx, double* d_out, cudaStream_t s) {
    const int nb = (int)((K + 127) / 128);
    if (p->dtype == LS_F64)
        ls_debug_modes_kernel<double><<<nb, 128, 0, s>>>(p->own_fft ? p->modes : p->grids, p->n, p->own_fft ? p->Nf : p->n, p->own_fft ? 1 : 0, p->Nf / 2, p->dinv, h_slot, w_slot, w2_slot,
                                                         K, (const long long*)d_kidx, d_out);
    else
        ls_debug_modes_kernel<float><<<nb, 128, 0, s>>>(p->own_fft ? p->modes : p->grids, p->n, p->own_fft ? p->Nf : p->n, p->own_fft ? 1 : 0, p->Nf / 2, p->dinv, h_slot, w_slot, w2_slot,
                                                        K, (const long long*)d_kidx, d_out);
    return cudaGetLastError();
}

}  // namespace lsb
