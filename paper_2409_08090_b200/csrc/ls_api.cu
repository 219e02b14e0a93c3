// ls_api.cu — the C-ABI boundary (include/ls.h): plan construction, the execute sequence,
// host-buffer execute, introspection.  Host logic only; every arithmetic step of the hot path
// runs in the kernels of ls_pre.cu / ls_spread.cu / ls_post.cu and in one cuFFT plan.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <map>
#include <mutex>
#include <new>
#include <tuple>

#include "ls_internal.h"

using lsb::dd;

namespace {

struct Pass {
    int s0, C;          // series [s0, s0 + C)
    int fft_slot0, fft_batch;
};

inline size_t real_bytes(int dtype) { return dtype == LS_F64 ? 8 : 4; }

// exact product of an integer-valued double and a double as a double-double
inline dd two_prod(double a, double b) {
    dd r;
    r.hi = a * b;
    r.lo = fma(a, b, -r.hi);
    return r;
}
// double-double + double (Knuth two-sum, then renormalise)
inline dd dd_add_d(dd a, double b) {
    const double s = a.hi + b;
    const double bb = s - a.hi;
    const double e = (a.hi - (s - bb)) + (b - bb);
    const double lo = e + a.lo;
    dd r;
    r.hi = s + lo;
    r.lo = lo - (r.hi - s);
    return r;
}

// smallest multiple of 4 >= lo whose prime factors are all in {2, 3, 5} (a multiple of 4 keeps every
// grid row 32-byte aligned for the vector stores of the spreading kernel, fp32 included)
int64_t next_smooth_even(int64_t lo) {
    if (lo < 4) lo = 4;
    for (int64_t m = (lo + 3) / 4 * 4;; m += 4) {
        int64_t r = m;
        while (r % 2 == 0) r /= 2;
        while (r % 3 == 0) r /= 3;
        while (r % 5 == 0) r /= 5;
        if (r == 1) return m;
    }
}

// Gauss-Legendre nodes/weights on [0, 1] (Newton on P_Q in long double).
void gauss_legendre_01(int Q, double* z, double* wt) {
    for (int i = 0; i < Q; ++i) {
        long double x = cosl(3.14159265358979323846264338327950288L * (i + 0.75L) / (Q + 0.5L));
        long double dp = 1;
        for (int it = 0; it < 100; ++it) {
            long double p0 = 1, p1 = x;
            for (int k = 2; k <= Q; ++k) {
                const long double p2 = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k;
                p0 = p1;
                p1 = p2;
            }
            dp = Q * (x * p1 - p0) / (x * x - 1);
            const long double dx = p1 / dp;
            x -= dx;
            if (fabsl(dx) < 1e-19L) break;
        }
        // recompute derivative at the converged root
        long double p0 = 1, p1 = x;
        for (int k = 2; k <= Q; ++k) {
            const long double p2 = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k;
            p0 = p1;
            p1 = p2;
        }
        dp = Q * (x * p1 - p0) / (x * x - 1);
        const long double wx = 2 / ((1 - x * x) * dp * dp);
        z[i] = (double)((x + 1) / 2);
        wt[i] = (double)(wx / 2);
    }
}

// Piecewise-polynomial fit of the ES kernel psi(s) = exp(beta (sqrt(1 - (2s/w)^2) - 1)) on each cell
// of its support: Chebyshev interpolation in eta in [-1, 1] per piece, converted to
// monomials in long double; the degree is raised until the measured error stops improving or is
// below `tol`.  Only the first ceil(w/2) pieces are kept (psi is even).
long double es_exact(long double s, int w, long double beta) {
    const long double z = 2.0L * s / w;
    const long double a = 1.0L - z * z;
    return a > 0 ? expl(beta * (sqrtl(a) - 1.0L)) : expl(-beta);
}

void fit_kernel_poly(int w, double beta, double tol, int max_deg, lsb::KernelPoly* kp) {
    const long double PI = 3.14159265358979323846264338327950288L;
    const int half = (w + 1) / 2;
    lsb::KernelPoly best{};
    double prev_err = 1e300;
    for (int D = 4; D <= max_deg; D += 2) {
        lsb::KernelPoly cur{};
        cur.w = w; cur.deg = D; cur.half = half;
        double worst = 0;
        for (int i = 0; i < half; ++i) {
            const long double centre = (long double)i - 0.5L * w + 0.5L;
            long double f[lsb::kMaxDeg + 1], a[lsb::kMaxDeg + 1];
            for (int j = 0; j <= D; ++j) f[j] = es_exact(cosl(PI * (j + 0.5L) / (D + 1)) / 2 + centre, w, beta);
            for (int k = 0; k <= D; ++k) {
                long double acc = 0;
                for (int j = 0; j <= D; ++j) acc += f[j] * cosl(PI * k * (j + 0.5L) / (D + 1));
                a[k] = acc * (k == 0 ? 1.0L : 2.0L) / (D + 1);
            }
            // sum_k a_k T_k(eta) -> monomials, T_{k+1} = 2 eta T_k - T_{k-1}
            long double m[lsb::kMaxDeg + 1] = {0}, t0[lsb::kMaxDeg + 2] = {0}, t1[lsb::kMaxDeg + 2] = {0},
                        t2[lsb::kMaxDeg + 2];
            t0[0] = 1; t1[1] = 1;
            m[0] += a[0];
            if (D >= 1) m[1] += a[1];
            for (int k = 2; k <= D; ++k) {
                for (int d = 0; d <= D; ++d) t2[d] = (d > 0 ? 2 * t1[d - 1] : 0) - t0[d];
                for (int d = 0; d <= D; ++d) { m[d] += a[k] * t2[d]; t0[d] = t1[d]; t1[d] = t2[d]; }
            }
            for (int d = 0; d <= lsb::kMaxDeg; ++d) cur.c[i][d] = d <= D ? (double)m[d] : 0.0;
            for (int q = 0; q <= 64; ++q) {
                const double eta = -1.0 + q / 32.0;
                double v = 0;
                for (int d = D; d >= 0; --d) v = v * eta + cur.c[i][d];
                const double ex = (double)es_exact((long double)eta / 2 + centre, w, beta);
                worst = std::max(worst, fabs(v - ex));
            }
        }
        cur.max_err = worst;
        if (worst > 0.5 * prev_err && best.deg) break;          // no longer improving: keep the previous degree
        best = cur;
        prev_err = worst;
        if (worst <= tol) break;
    }
    *kp = best;
}

// Autotuned grid size, used when the power-of-two grid would be much larger than needed (sigma > 1.6;
// measured at config 5: 3 x 2^28 C2C 10.1 ms, 3 x 1.6e8 6.3 ms).  cuFFT's time follows its pass structure
// rather than n, so the few smallest {2,3,5}-smooth sizes >= 1.25 Nf, 3*2^k and 5*2^k are TIMED (three
// transforms, scratch data) and the cheapest by  t_fft + own-kernel grid traffic  is taken.
int64_t autotune_grid_size(int64_t Nf, int dtype, int64_t n_pow2, int ntrans) {
    const cufftType type = dtype == LS_F64 ? CUFFT_Z2Z : CUFFT_C2C;
    const size_t cell = dtype == LS_F64 ? 16 : 8;
    std::vector<int64_t> cand;
    cand.push_back(n_pow2);
    const int64_t lo = (int64_t)ceil(1.25 * (double)Nf);
    int64_t m = lo;
    for (int i = 0; i < 5; ++i) {                      // the five smallest smooth sizes
        m = next_smooth_even(m);
        if (m >= n_pow2) break;
        cand.push_back(m);
        m += 4;
    }
    for (int64_t f : {3, 5}) {                         // few-pass sizes: 3 * 2^k, 5 * 2^k
        int64_t v = f * 4;
        while (v < lo) v *= 2;
        if (v < n_pow2 && std::find(cand.begin(), cand.end(), v) == cand.end()) cand.push_back(v);
    }
    if (cand.size() == 1) return n_pow2;
    void* buf = nullptr;
    // time with as many transforms as one execute pass has, capped so that the scratch stays <= 1 GB
    const int nb = (int)std::max<size_t>(3, std::min<size_t>((size_t)ntrans, ((size_t)1 << 30) / ((size_t)n_pow2 * cell)));
    if (cudaMalloc(&buf, (size_t)n_pow2 * cell * nb) != cudaSuccess) { cudaGetLastError(); return n_pow2; }
    cudaMemset(buf, 0, (size_t)n_pow2 * cell * nb);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    int64_t best = n_pow2;
    double best_cost = 1e300;
    for (int64_t n : cand) {
        cufftHandle h;
        if (cufftCreate(&h) != CUFFT_SUCCESS) continue;
        long long nn[1] = {(long long)n};
        size_t ws = 0;
        void* work = nullptr;
        bool ok = cufftSetAutoAllocation(h, 0) == CUFFT_SUCCESS &&
                  cufftMakePlanMany64(h, 1, nn, nullptr, 1, n, nullptr, 1, n, type, nb, &ws) == CUFFT_SUCCESS &&
                  cudaMalloc(&work, ws ? ws : 16) == cudaSuccess && cufftSetWorkArea(h, work) == CUFFT_SUCCESS;
        float ms = 0;
        if (ok) {
            for (int it = 0; it < 3 && ok; ++it) {      // two warm-ups, the third is timed
                if (it == 2) cudaEventRecord(e0, 0);
                ok = (dtype == LS_F64 ? cufftExecZ2Z(h, (cufftDoubleComplex*)buf, (cufftDoubleComplex*)buf, CUFFT_INVERSE)
                                      : cufftExecC2C(h, (cufftComplex*)buf, (cufftComplex*)buf, CUFFT_INVERSE)) == CUFFT_SUCCESS;
            }
            cudaEventRecord(e1, 0);
            ok = ok && cudaEventSynchronize(e1) == cudaSuccess && cudaEventElapsedTime(&ms, e0, e1) == cudaSuccess;
        }
        cufftDestroy(h);
        cudaFree(work);
        cudaGetLastError();
        if (!ok) continue;
        // own kernels: the grids are written once (spread, ~3.5 TB/s effective); the modes read do not depend on n
        const double cost = ms + (double)nb * (double)n * cell / 3.5e9;
        if (cost < best_cost) { best_cost = cost; best = n; }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    return best;
}

// Plan-owned device memory.  With the environment variable LS_B200_GUARD set when the plan is made, every allocation
// is wrapped in two 256-byte guard zones filled with 0xA5 that ls_debug_guards checks: an out-of-bounds WRITE of any
// kernel shows up as a damaged guard (compute-sanitizer is closed on this GPU pool, profiles/r2_checks.md).
constexpr size_t kGuardBytes = 256;
template <typename T>
cudaError_t dmalloc(ls_plan_s* p, T** ptr, size_t bytes) {
    if (bytes == 0) bytes = 16;
    const size_t g = p->guard ? kGuardBytes : 0;
    char* base = nullptr;
    cudaError_t e = cudaMalloc((void**)&base, bytes + 2 * g);
    if (e != cudaSuccess) return e;
    if (g) {
        if ((e = cudaMemset(base, 0xA5, g)) != cudaSuccess || (e = cudaMemset(base + g + bytes, 0xA5, g)) != cudaSuccess) return e;
        p->guards.push_back({base, bytes});
    }
    p->total_bytes += bytes;
    *ptr = (T*)(base + g);
    return cudaSuccess;
}
void dfree(ls_plan_s* p, void* ptr) {
    if (!ptr) return;
    if (p->guard) {
        for (auto& gz : p->guards)
            if (gz.first && gz.first + kGuardBytes == (char*)ptr) {
                cudaFree(gz.first);
                gz.first = nullptr;
                return;
            }
    }
    cudaFree(ptr);
}

void build_passes(const ls_plan_s* p, std::vector<Pass>& out) {
    out.clear();
    const bool per = p->opts.dy_per_series != 0;
    for (int s0 = 0; s0 < p->batch; s0 += p->chunk) {
        Pass ps;
        ps.s0 = s0;
        ps.C = std::min(p->chunk, p->batch - s0);
        // fixed mean (opts.no_floating_mean): the w transform at x1 is not needed — the paper's "pair of NUFFTs"
        // (PAPER.md:17): w at x2 and h at x1 only
        const int nw = p->opts.no_floating_mean ? 0 : 1;
        if (per) { ps.fft_slot0 = 0; ps.fft_batch = (2 + nw) * ps.C; }
        else if (s0 == 0) { ps.fft_slot0 = 0; ps.fft_batch = 1 + nw + ps.C; }
        else { ps.fft_slot0 = 1 + nw; ps.fft_batch = ps.C; }
        out.push_back(ps);
    }
}

struct FftPlans {
    int batch[3];
    cufftHandle h[3];
    int count;
};

cufftHandle find_fft(const ls_plan_s* p, int batch) {
    if (p->has_first && p->first_batch == batch) return p->fft_first;
    if (p->has_rem && p->rem_batch == batch) return p->fft_rem;
    return p->fft_chunk;
}

int make_fft(ls_plan_s* p, cufftHandle* h, int batch, size_t* work) {
    if (cufftCreate(h) != CUFFT_SUCCESS) return LS_ERR_CUFFT;
    if (cufftSetAutoAllocation(*h, 0) != CUFFT_SUCCESS) return LS_ERR_CUFFT;
    long long nn[1] = {(long long)p->n};
    size_t ws = 0;
    const cufftType type = p->dtype == LS_F64 ? CUFFT_Z2Z : CUFFT_C2C;
    if (cufftMakePlanMany64(*h, 1, nn, nullptr, 1, p->n, nullptr, 1, p->n, type, batch, &ws) != CUFFT_SUCCESS)
        return LS_ERR_CUFFT;
    *work = std::max(*work, ws);
    return LS_OK;
}

void stage_begin(ls_plan_s* p, int stage, cudaStream_t s) {
    if (!p->opts.timing) return;
    if (p->events_used == p->events.size()) {
        lsb::StageEvent ev;
        ev.stage = stage;
        cudaEventCreate(&ev.beg);
        cudaEventCreate(&ev.end);
        p->events.push_back(ev);
    }
    p->events[p->events_used].stage = stage;
    cudaEventRecord(p->events[p->events_used].beg, s);
}
void stage_end(ls_plan_s* p, cudaStream_t s) {
    if (!p->opts.timing) return;
    cudaEventRecord(p->events[p->events_used].end, s);
    ++p->events_used;
}

}  // namespace

extern "C" {

const char* ls_strerror(int code) {
    switch (code) {
        case LS_OK: return "success";
        case LS_ERR_INVALID_VALUE: return "invalid argument";
        case LS_ERR_ALLOC: return "allocation failed";
        case LS_ERR_CUDA: return "CUDA error or no usable device";
        case LS_ERR_CUFFT: return "cuFFT error";
        case LS_ERR_UNSUPPORTED: return "problem size not supported";
        case LS_ERR_NOT_READY: return "requested information is not available yet";
        case LS_ERR_TOO_LARGE: return "size beyond the fixed scratch of a no-allocation entry point (Nd > LS_NOALLOC_MAX_ND)";
        default: return "unknown error code";
    }
}

int ls_destroy(ls_plan_t p) {
    if (!p) return LS_OK;
    if (p->gexec) cudaGraphExecDestroy(p->gexec);
    if (p->has_first) cufftDestroy(p->fft_first);
    if (p->has_chunk) cufftDestroy(p->fft_chunk);
    if (p->has_rem) cufftDestroy(p->fft_rem);
    if (!p->external_ws) {
        dfree(p, p->fft_work);
        dfree(p, p->grids);
        dfree(p, p->modes);
    }
    dfree(p, p->dinv);
    dfree(p, p->t64);
    dfree(p, p->fft_wlo);
    dfree(p, p->fft_whi);
    dfree(p, p->ftab);
    dfree(p, p->tile_list);
    dfree(p, p->zeroed);                     // sums and both histograms live in this allocation
    dfree(p, p->scan_tmp);
    for (int i = 0; i < 2; ++i) {
        dfree(p, p->ps[i].bin_start);
        dfree(p, p->ps[i].perm);
        dfree(p, p->ps[i].rec);
        dfree(p, p->ps[i].rows);
    }
    dfree(p, p->st_t);
    dfree(p, p->st_y);
    dfree(p, p->st_dy);
    dfree(p, p->st_p);
    if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
    if (p->copy_ev) cudaEventDestroy(p->copy_ev);
    for (auto& ev : p->events) {
        cudaEventDestroy(ev.beg);
        cudaEventDestroy(ev.end);
    }
    delete p;
    return LS_OK;
}

int ls_plan(ls_plan_t* out, int64_t Nd, int64_t Nf, double f0, double df, double eps, int dtype, int batch,
            const ls_opts* opts) {
    if (!out) return LS_ERR_INVALID_VALUE;
    *out = nullptr;
    if (Nd < 1 || Nf < 1 || batch < 1 || batch > 65535) return LS_ERR_INVALID_VALUE;
    if (!(df > 0.0) || !isfinite(df) || !(f0 >= 0.0) || !isfinite(f0)) return LS_ERR_INVALID_VALUE;
    if (dtype != LS_F32 && dtype != LS_F64) return LS_ERR_INVALID_VALUE;
    const double eps_lo = dtype == LS_F64 ? 1e-14 : 1e-6;
    if (!(eps >= eps_lo) || !(eps <= 1e-1)) return LS_ERR_INVALID_VALUE;
    if (Nd >= (int64_t)1 << 31) return LS_ERR_UNSUPPORTED;
    ls_opts o;
    memset(&o, 0, sizeof o);
    if (opts) o = *opts;
    if (o.upsampfac != 0.0 && !(o.upsampfac >= 1.2 && o.upsampfac <= 4.0)) return LS_ERR_INVALID_VALUE;
    if (o.kernel_width != 0 && (o.kernel_width < 2 || o.kernel_width > lsb::kMaxWidth)) return LS_ERR_INVALID_VALUE;
    // spreading tiles: one, two or four cells per thread of a 256-thread CTA (the instantiated kernels); a batch
    // accumulates four transforms per CTA and has registers for two cells per thread
    if (o.tile_cells != 0 && o.tile_cells != 256 && o.tile_cells != 512 && o.tile_cells != 1024) return LS_ERR_INVALID_VALUE;
    if (o.tile_cells == 1024 && batch > 1) return LS_ERR_INVALID_VALUE;
    if (o.t_is_dtype < 0 || o.t_is_dtype > 1) return LS_ERR_INVALID_VALUE;
    if (o.reserved[0] < 0 || o.reserved[0] > 2 || o.reserved[1] < 0 || o.reserved[1] > 8) return LS_ERR_INVALID_VALUE;
    if (o.batch_chunk < 0 || o.graph < 0 || o.graph > 2 || o.fft_impl < 0 || o.fft_impl > 3 ||
        o.no_floating_mean < 0 || o.no_floating_mean > 1 || o.normalization < 0 || o.normalization > 3)
        return LS_ERR_INVALID_VALUE;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1 || o.device < 0 || o.device >= ndev) return LS_ERR_CUDA;
    if (cudaSetDevice(o.device) != cudaSuccess) return LS_ERR_CUDA;

    ls_plan_s* p = new (std::nothrow) ls_plan_s;
    if (!p) return LS_ERR_ALLOC;
    p->Nd = Nd; p->Nf = Nf; p->f0 = f0; p->df = df; p->eps = eps; p->dtype = dtype; p->batch = batch;
    p->guard = getenv("LS_B200_GUARD") != nullptr;
    p->opts = o;
    if (cudaDeviceGetAttribute(&p->num_sms, cudaDevAttrMultiProcessorCount, o.device) != cudaSuccess || p->num_sms < 1) {
        cudaGetLastError();
        p->num_sms = 148;
    }

    // ---- (sigma, w, beta, n) from eps: reading A10.  Auto: the fine grid is the power of two in
    // [1.25 Nf, 2.5 Nf) (the FFT pass count, not the cell count, decides its time), the
    // width follows from the realised sigma = n/Nf, plus two (fp64) / one (fp32) cells of safety so
    // that a pointwise reading of the tolerance also holds (A8, A9).
    bool auto5 = false;                                 // the plan chose a 5 x 2^k grid for the own fused transform
    if (o.upsampfac != 0.0) {
        const double want = ceil(o.upsampfac * (double)Nf);
        if (want >= 2147483000.0) { delete p; return LS_ERR_UNSUPPORTED; }
        p->n = next_smooth_even(std::max<int64_t>((int64_t)want, 2 * lsb::kMaxWidth));
    } else {
        const double want = ceil(1.25 * (double)Nf);
        if (want >= 2147483000.0) { delete p; return LS_ERR_UNSUPPORTED; }
        int64_t m = 64;                                 // >= 2 kMaxWidth
        while ((double)m < want) m *= 2;
        p->n = m;
        const int ntrans = (o.dy_per_series ? 3 * batch : batch + 2) - (o.no_floating_mean ? (o.dy_per_series ? batch : 1) : 0);
        // A batch of small fp64 grids with shared dy: where 5 x 2^k (k = 13 .. 16) lies between 1.25 Nf and the power of two,
        // the own two-pass transform on it with the assembly fused into the last pass moves the fewest bytes (config 4:
        // 163 840 cells instead of 2^18, or of cuFFT on 160 000: 3.17 -> 2.72 ms per 1000 series).
        int64_t n5 = 0;
        for (int k = 13; k <= 16; ++k)
            if ((double)(5LL << k) >= want && (5LL << k) < m) n5 = n5 ? n5 : (5LL << k);
        if (n5 && dtype == LS_F64 && !o.dy_per_series && o.fft_impl != 1 && !o.no_autotune && (double)n5 * ntrans * 16.0 > 64e6) {
            p->n = n5;
            auto5 = true;
        } else if (dtype == LS_F32 && o.fft_impl != 1 && !o.no_autotune && ntrans <= 8 && [&] {
                       // fp32, a few very long transforms (config 5): 5 x 2^k cells, k = 22 .. 25, where that lies between
                       // 1.25 Nf and the power of two: the own three-pass transform (ls_fft_f32.cu) instead of cuFFT on a
                       // 2,3,5-smooth size, and no zero fill of the empty tiles
                       for (int k = 22; k <= 25; ++k)
                           if ((double)(5LL << k) >= want && (5LL << k) < m) { p->n = 5LL << k; return true; }
                       return false;
                   }()) {
            auto5 = true;
        } else
        if ((double)m > 1.6 * (double)Nf && (double)m * ntrans >= (double)((int64_t)1 << 20) && !o.no_autotune) {
            // the timed choice is cached per (Nf, dtype, transforms, device): the same arguments give the same grid — and
            // therefore the same results — for the life of the process (between processes it may differ: ls.h)
            static std::mutex mu;
            static std::map<std::tuple<int64_t, int, int, int>, int64_t> cache;
            std::lock_guard<std::mutex> lock(mu);
            const auto key = std::make_tuple(Nf, dtype, ntrans, o.device);
            auto it = cache.find(key);
            if (it == cache.end()) it = cache.emplace(key, autotune_grid_size(Nf, dtype, m, ntrans)).first;
            p->n = it->second;
        }
    }
    if (p->n >= ((int64_t)1 << 31) - 4096) { delete p; return LS_ERR_UNSUPPORTED; }
    p->sigma = (double)p->n / (double)Nf;
    int w = o.kernel_width;
    if (w == 0) {
        const double s = std::min(p->sigma, 2.0);      // tiny Nf: n is floored at 64 cells
        // Measured (single point, sup norm over its position): the ES kernel's error is
        // ~ 30 exp(-w rate) for sigma in [1.25, 2].  fp64: aim a decade below eps so that a pointwise
        // reading of the tolerance holds too (A8) — 12 cells at sigma = 2, 17 at 1.34, 19 at 1.25, for
        // eps = 1e-9.  fp32: the grid's own rounding (6e-8) dominates early; the plain rule plus one cell.
        auto width_for = [&](double sg) {
            const double rt = M_PI * sqrt(1.0 - 1.0 / std::min(sg, 2.0));
            return dtype == LS_F64 ? (int)ceil((-log(eps) + log(300.0)) / rt - 1e-9) : (int)ceil(-log(eps) / rt - 1e-9) + 1;
        };
        w = width_for(s);
        // The kernels hold at most kMaxWidth cells.  Where the tolerance asks for more at this sigma, the automatic grid
        // doubles (sigma >= 2 needs <= 17 cells down to eps = 1e-14); with a grid size the caller fixed, the plan is refused
        // rather than silently missing the tolerance.
        while (w > lsb::kMaxWidth && o.upsampfac == 0.0 && p->n < ((int64_t)1 << 30)) {
            p->n *= 2;
            p->sigma = (double)p->n / (double)Nf;
            w = width_for(p->sigma);
        }
        if (w > lsb::kMaxWidth) { delete p; return LS_ERR_UNSUPPORTED; }
        w = std::max(2, w);
    }
    p->w = w;
    p->beta = 0.97 * M_PI * w * (1.0 - 1.0 / (2.0 * std::min(p->sigma, 2.0)));
    fit_kernel_poly(w, p->beta, 1e-3 * eps, dtype == LS_F64 ? 12 : 8, &p->poly);
    p->L = o.tile_cells ? o.tile_cells : 1024;
    if (batch > 1) p->L = std::min(p->L, 512);      // four transforms per CTA: two cells per thread
    p->nbins = (int)((p->n + lsb::kBinCells - 1) / lsb::kBinCells);
    p->ntiles = (int)((p->n + p->L - 1) / p->L);
    {
        auto gcd = [](long long a, long long b) { while (b) { const long long r = a % b; a = b; b = r; } return a; };
        long long st = std::max<long long>(1, (long long)(0.6180339887 * p->ntiles));
        while (gcd(st, p->ntiles) != 1) ++st;
        p->tile_stride = (int)(st % p->ntiles == 0 ? 1 : st % p->ntiles);
    }
    const bool per = o.dy_per_series != 0;
    const int nw = o.no_floating_mean ? 0 : 1;     // the w transform at x1 exists only with the floating mean
    p->M = per ? (2 + nw) * batch : batch + 1 + nw;
    const size_t B = real_bytes(dtype);
    const size_t grid_bytes = (size_t)p->n * 2 * B;
    if (o.batch_chunk > 0) p->chunk = std::min(o.batch_chunk, batch);
    else {
        // Measured (config 4, B200): keeping a chunk's grids L2-sized does not pay — cuFFT and the own
        // kernels stream at HBM rate either way and small passes are launch/tail-bound (8.2 ms per 1000
        // series with 64 MB chunks, 5.3 ms in one pass).  So: as many series per pass as 8 GB of grids hold.
        p->chunk = (int)std::max<size_t>(1, std::min<size_t>((size_t)batch, ((size_t)8 << 30) / grid_bytes));
    }
    p->slots = per ? (2 + nw) * p->chunk : 1 + nw + p->chunk;

    // own FFT: wherever it exists when asked for (fft_impl 2, 3); in auto mode for the pruned sizes (n >= 2^20) and, below
    // them, for problems small enough to be latency-bound (cuFFT runs a 2^14-point fp64 transform in ONE CTA: 29 us of
    // config 1's 58), but not for large batches of small grids, where cuFFT's pass structure moves fewer bytes
    p->own_fft = o.fft_impl != 1 && lsb::own_fft_supported(p);
    if (p->own_fft && o.fft_impl == 0 && !auto5 && !lsb::own_fft_prunes(p) && (double)p->M * (double)p->n * 16.0 > 64e6) p->own_fft = false;
    p->fft_prune = p->own_fft && lsb::own_fft_prunes(p);
    // cuFFT path, few transforms over very many tiles (config 5: 3 x 154 000): one sweep kernel zero-fills the empty tiles
    // and lists the occupied ones for a persistent spreading launch.  Measured: config 5 spread 1.51 -> 1.34 ms; config 4
    // (1002 transforms over 313 tiles) 0.54 -> 0.78 ms, so batches keep one CTA per (tile, row group).
    // (reserved[0] = 1: never)
    p->list_tiles = !p->own_fft && o.reserved[0] != 1 && ((p->M <= 8 && p->ntiles >= 32 * p->num_sms) || o.reserved[0] == 2);   // 2: always (tests)
    if (o.fft_impl >= 2 && !p->own_fft) { delete p; return LS_ERR_UNSUPPORTED; }
    // Measured at config 3 (profiles/r1e_cfg3.md): with the cheaper assembly arithmetic the separate
    // assembly kernel (0.118 ms at 81 % of DRAM peak) plus an unfused third pass beats the fused kernel, which is
    // bound by its 2-CTAs-per-SM arithmetic, by 1 % — so fusion is opt-in (fft_impl = 2), not the default.
    // ... except for batches on the 5 x 2^k grids: there the modes round trip (2 x 16 bytes per frequency and series) is the
    // largest item left and the fused pass reads its per-frequency terms from a table (config 4: 2.88 -> 2.45 ms)
    p->fuse_assemble = p->own_fft && dtype == LS_F64 && (o.fft_impl == 2 || (o.fft_impl == 0 && lsb::own_fft_rm5(p) && batch >= 8)) && !o.dy_per_series;
    // Passes 2 and 3 as one persistent kernel with the intermediate kept in L2 (ls_fft.cu): the default wherever
    // the pruned three-pass transform runs; fft_impl = 3 keeps the three separate launches (for comparison).
    p->fuse_pass23 = p->fft_prune && dtype == LS_F64 && !lsb::own_fft_rm5(p) && !p->fuse_assemble && o.fft_impl != 3;

    // double-double constants (host): n*df exactly, f_c = f0 + floor(Nf/2) df
    p->ndf = two_prod((double)p->n, df);
    p->fc = dd_add_d(two_prod((double)(Nf / 2), df), f0);

    p->model_bytes = 8.0 * Nd + (double)batch * Nd * B + (per ? (double)batch : 1.0) * Nd * B + 8.0 * Nd +
                     (double)p->M * p->n * 2 * B + (double)p->M * Nf * 2 * B + (double)batch * Nf * B;

    p->use_graph = !o.timing && o.graph != 1;

    int rc = LS_OK;
    cudaError_t ce = cudaSuccess;
    do {
        p->grids_bytes = (size_t)p->slots * grid_bytes;
        if ((ce = dmalloc(p, &p->grids, p->grids_bytes)) != cudaSuccess) break;
        if ((ce = dmalloc(p, &p->dinv, (size_t)(Nf / 2 + 1) * 8)) != cudaSuccess) break;
        if (o.t_is_dtype && dtype == LS_F32 && (ce = dmalloc(p, &p->t64, (size_t)Nd * 8)) != cudaSuccess) break;
        if (p->own_fft) {
            if ((ce = dmalloc(p, (char**)&p->fft_wlo, (size_t)4096 * 16)) != cudaSuccess) break;
            if ((ce = dmalloc(p, (char**)&p->fft_whi, (size_t)std::max<int64_t>(4096, p->n / 4096) * 16)) != cudaSuccess) break;
            p->modes_bytes = (size_t)p->slots * Nf * 2 * B;
            if ((ce = dmalloc(p, (char**)&p->modes, p->modes_bytes)) != cudaSuccess) break;
            if (p->fuse_assemble && (ce = dmalloc(p, (char**)&p->ftab, (size_t)Nf * 32)) != cudaSuccess) break;
            if ((ce = lsb::own_fft_init(p, 0)) != cudaSuccess) break;
        }
        // sums and both histograms live in ONE allocation so a single memset clears them per execute
        const size_t sums_bytes = ((size_t)batch * 4 * 8 + 255) & ~(size_t)255;
        const size_t hist_bytes = ((size_t)2 * p->nbins * 4 + 255) & ~(size_t)255;
        const size_t mask_bytes = p->fft_prune ? (size_t)2 * std::max(65536 / p->L, lsb::own_fft_ncoltiles(p)) * std::max(16, lsb::own_fft_rb(p)) * 4 + 256 : (p->list_tiles ? 256 : 0);   // masks + 2 list counters
        const size_t queue_bytes = p->fuse_pass23 ? (((size_t)(2 + 32 * p->slots) * 4 + 255) & ~(size_t)255) : 0;
        p->zeroed_bytes = sums_bytes + hist_bytes + mask_bytes + queue_bytes;
        if ((ce = dmalloc(p, (char**)&p->zeroed, p->zeroed_bytes)) != cudaSuccess) break;
        if (queue_bytes) p->fft_queue = (int*)((char*)p->zeroed + sums_bytes + hist_bytes + mask_bytes);
        if (p->fft_prune || p->list_tiles) {
            p->tile_counts = (int*)((char*)p->zeroed + sums_bytes + hist_bytes);
            if (p->fft_prune) p->row_masks = (unsigned*)((char*)p->zeroed + sums_bytes + hist_bytes + 256);
            if ((ce = dmalloc(p, &p->tile_list, (size_t)2 * p->ntiles * 4)) != cudaSuccess) break;
        }
        p->sums = (double*)p->zeroed;
        p->ps[0].hist = (int*)((char*)p->zeroed + sums_bytes);
        p->ps[1].hist = p->ps[0].hist + p->nbins;
        const int nchunks = (p->nbins + 4095) / 4096;
        if ((ce = dmalloc(p, &p->scan_tmp, (size_t)2 * (nchunks + 1) * 4)) != cudaSuccess) break;
        if ((ce = cudaMemset(p->scan_tmp, 0, (size_t)2 * (nchunks + 1) * 4)) != cudaSuccess) break;
        for (int i = 0; i < 2 && ce == cudaSuccess; ++i) {
            lsb::PointSet& ps = p->ps[i];
            // stored strength rows (shared dy: the weights live in the records, only y - ybar is stored)
            ps.nrows = i == 0 ? (per ? (1 + nw) * batch : batch) : (per ? batch : 0);
            if ((ce = dmalloc(p, &ps.bin_start, (size_t)(p->nbins + 1) * 4)) != cudaSuccess) break;
            if ((batch > 1 || per) && (ce = dmalloc(p, &ps.perm, (size_t)Nd * 4)) != cudaSuccess) break;
            if ((ce = dmalloc(p, (char**)&ps.rec, (size_t)Nd * 4 * B)) != cudaSuccess) break;
            if ((ce = dmalloc(p, (char**)&ps.rows, (size_t)ps.nrows * Nd * B)) != cudaSuccess) break;
        }
        if (ce != cudaSuccess) break;

        // cuFFT plans for every distinct batch size the pass list needs, one shared work area
        std::vector<Pass> passes;
        build_passes(p, passes);
        size_t work = 0;
        if (!p->own_fft) {
        p->first_batch = passes.front().fft_batch;
        if ((rc = make_fft(p, &p->fft_first, p->first_batch, &work)) != LS_OK) break;
        p->has_first = true;
        if (passes.size() > 1) {
            const int cb = passes[1].fft_batch;
            if (cb != p->first_batch) {
                if ((rc = make_fft(p, &p->fft_chunk, cb, &work)) != LS_OK) break;
                p->has_chunk = true;
            } else p->fft_chunk = p->fft_first;
            const int rb = passes.back().fft_batch;
            if (rb != cb && rb != p->first_batch) {
                p->rem_batch = rb;
                if ((rc = make_fft(p, &p->fft_rem, rb, &work)) != LS_OK) break;
                p->has_rem = true;
            }
        } else p->fft_chunk = p->fft_first;
        p->fft_work_bytes = work;
        if ((ce = dmalloc(p, (char**)&p->fft_work, work)) != cudaSuccess) break;
        if (cufftSetWorkArea(p->fft_first, p->fft_work) != CUFFT_SUCCESS) { rc = LS_ERR_CUFFT; break; }
        if (p->has_chunk && cufftSetWorkArea(p->fft_chunk, p->fft_work) != CUFFT_SUCCESS) { rc = LS_ERR_CUFFT; break; }
        if (p->has_rem && cufftSetWorkArea(p->fft_rem, p->fft_work) != CUFFT_SUCCESS) { rc = LS_ERR_CUFFT; break; }
        }
        if (rc != LS_OK) break;

        // P0: deconvolution table on the device
        double hz[lsb::kQuadNodes], hw[lsb::kQuadNodes];
        gauss_legendre_01(lsb::kQuadNodes, hz, hw);
        double* dq = nullptr;
        if ((ce = cudaMalloc((void**)&dq, sizeof(double) * 2 * lsb::kQuadNodes)) != cudaSuccess) break;
        ce = cudaMemcpy(dq, hz, sizeof hz, cudaMemcpyHostToDevice);
        if (ce == cudaSuccess) ce = cudaMemcpy(dq + lsb::kQuadNodes, hw, sizeof hw, cudaMemcpyHostToDevice);
        if (ce == cudaSuccess) ce = lsb::launch_deconv_table(p, dq, dq + lsb::kQuadNodes, 0);
        if (ce == cudaSuccess) ce = cudaDeviceSynchronize();
        cudaFree(dq);
    } while (0);
    if (ce != cudaSuccess) rc = (ce == cudaErrorMemoryAllocation) ? LS_ERR_ALLOC : LS_ERR_CUDA;
    if (rc != LS_OK) {
        cudaGetLastError();
        ls_destroy(p);
        return rc;
    }
    *out = p;
    return LS_OK;
}

// Enqueue the whole stage sequence on stream s (directly, or into a stream capture).
//
// host_power != nullptr (ls_execute_host, direct launches only): every finished piece of `power` — a pass's series, or
// with a single pass a quarter of the frequencies — is copied to the host on p->copy_stream while the kernels of the
// next piece run; the caller joins copy_stream.
static int enqueue_execute(ls_plan_t p, const void* t, const void* y, const void* dy, void* power, cudaStream_t s,
                           char* host_power = nullptr) {
    const bool per = p->opts.dy_per_series != 0;
    int own = 0, ffts = 0;
    cudaError_t ce = cudaSuccess;
    p->events_used = 0;
#define LS_TRY(call)                 \
    do {                             \
        ce = (call);                 \
        if (ce != cudaSuccess) {     \
            cudaGetLastError();      \
            return LS_ERR_CUDA;      \
        }                            \
    } while (0)

    stage_begin(p, LS_STAGE_TOTAL, s);
    const size_t total_slot = p->events_used;   // the TOTAL event pair is closed at the very end
    if (p->opts.timing) ++p->events_used;

    stage_begin(p, LS_STAGE_STATS, s);              // K1 + the bin histogram of K3 (one kernel)
    if (p->t64) {                                   // float times: promoted once, read as double from here on
        LS_TRY(lsb::launch_promote_t(p, t, s)); ++own;
        t = p->t64;
    }
    LS_TRY(cudaMemsetAsync(p->zeroed, 0, p->zeroed_bytes, s));
    LS_TRY(lsb::launch_stats_count(p, (const double*)t, y, dy, s)); ++own;
    stage_end(p, s);

    stage_begin(p, LS_STAGE_SORT, s);
    LS_TRY(lsb::launch_bin_scan(p, s)); own += p->nbins > 4096 ? 2 : 1;
    if (p->fft_prune) { LS_TRY(lsb::launch_tile_list(p, s)); ++own; }
    stage_end(p, s);

    stage_begin(p, LS_STAGE_PREMUL, s);
    LS_TRY(lsb::launch_premultiply(p, (const double*)t, y, dy, s)); ++own;
    if (p->batch > 1 || per) { LS_TRY(lsb::launch_rows(p, y, dy, s)); ++own; }
    stage_end(p, s);

    {
        std::vector<Pass> passes;
        build_passes(p, passes);
        for (const Pass& ps : passes) {
            int h_slot, h_stride, w_slot, w_stride, w2_slot, w2_stride;
            stage_begin(p, LS_STAGE_SPREAD, s);
            const int nw = p->opts.no_floating_mean ? 0 : 1;
            if (p->list_tiles) {                            // cuFFT path: zeros into the empty tiles, occupied tiles listed
                if (per) LS_TRY(lsb::launch_zero_list(p, ps.C, 0, (1 + nw) * ps.C, ps.C, ps.s0 == 0, s));
                else if (ps.s0 == 0) LS_TRY(lsb::launch_zero_list(p, 1, 0, nw + ps.C, 1, 1, s));
                else LS_TRY(lsb::launch_zero_list(p, 0, 0, ps.C, 1 + nw, 0, s));
                ++own;
            }
            if (per) {
                // slots [0, C): w2_s ; slots [C, 3C): (w_s, h_s) pairs — fixed mean: [C, 2C): h_s (the rows kernel then
                // stores the h rows only)
                LS_TRY(lsb::launch_spread(p, ps.s0, ps.C, 0, (1 + nw) * ps.s0, (1 + nw) * ps.C, ps.C, s)); ++own;
                w2_slot = 0; w2_stride = 1; h_slot = ps.C + nw; h_stride = 1 + nw;
                w_slot = nw ? ps.C : 0; w_stride = nw ? 2 : 1;                 // fixed mean: unused (x 0): any finite modes
            } else {
                // slot 0: w2, slot 1: w, slots 2..: h_s of this pass — fixed mean: slot 0: w2, slots 1..: h_s (logical row 0
                // of the x1 point set, the w transform, is skipped)
                if (ps.s0 == 0) LS_TRY(lsb::launch_spread(p, 0, 1, 0, 1 - nw, nw + ps.C, 1, s));
                else LS_TRY(lsb::launch_spread(p, 0, 0, 0, 1 + ps.s0, ps.C, 1 + nw, s));
                ++own;
                w2_slot = 0; w2_stride = 0; w_slot = nw; w_stride = 0; h_slot = 1 + nw; h_stride = 1;
            }
            stage_end(p, s);
            if (p->debug_stop_after_spread) break;      // ls_debug_grid: the fine grids as the spreading kernel left them

            if (p->own_fft) {
                // own three-pass FFT: pass 1 skips the tiles spreading left unwritten; pass 3 emits compact modes
                // (fused mode: only of w2, w — the h transforms' pass 3 is part of the assembly kernel below)
                const int n_x2 = per ? ps.C : (ps.s0 == 0 ? 1 : 0);
                const int n_modes = !p->fuse_assemble ? ps.fft_batch : (ps.s0 == 0 ? 1 + nw : 0);
                stage_begin(p, LS_STAGE_FFT_PASS1, s);
                LS_TRY(lsb::launch_own_fft_pass1(p, ps.fft_slot0, ps.fft_batch, n_x2, s));
                stage_end(p, s);
                if (p->fuse_pass23) {
                    // passes 2 + 3 in one persistent kernel, intermediate in L2 (its time is reported as pass 2)
                    stage_begin(p, LS_STAGE_FFT_PASS2, s);
                    LS_TRY(lsb::launch_own_fft_pass23(p, ps.fft_slot0, ps.fft_batch, s));
                    stage_end(p, s);
                    own += 2;
                } else {
                stage_begin(p, LS_STAGE_FFT_PASS2, s);
                LS_TRY(lsb::launch_own_fft_pass2(p, ps.fft_slot0, ps.fft_batch, s));
                stage_end(p, s);
                stage_begin(p, LS_STAGE_FFT_PASS3, s);
                LS_TRY(lsb::launch_own_fft_pass3(p, ps.fft_slot0, n_modes, s));
                stage_end(p, s);
                own += 1 + ((p->n > 65536 && !lsb::own_fft_rm5(p)) ? 1 : 0) + (n_modes > 0 ? 1 : 0);
                }
            } else {
                stage_begin(p, LS_STAGE_FFT, s);
                cufftHandle h = find_fft(p, ps.fft_batch);
                if (cufftSetStream(h, s) != CUFFT_SUCCESS) return LS_ERR_CUFFT;
                char* base = (char*)p->grids + (size_t)ps.fft_slot0 * p->n * 2 * real_bytes(p->dtype);
                // B_k = sum_l b_l e^{+2 pi i k l / n}  (reading A7)  ==  cuFFT's unnormalised inverse
                cufftResult fr = p->dtype == LS_F64
                                     ? cufftExecZ2Z(h, (cufftDoubleComplex*)base, (cufftDoubleComplex*)base, CUFFT_INVERSE)
                                     : cufftExecC2C(h, (cufftComplex*)base, (cufftComplex*)base, CUFFT_INVERSE);
                if (fr != CUFFT_SUCCESS) return LS_ERR_CUFFT;
                ++ffts;
                stage_end(p, s);
            }

            stage_begin(p, LS_STAGE_ASSEMBLE, s);
            const size_t RB = real_bytes(p->dtype);
            auto copy_out = [&](size_t off, size_t bytes) -> cudaError_t {      // power[off, off + bytes) is final on s
                cudaError_t e = cudaEventRecord(p->copy_ev, s);
                if (e == cudaSuccess) e = cudaStreamWaitEvent(p->copy_stream, p->copy_ev, 0);
                if (e == cudaSuccess) e = cudaMemcpyAsync(host_power + off, (const char*)power + off, bytes, cudaMemcpyDeviceToHost, p->copy_stream);
                return e;
            };
            if (p->fuse_assemble) {
                LS_TRY(lsb::launch_own_fft_assemble(p, h_slot, ps.C, ps.s0, w_slot, w2_slot, power, s));
                if (host_power) LS_TRY(copy_out((size_t)ps.s0 * p->Nf * RB, (size_t)ps.C * p->Nf * RB));
            } else if (host_power && passes.size() == 1 && p->batch == 1 && p->Nf >= (1 << 22)) {
                constexpr int kPieces = 4;                                       // one long series: frequency quarters
                const long long step = ((p->Nf + kPieces - 1) / kPieces + 255) & ~255LL;
                for (long long k0 = 0; k0 < p->Nf; k0 += step) {
                    const long long k1 = std::min<long long>(p->Nf, k0 + step);
                    LS_TRY(lsb::launch_assemble(p, ps.s0, ps.C, h_slot, h_stride, w_slot, w_stride, w2_slot, w2_stride, power, s, k0, k1));
                    LS_TRY(copy_out((size_t)k0 * RB, (size_t)(k1 - k0) * RB));
                    if (k0) ++own;
                }
            } else {
                LS_TRY(lsb::launch_assemble(p, ps.s0, ps.C, h_slot, h_stride, w_slot, w_stride, w2_slot, w2_stride, power, s));
                if (host_power) LS_TRY(copy_out((size_t)ps.s0 * p->Nf * RB, (size_t)ps.C * p->Nf * RB));
            }
            ++own;
            stage_end(p, s);
        }
    }
    if (p->opts.timing) {
        cudaEventRecord(p->events[total_slot].end, s);
        p->timed_once = true;
    }
    p->own_kernels = own;
    p->fft_execs = ffts;
    return LS_OK;
#undef LS_TRY
}

int ls_execute(ls_plan_t p, const void* t, const void* y, const void* dy, void* power, void* cuda_stream) {
    if (!p || !t || !y || !dy || !power) return LS_ERR_INVALID_VALUE;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    // Small problems are launch-latency-bound ("GPU overheads"): replay the sequence as one graph.
    // A legacy default stream cannot be captured; any capture failure falls back to direct launches for good.
    if (!p->use_graph || s == nullptr) return enqueue_execute(p, t, y, dy, power, s);
    if (!p->gexec || p->g_t != t || p->g_y != y || p->g_dy != dy || p->g_power != power) {
        // auto mode: a caller that changes buffers on every call gains nothing from replay — stop capturing
        if (p->gexec && p->opts.graph == 0 && ++p->g_misses >= 3) {
            cudaGraphExecDestroy(p->gexec);
            p->gexec = nullptr;
            p->use_graph = false;
            return enqueue_execute(p, t, y, dy, power, s);
        }
        if (p->gexec) { cudaGraphExecDestroy(p->gexec); p->gexec = nullptr; }
        cudaGraph_t graph = nullptr;
        int rc = LS_ERR_CUDA;
        if (cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            rc = enqueue_execute(p, t, y, dy, power, s);
            if (cudaStreamEndCapture(s, &graph) != cudaSuccess || !graph) rc = LS_ERR_CUDA;
            if (rc == LS_OK && cudaGraphInstantiate(&p->gexec, graph, 0) != cudaSuccess) rc = LS_ERR_CUDA;
            if (graph) cudaGraphDestroy(graph);
        }
        if (rc != LS_OK) {
            cudaGetLastError();
            p->gexec = nullptr;
            p->use_graph = false;
            return enqueue_execute(p, t, y, dy, power, s);
        }
        p->g_t = t; p->g_y = y; p->g_dy = dy; p->g_power = power;
    }
    else p->g_misses = 0;
    if (cudaGraphLaunch(p->gexec, s) != cudaSuccess) { cudaGetLastError(); return LS_ERR_CUDA; }
    return LS_OK;
}

int ls_execute_host(ls_plan_t p, const void* t, const void* y, const void* dy, void* power, void* cuda_stream) {
    if (!p || !t || !y || !dy || !power) return LS_ERR_INVALID_VALUE;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t B = real_bytes(p->dtype);
    const size_t bt = (size_t)p->Nd * (p->t64 ? 4 : 8), by = (size_t)p->batch * p->Nd * B;
    const size_t bdy = (size_t)(p->opts.dy_per_series ? p->batch : 1) * p->Nd * B;
    const size_t bp = (size_t)p->batch * p->Nf * B;
    if (!p->st_p) {                                   // staging buffers, made on first use; st_p is the last one made
        if ((!p->st_t && dmalloc(p, (char**)&p->st_t, bt) != cudaSuccess) ||
            (!p->st_y && dmalloc(p, (char**)&p->st_y, by) != cudaSuccess) ||
            (!p->st_dy && dmalloc(p, (char**)&p->st_dy, bdy) != cudaSuccess) ||
            dmalloc(p, (char**)&p->st_p, bp) != cudaSuccess) {
            cudaGetLastError();
            return LS_ERR_ALLOC;
        }
    }
    if (cudaMemcpyAsync(p->st_t, t, bt, cudaMemcpyHostToDevice, s) != cudaSuccess ||
        cudaMemcpyAsync(p->st_y, y, by, cudaMemcpyHostToDevice, s) != cudaSuccess ||
        cudaMemcpyAsync(p->st_dy, dy, bdy, cudaMemcpyHostToDevice, s) != cudaSuccess) {
        cudaGetLastError();
        return LS_ERR_CUDA;
    }
    if (bp < ((size_t)8 << 20)) {                     // small output: launch-latency-bound, one graph replay and one copy
        const int rc = ls_execute(p, p->st_t, p->st_y, p->st_dy, p->st_p, cuda_stream);
        if (rc != LS_OK) return rc;
        if (cudaMemcpyAsync(power, p->st_p, bp, cudaMemcpyDeviceToHost, s) != cudaSuccess || cudaStreamSynchronize(s) != cudaSuccess) {
            cudaGetLastError();
            return LS_ERR_CUDA;
        }
        return LS_OK;
    }
    // Direct launches (their host cost hides behind the input copies), the power copied out piece by piece on a second
    // stream while the next piece is computed; the stream s is joined with it before the final synchronise.
    if (!p->copy_stream && (cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking) != cudaSuccess ||
                            cudaEventCreateWithFlags(&p->copy_ev, cudaEventDisableTiming) != cudaSuccess)) {
        cudaGetLastError();
        return LS_ERR_CUDA;
    }
    const int rc = enqueue_execute(p, p->st_t, p->st_y, p->st_dy, p->st_p, s, (char*)power);
    if (rc != LS_OK) {
        cudaStreamSynchronize(p->copy_stream);
        return rc;
    }
    if (cudaEventRecord(p->copy_ev, p->copy_stream) != cudaSuccess || cudaStreamWaitEvent(s, p->copy_ev, 0) != cudaSuccess ||
        cudaStreamSynchronize(s) != cudaSuccess) {
        cudaGetLastError();
        return LS_ERR_CUDA;
    }
    return LS_OK;
}

int ls_get_info(ls_plan_t p, double* sigma, int* w, double* beta, int64_t* n, int* M, double* model_bytes) {
    if (!p) return LS_ERR_INVALID_VALUE;
    if (sigma) *sigma = (double)p->n / (double)p->Nf;
    if (w) *w = p->w;
    if (beta) *beta = p->beta;
    if (n) *n = p->n;
    if (M) *M = p->M;
    if (model_bytes) *model_bytes = p->model_bytes;
    return LS_OK;
}

size_t ls_workspace_bytes(ls_plan_t p) { return p ? p->total_bytes : 0; }

int ls_set_workspace(ls_plan_t p, void* dptr, size_t bytes) {
    if (!p || !dptr || ((uintptr_t)dptr & 255) != 0) return LS_ERR_INVALID_VALUE;
    auto up = [](size_t b) { return (b + 255) & ~(size_t)255; };
    const size_t need = up(p->grids_bytes) + up(p->modes_bytes) + up(p->fft_work_bytes);
    if (bytes < need || bytes < p->total_bytes) return LS_ERR_INVALID_VALUE;
    if (cudaSetDevice(p->opts.device) != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) {
        cudaGetLastError();
        return LS_ERR_CUDA;
    }
    if (!p->external_ws) {
        dfree(p, p->grids);
        dfree(p, p->modes);
        dfree(p, p->fft_work);
    }
    char* base = (char*)dptr;
    p->grids = base;
    p->modes = p->modes_bytes ? base + up(p->grids_bytes) : nullptr;
    p->fft_work = base + up(p->grids_bytes) + up(p->modes_bytes);
    p->external_ws = true;
    if (p->gexec) { cudaGraphExecDestroy(p->gexec); p->gexec = nullptr; }     // captured pointers are stale
    if (p->own_fft && lsb::own_fft_make_tmap(p) != cudaSuccess) { cudaGetLastError(); return LS_ERR_CUDA; }
    if (!p->own_fft) {
        if (cufftSetWorkArea(p->fft_first, p->fft_work) != CUFFT_SUCCESS) return LS_ERR_CUFFT;
        if (p->has_chunk && cufftSetWorkArea(p->fft_chunk, p->fft_work) != CUFFT_SUCCESS) return LS_ERR_CUFFT;
        if (p->has_rem && cufftSetWorkArea(p->fft_rem, p->fft_work) != CUFFT_SUCCESS) return LS_ERR_CUFFT;
    }
    return LS_OK;
}

int ls_get_stage_ms(ls_plan_t p, float* ms, int n_stages) {
    if (!p || !ms || n_stages < 1) return LS_ERR_INVALID_VALUE;
    if (!p->opts.timing || !p->timed_once) return LS_ERR_NOT_READY;
    float acc[LS_NUM_STAGES] = {0};
    for (size_t i = 0; i < p->events_used; ++i) {
        const lsb::StageEvent& ev = p->events[i];
        if (cudaEventSynchronize(ev.end) != cudaSuccess) { cudaGetLastError(); return LS_ERR_CUDA; }
        float v = 0;
        if (cudaEventElapsedTime(&v, ev.beg, ev.end) != cudaSuccess) { cudaGetLastError(); return LS_ERR_CUDA; }
        acc[ev.stage] += v;
        if (ev.stage >= LS_STAGE_FFT_PASS1 && ev.stage <= LS_STAGE_FFT_PASS3) acc[LS_STAGE_FFT] += v;
    }
    for (int i = 0; i < n_stages && i < LS_NUM_STAGES; ++i) ms[i] = acc[i];
    return LS_OK;
}

int ls_get_launch_counts(ls_plan_t p, int* own_kernels, int* fft_execs) {
    if (!p) return LS_ERR_INVALID_VALUE;
    if (p->own_kernels == 0) return LS_ERR_NOT_READY;
    if (own_kernels) *own_kernels = p->own_kernels;
    if (fft_execs) *fft_execs = p->fft_execs;
    return LS_OK;
}

int ls_debug_stats(ls_plan_t p, double* out) {
    if (!p || !out) return LS_ERR_INVALID_VALUE;
    std::vector<double> h((size_t)p->batch * 4);
    if (cudaDeviceSynchronize() != cudaSuccess ||
        cudaMemcpy(h.data(), p->sums, h.size() * 8, cudaMemcpyDeviceToHost) != cudaSuccess) {
        cudaGetLastError();
        return LS_ERR_CUDA;
    }
    const bool per = p->opts.dy_per_series != 0;
    for (int s = 0; s < p->batch; ++s) {
        const double W = h[per ? 4 * s : 0];
        out[3 * s + 0] = W;
        out[3 * s + 1] = h[4 * s + 1] / W;
        out[3 * s + 2] = h[4 * s + 2];
    }
    return LS_OK;
}

int ls_debug_modes(ls_plan_t p, int series, int64_t K, const int64_t* kidx, double* out) {
    if (!p || !kidx || !out || K < 1 || series < 0 || series >= p->batch) return LS_ERR_INVALID_VALUE;
    if (p->chunk < p->batch) return LS_ERR_NOT_READY;          // grids of earlier passes are gone
    for (int64_t i = 0; i < K; ++i)
        if (kidx[i] < 0 || kidx[i] >= p->Nf) return LS_ERR_INVALID_VALUE;
    const bool per = p->opts.dy_per_series != 0;
    const int C = p->batch;
    const int nw = p->opts.no_floating_mean ? 0 : 1;
    const int w2_slot = per ? series : 0;
    const int h_slot = per ? C + (1 + nw) * series + nw : 1 + nw + series;
    const int w_slot = !nw ? w2_slot : (per ? C + 2 * series : 1);     // fixed mean: no w transform (reported as w2's)
    int64_t* dk = nullptr;
    double* dout = nullptr;
    int rc = LS_OK;
    if (cudaMalloc((void**)&dk, K * 8) != cudaSuccess || cudaMalloc((void**)&dout, K * 48) != cudaSuccess) rc = LS_ERR_ALLOC;
    if (rc == LS_OK && (cudaDeviceSynchronize() != cudaSuccess ||
                        (p->fuse_assemble && lsb::launch_own_fft_pass3(p, h_slot, 1, 0) != cudaSuccess) ||
                        cudaMemcpy(dk, kidx, K * 8, cudaMemcpyHostToDevice) != cudaSuccess ||
                        lsb::launch_debug_modes(p, h_slot, w_slot, w2_slot, K, dk, dout, 0) != cudaSuccess ||
                        cudaMemcpy(out, dout, K * 48, cudaMemcpyDeviceToHost) != cudaSuccess))
        rc = LS_ERR_CUDA;
    cudaFree(dk);
    cudaFree(dout);
    if (rc != LS_OK) cudaGetLastError();
    return rc;
}

// ---- stage pins (tests only): intermediates of the pre-processing, spreading and assembly stages ------------------
int ls_debug_points(ls_plan_t p, int set, double* out) {
    if (!p || !out || set < 0 || set > 1) return LS_ERR_INVALID_VALUE;
    if (cudaDeviceSynchronize() != cudaSuccess) { cudaGetLastError(); return LS_ERR_CUDA; }
    const size_t Nd = (size_t)p->Nd;
    if (p->dtype == LS_F64) {
        std::vector<lsb::Rec64> h(Nd);
        if (cudaMemcpy(h.data(), p->ps[set].rec, Nd * sizeof(lsb::Rec64), cudaMemcpyDeviceToHost) != cudaSuccess) { cudaGetLastError(); return LS_ERR_CUDA; }
        for (size_t i = 0; i < Nd; ++i) { out[4 * i] = h[i].eta; out[4 * i + 1] = h[i].l0; out[4 * i + 2] = h[i].qx; out[4 * i + 3] = h[i].qy; }
    } else {
        std::vector<lsb::Rec32> h(Nd);
        if (cudaMemcpy(h.data(), p->ps[set].rec, Nd * sizeof(lsb::Rec32), cudaMemcpyDeviceToHost) != cudaSuccess) { cudaGetLastError(); return LS_ERR_CUDA; }
        for (size_t i = 0; i < Nd; ++i) { out[4 * i] = h[i].eta; out[4 * i + 1] = h[i].l0; out[4 * i + 2] = h[i].qx; out[4 * i + 3] = h[i].qy; }
    }
    return LS_OK;
}

int ls_debug_bins(ls_plan_t p, int set, int* out) {
    if (!p || !out || set < 0 || set > 1) return LS_ERR_INVALID_VALUE;
    if (cudaDeviceSynchronize() != cudaSuccess ||
        cudaMemcpy(out, p->ps[set].bin_start, (size_t)(p->nbins + 1) * 4, cudaMemcpyDeviceToHost) != cudaSuccess) {
        cudaGetLastError();
        return LS_ERR_CUDA;
    }
    return LS_OK;
}

int ls_debug_grid(ls_plan_t p, const void* t, const void* y, const void* dy, int slot, double* out) {
    if (!p || !t || !y || !dy || !out || slot < 0 || slot >= p->slots) return LS_ERR_INVALID_VALUE;
    if (p->fft_prune) return LS_ERR_UNSUPPORTED;           // tiles without points do not exist on the pruned path
    p->debug_stop_after_spread = true;
    const int rc = enqueue_execute(p, t, y, dy, nullptr, 0);
    p->debug_stop_after_spread = false;
    if (rc != LS_OK) return rc;
    if (cudaDeviceSynchronize() != cudaSuccess) { cudaGetLastError(); return LS_ERR_CUDA; }
    const size_t n = (size_t)p->n;
    if (p->dtype == LS_F64) {
        if (cudaMemcpy(out, (const char*)p->grids + (size_t)slot * n * 16, n * 16, cudaMemcpyDeviceToHost) != cudaSuccess) { cudaGetLastError(); return LS_ERR_CUDA; }
    } else {
        std::vector<float> h(2 * n);
        if (cudaMemcpy(h.data(), (const char*)p->grids + (size_t)slot * n * 8, n * 8, cudaMemcpyDeviceToHost) != cudaSuccess) { cudaGetLastError(); return LS_ERR_CUDA; }
        for (size_t i = 0; i < 2 * n; ++i) out[i] = h[i];
    }
    return LS_OK;
}

int ls_debug_dinv(ls_plan_t p, int64_t K, const int64_t* kabs, double* out) {
    if (!p || !kabs || !out || K < 1) return LS_ERR_INVALID_VALUE;
    if (cudaDeviceSynchronize() != cudaSuccess) { cudaGetLastError(); return LS_ERR_CUDA; }
    for (int64_t i = 0; i < K; ++i) {
        if (kabs[i] < 0 || kabs[i] > p->Nf / 2) return LS_ERR_INVALID_VALUE;
        if (cudaMemcpy(out + i, p->dinv + kabs[i], 8, cudaMemcpyDeviceToHost) != cudaSuccess) { cudaGetLastError(); return LS_ERR_CUDA; }
    }
    return LS_OK;
}

int ls_debug_assemble(int64_t K, const double* sums, double YY, double W, int no_floating_mean, int normalization, double* out) {
    if (!sums || !out || K < 1 || normalization < 0 || normalization > 3) return LS_ERR_INVALID_VALUE;
    double *ds = nullptr, *dout = nullptr;
    int rc = LS_OK;
    if (cudaMalloc((void**)&ds, K * 48) != cudaSuccess || cudaMalloc((void**)&dout, K * 8) != cudaSuccess) rc = LS_ERR_ALLOC;
    if (rc == LS_OK && (cudaMemcpy(ds, sums, K * 48, cudaMemcpyHostToDevice) != cudaSuccess ||
                        lsb::launch_debug_assemble(K, ds, YY, W, no_floating_mean, normalization, dout, 0) != cudaSuccess ||
                        cudaMemcpy(out, dout, K * 8, cudaMemcpyDeviceToHost) != cudaSuccess))
        rc = LS_ERR_CUDA;
    cudaFree(ds);
    cudaFree(dout);
    if (rc != LS_OK) cudaGetLastError();
    return rc;
}

int ls_debug_guards(ls_plan_t p, int64_t* damaged_bytes) {
    if (!p || !damaged_bytes) return LS_ERR_INVALID_VALUE;
    if (!p->guard) return LS_ERR_NOT_READY;
    if (cudaDeviceSynchronize() != cudaSuccess) { cudaGetLastError(); return LS_ERR_CUDA; }
    int64_t bad = 0;
    unsigned char h[kGuardBytes];
    for (const auto& gz : p->guards) {
        if (!gz.first) continue;
        for (int side = 0; side < 2; ++side) {
            const char* src = gz.first + (side ? kGuardBytes + gz.second : 0);
            if (cudaMemcpy(h, src, kGuardBytes, cudaMemcpyDeviceToHost) != cudaSuccess) { cudaGetLastError(); return LS_ERR_CUDA; }
            for (size_t i = 0; i < kGuardBytes; ++i) bad += h[i] != 0xA5;
        }
    }
    *damaged_bytes = bad;
    return LS_OK;
}

}  // extern "C"
