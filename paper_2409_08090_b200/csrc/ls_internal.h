// ls_internal.h — plan structure and kernel launchers shared by the library's translation units.
// Internal to libls_b200.so; the public boundary is include/ls.h.  Nothing here is shared with
// oracle/ (the CPU oracle is test infrastructure and has its own, independent arithmetic).
#pragma once

#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>

#include <algorithm>
#include <utility>
#include <vector>

#include "../../include/ls.h"

namespace lsb {

constexpr int kMaxWidth = 20;        // widest spreading kernel supported (cells)
constexpr int kBinCells = 64;        // sort-bin length in fine-grid cells (>= kMaxWidth/2 + 1)
constexpr int kSpreadThreads = 256;  // threads per spreading CTA
constexpr int kChunkPts = 256;       // candidates a spreading CTA stages per pass (one per thread)
constexpr int kQuadNodes = 64;       // Gauss-Legendre nodes on [0,1] for psihat
constexpr int kMaxDeg = 12;          // highest degree of the piecewise-polynomial kernel (even; fp32 uses 8)
constexpr int kHalfMax = (kMaxWidth + 1) / 2;

// double-double constant (hi + lo), built on the host with FMA error-free products.
struct dd {
    double hi, lo;
};

// Piecewise-polynomial form of the spreading kernel ("piecewise polynomial kernel
// approximation"): on cell i of the support, psi(eta/2 + i - w/2 + 1/2) = sum_d c[i][d] eta^d for
// eta in [-1, 1).  psi is even, so piece w-1-i is piece i at -eta: only ceil(w/2) pieces are kept
// and each evaluation of (even part, odd part) yields two kernel values.
struct KernelPoly {
    int w = 0, deg = 0, half = 0;
    double c[kHalfMax][kMaxDeg + 1];
    double max_err = 0;              // measured on the host against exp/sqrt at plan time
};

// One bin-sorted non-uniform point, as the spreading kernel reads it (one 32-byte / 16-byte load).
//   eta  position of the point inside its cell pattern: the first touched cell l0 lies
//        x0 = (eta + 1)/2 - w/2 cells from the point, x0 in [-w/2, -w/2 + 1)
//   l0   first fine-grid cell touched (unfolded: may be < 0 or >= n by less than w)
//   q    unit phasor e^{2 pi i f_c t} (x1 point set) or its square (x2)
struct __align__(32) Rec64 {
    double eta;
    int l0, pad;
    double qx, qy;
};
struct __align__(16) Rec32 {
    float eta;
    int l0;
    float qx, qy;
};

// One non-uniform point set in bin-sorted order (x1 = n df t, or x2 = 2 x1).
struct PointSet {
    int* hist = nullptr;       // [nbins]   bin counts -> running cursors during the scatter
    int* bin_start = nullptr;  // [nbins+1] exclusive scan of the counts
    int* perm = nullptr;       // [Nd]      input index of sorted slot s (when a rows kernel runs)
    void* rec = nullptr;       // [Nd]      Rec64 / Rec32, sorted order
    void* rows = nullptr;      // [nrows][Nd] T  stored real strengths, sorted order (shared dy: y - ybar only)
    int nrows = 0;
};

struct StageEvent {
    int stage;
    cudaEvent_t beg, end;
};

}  // namespace lsb

struct ls_plan_s {
    // problem
    int64_t Nd = 0, Nf = 0, n = 0;
    double f0 = 0, df = 0, eps = 0;
    int dtype = LS_F64, batch = 1;
    ls_opts opts{};
    // chosen parameters
    double sigma = 2.0, beta = 0;
    int w = 0;
    int L = 1024;          // spreading tile length (cells), multiple of kBinCells
    int nbins = 0;         // ceil(n / kBinCells)
    int ntiles = 0;        // ceil(n / L)
    int num_sms = 148;     // multiprocessors of the plan's device (filler CTAs of the spread kernel)
    int tile_stride = 1;   // launch-order permutation of the tiles: coprime to ntiles, ~0.618 ntiles
    int M = 0;             // transforms per execute
    int chunk = 1;         // series per pass
    int slots = 0;         // grid slots allocated
    lsb::dd ndf{}, fc{};   // n*df and f_c = f0 + floor(Nf/2) df as double-doubles
    // device buffers
    void* grids = nullptr;      // [slots][n] complex T
    double* dinv = nullptr;     // [floor(Nf/2)+1] 1/psihat(k')
    double* t64 = nullptr;      // [Nd] times promoted from float (opts.t_is_dtype on an LS_F32 plan)
    double* sums = nullptr;     // [batch][4]  (sum dy^-2, sum dy^-2 y, YY, unused); first part of `zeroed`
    void* zeroed = nullptr;     // sums + both histograms: one allocation, one memset per execute
    size_t zeroed_bytes = 0;
    lsb::KernelPoly poly;       // piecewise-polynomial spreading kernel (host copy; passed by value)
    int* scan_tmp = nullptr;    // block sums + ticket for the bin scan (both point sets)
    lsb::PointSet ps[2];
    // host staging for ls_execute_host
    void *st_t = nullptr, *st_y = nullptr, *st_dy = nullptr, *st_p = nullptr;
    cudaStream_t copy_stream = nullptr;             // ls_execute_host: device -> host copies of finished power, beside the kernels
    cudaEvent_t copy_ev = nullptr;
    // cuFFT
    cufftHandle fft_first = 0, fft_chunk = 0, fft_rem = 0;
    bool has_first = false, has_chunk = false, has_rem = false;
    int first_batch = 0, rem_batch = 0;
    void* fft_work = nullptr;
    size_t fft_work_bytes = 0;
    size_t total_bytes = 0;
    size_t grids_bytes = 0, modes_bytes = 0;
    bool external_ws = false;   // grids / modes / fft_work live in caller memory (ls_set_workspace)
    // own FFT (ls_fft.cu): fp64, n = 2^12 .. 2^24 (first pass pruned from 2^20 on); opts.fft_impl
    bool own_fft = false;
    bool fft_prune = false;                         // spreading skips empty tiles, FFT pass 1 prunes by liveness masks
    bool list_tiles = false;                        // cuFFT path: empty tiles zero-filled by a sweep kernel, spreading walks
                                                    // the list of occupied tiles (ls_tile_zero_list_kernel)
    void* ftab = nullptr;                           // fuse_assemble: [Nf][2] double2 per-frequency assembly terms
    bool fuse_assemble = false;                    // third pass of the h transforms fused with K5 + K6
    bool fuse_pass23 = false;                      // FFT passes 2 + 3 as one persistent kernel (intermediate in L2)
    void *fft_wlo = nullptr, *fft_whi = nullptr;   // twiddle tables w_n^x, w_n^{4096 y}
    void* modes = nullptr;                          // [slots][Nf] complex: kept modes in frequency order
    int* tile_list = nullptr;                       // [2][ntiles] occupied spreading tiles per point set (x2, x1)
    int* tile_counts = nullptr;                     // [2] list lengths (in `zeroed`)
    int* fft_queue = nullptr;                       // [2 + 16 slots] work queue of the fused FFT passes 2 + 3 (in `zeroed`)
    unsigned* row_masks = nullptr;                  // [2][65536/L][<=16] liveness bits for FFT pass 1 (in `zeroed`)
    alignas(64) unsigned char fft_tmap[128] = {0};  // CUtensorMap over the fine grids (pass-2 tiles of the fused FFT kernel)
    // CUDA-graph replay of the execute sequence (launch-latency-bound small problems; opts.graph)
    bool use_graph = false;
    cudaGraphExec_t gexec = nullptr;
    const void *g_t = nullptr, *g_y = nullptr, *g_dy = nullptr;
    void* g_power = nullptr;
    int g_misses = 0;           // consecutive executes that had to re-capture (auto mode gives up at 3)
    // timing
    std::vector<lsb::StageEvent> events;
    size_t events_used = 0;
    bool timed_once = false;
    int own_kernels = 0, fft_execs = 0;
    bool debug_stop_after_spread = false;   // ls_debug_grid
    bool guard = false;                     // LS_B200_GUARD: allocations carry guard zones (ls_debug_guards)
    std::vector<std::pair<char*, size_t>> guards;   // (base of the guarded allocation, payload bytes)
    double model_bytes = 0;
};

namespace lsb {

// ---- ls_pre.cu: K1 stats + K3 bin count, K3 scan, K2 premultiply + scatter (+ rows) -------
cudaError_t launch_promote_t(ls_plan_s* p, const void* t_f32, cudaStream_t s);
cudaError_t launch_stats_count(ls_plan_s* p, const double* t, const void* y, const void* dy, cudaStream_t s);
cudaError_t launch_bin_scan(ls_plan_s* p, cudaStream_t s);
cudaError_t launch_premultiply(ls_plan_s* p, const double* t, const void* y, const void* dy, cudaStream_t s);
cudaError_t launch_rows(ls_plan_s* p, const void* y, const void* dy, cudaStream_t s);
// ---- ls_spread.cu: K4 ----------------------------------------------------------------------
// One launch spreads rows [row0_x2, +nrows_x2) of the x2 point set into slots slot0_x2.. and rows
// [row0_x1, +nrows_x1) of the x1 point set into slots slot0_x1.. (either count may be 0).
cudaError_t launch_spread(ls_plan_s* p, int row0_x2, int nrows_x2, int slot0_x2, int row0_x1, int nrows_x1,
                          int slot0_x1, cudaStream_t s);
int spread_rows_per_group(const ls_plan_s* p);
cudaError_t launch_tile_list(ls_plan_s* p, cudaStream_t s);
cudaError_t launch_zero_list(ls_plan_s* p, int nrows_x2, int slot0_x2, int nrows_x1, int slot0_x1, int build_list, cudaStream_t s);
// ---- ls_fft.cu: own FFT (fp64, n = 2^12 .. 2^24; first pass pruned and passes 2 + 3 fused from 2^20 on) ------
bool own_fft_supported(const ls_plan_s* p);
// ---- ls_fft_f32.cu: the own FFT for fp32 grids of 5 x 2^22 .. 5 x 2^25 cells (three passes 80 RM x 256 x 512)
int own_fft_f32_rm(const ls_plan_s* p);           // RM of those sizes (fp32 plans only), else 0
cudaError_t own_fft_f32_init(ls_plan_s* p, cudaStream_t s);
cudaError_t launch_own_fft_f32_pass1(ls_plan_s* p, int slot0, int ntrans, int n_x2, cudaStream_t s);
cudaError_t launch_own_fft_f32_pass2(ls_plan_s* p, int slot0, int ntrans, cudaStream_t s);
cudaError_t launch_own_fft_f32_pass3(ls_plan_s* p, int slot0, int ntrans, cudaStream_t s);
int own_fft_rm5(const ls_plan_s* p);              // n = 5 x 2^k (two passes 80 RM x 256): RM, else 0
bool own_fft_prunes(const ls_plan_s* p);          // first pass pruned by liveness masks (n >= 2^20)
int own_fft_ncoltiles(const ls_plan_s* p);        // spreading tiles per liveness-mask column
int own_fft_rb(const ls_plan_s* p);               // pass-1 radix / 16 (where that pass is the 16 x RB kernel)
cudaError_t own_fft_init(ls_plan_s* p, cudaStream_t s);
cudaError_t own_fft_make_tmap(ls_plan_s* p);      // (re-)encode the tensor map of the fine grids (plan, ls_set_workspace)
cudaError_t launch_own_fft_pass1(ls_plan_s* p, int slot0, int ntrans, int n_x2, cudaStream_t s);
cudaError_t launch_own_fft_pass2(ls_plan_s* p, int slot0, int ntrans, cudaStream_t s);
cudaError_t launch_own_fft_pass3(ls_plan_s* p, int slot0, int ntrans, cudaStream_t s);
cudaError_t launch_own_fft_pass23(ls_plan_s* p, int slot0, int ntrans, cudaStream_t s);
cudaError_t launch_own_fft_assemble(ls_plan_s* p, int h_slot0, int nseries, int series0, int w_slot, int w2_slot,
                                    void* power, cudaStream_t s);
// ---- ls_post.cu: P0 table, K5+K6 -----------------------------------------------------------
cudaError_t launch_deconv_table(ls_plan_s* p, const double* nodes, const double* weights, cudaStream_t s);
cudaError_t launch_assemble(ls_plan_s* p, int series0, int nseries, int h_slot, int h_stride, int w_slot,
                            int w_stride, int w2_slot, int w2_stride, void* power, cudaStream_t s, long long k0 = 0,
                            long long k1 = -1);      // frequencies [k0, k1); k1 < 0: to Nf
cudaError_t launch_debug_modes(ls_plan_s* p, int h_slot, int w_slot, int w2_slot, int64_t K,
                               const int64_t* d_kidx, double* d_out, cudaStream_t s);
cudaError_t launch_debug_assemble(int64_t K, const double* d_sums, double YY, double W, int no_float, int norm,
                                  double* d_out, cudaStream_t s);

}  // namespace lsb
