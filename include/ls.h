/*
 * ls.h — C ABI of the B200-native floating-mean Lomb-Scargle hot path (libls_b200.so).
 *
 * What the library computes (citations: PAPER.md = /root/reference/PAPER.md of arXiv:2409.08090;
 * north_star = BASELINE.json "north_star"; readings A1..A17 = DESIGN.md §3):
 *
 *   For each series b of a batch sharing one time array t[Nd] (batched mode) the
 *   standard-normalised, weighted, floating-mean Lomb-Scargle power at f_k = f0 + k df,
 *   k = 0..Nf-1 (Eq. 1; A1), obtained from the six trigonometric sums
 *       Sh,Ch = sum_j h_j {sin,cos}(2 pi f_k t_j)     h_j = w_j (y_j - ybar_w)
 *       S ,C  = sum_j w_j {sin,cos}(2 pi f_k t_j)     w_j = dy_j^-2 / sum dy^-2
 *       S2,C2 = sum_j w_j {sin,cos}(4 pi f_k t_j)
 *   which are the real/imaginary parts of three type-1 (non-uniform -> uniform) NUFFTs
 *   (PAPER.md:24-27 Eq. 2, :45): strengths pre-multiplied by e^{2 pi i f_c t_j}
 *   (f_c = f0 + floor(Nf/2) df; A4), spread onto a fine grid of n ~ sigma Nf cells with the
 *   "exponential of semicircle" kernel, one equispaced FFT, diagonal rescaling
 *   (PAPER.md:47), then the tau / YY,YC,YS,CC,SS assembly named by north_star.
 *
 * Every step runs in hand-written sm_100a kernels (stats, bin-count + scan, premultiply-scatter,
 * tile-owner spread, deconvolve + assemble).  The fine-grid FFT is the library's own three-pass
 * transform for fp64 power-of-two grids of 2^12..2^24 cells (first pass pruned from 2^20 cells on)
 * and one cuFFT plan for every other grid.  There is NO CPU fallback: every entry point
 * fails with LS_ERR_CUDA when no device is usable.  From 2^20 cells on, passes 2 + 3 of the own FFT are one
 * persistent kernel that moves its tiles with TMA (cp.async.bulk.tensor / cp.async.bulk + mbarriers).
 *
 * Conventions
 *   - All functions return an int status (LS_OK == 0); nothing throws, prints or exits.
 *   - Pointers passed to ls_execute are DEVICE pointers; to ls_execute_host they are HOST
 *     pointers.  The caller owns them; the library never frees or writes inputs.
 *   - Layouts (row-major, contiguous):  t[Nd] (double; float only with opts.t_is_dtype on an
 *     LS_F32 plan);  y[batch][Nd], power[batch][Nf] in `dtype`;  dy[Nd] (shared by the batch) or
 *     dy[batch][Nd] when opts.dy_per_series.
 *     power[b][k] is the periodogram of series b at f0 + k*df.
 *   - ls_execute only ENQUEUES work on `cuda_stream` (a cudaStream_t; NULL = legacy default
 *     stream) and returns; it performs no device synchronisation.  One execute may be in flight
 *     per plan (plan-owned scratch); use one plan per stream for concurrency.
 *   - ls_plan makes opts.device the calling thread's current device and leaves it so; ls_execute,
 *     ls_execute_host and ls_direct_power expect the plan's device to be current and `cuda_stream`
 *     to belong to it (they never switch devices themselves).
 *   - dy_j <= 0 or non-finite inputs give undefined (NaN-propagating) output; there is no
 *     device-side validation on the hot path.
 */
#ifndef LS_B200_H
#define LS_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ls_plan_s* ls_plan_t;            /* opaque; owns cuFFT plan, tables, scratch */

enum { LS_NORM_STANDARD = 0, LS_NORM_MODEL = 1, LS_NORM_LOG = 2, LS_NORM_PSD = 3 };
enum { LS_F32 = 0, LS_F64 = 1 };                /* dtype of y, dy, power, fine grid and FFT (A9:
                                                   t, grid coordinates, phase reduction and the
                                                   assembly are fp64 for both) */
enum {
    LS_OK = 0,
    LS_ERR_INVALID_VALUE = 1,   /* bad argument (see ls_plan) */
    LS_ERR_ALLOC = 2,           /* host or device allocation failed */
    LS_ERR_CUDA = 3,            /* CUDA runtime error, or no usable device */
    LS_ERR_CUFFT = 4,           /* cuFFT error */
    LS_ERR_UNSUPPORTED = 5,     /* size outside what the kernels index (n >= 2^31) */
    LS_ERR_NOT_READY = 6,       /* information requested before it exists */
    LS_ERR_TOO_LARGE = 7        /* size beyond the fixed scratch of a no-allocation entry point (LS_NOALLOC_MAX_ND) */
};

/* Stage indices for ls_get_stage_ms (CUDA-event timings of the last execute when opts.timing). */
enum {
    LS_STAGE_STATS = 0,         /* K1  weights, weighted mean                                    */
    LS_STAGE_SORT = 1,          /* K3  bin count + scan (both point sets)                        */
    LS_STAGE_PREMUL = 2,        /* K2  time-rescale, phase premultiply, scatter to bin order, YY */
    LS_STAGE_SPREAD = 3,        /* K4  tile-owner spreading of all M grids                       */
    LS_STAGE_FFT = 4,           /* F   the fine-grid FFT: cuFFT, or the own passes 1-3 (reported
                                       separately, north_star)                                   */
    LS_STAGE_ASSEMBLE = 5,      /* K5+K6 mode extraction, deconvolution, tau + power assembly; with
                                       fft_impl = 2 it contains the h transforms' third FFT pass,
                                       which is fused with it                    */
    LS_STAGE_TOTAL = 6,         /* whole execute                                                 */
    LS_STAGE_FFT_PASS1 = 7,     /* own FFT only: the three passes, also summed into LS_STAGE_FFT  */
    LS_STAGE_FFT_PASS2 = 8,     /*   (auto mode, n >= 2^20: the fused passes 2 + 3; PASS3 is then 0)            */
    LS_STAGE_FFT_PASS3 = 9,     /*   (pass 3 of the transforms whose modes go to the compact array) */
    LS_NUM_STAGES = 10
};

/* Optional tuning; a zero-initialised struct (or NULL) selects the defaults. */
typedef struct {
    int dy_per_series;      /* 0: dy[Nd] shared by the batch (A13, default); 1: dy[batch][Nd]     */
    double upsampfac;       /* sigma; 0 = auto: n = the power of two in [1.25 Nf, 2.5 Nf) (or, where that is much
                               larger than needed, the fastest of a few timed smooth sizes: the choice is cached
                               per process, and may differ between processes / devices, as do the last bits of the
                               results: scatter order inside a sort bin and the statistics' atomic sums are
                               unordered).  Non-zero: n = the smallest even 5-smooth size >= upsampfac * Nf   */
    int kernel_width;       /* w in fine-grid cells, 2..20; 0 = auto from eps (A10).  The kernels hold at most 20
                               cells: where eps needs more at the automatic sigma the grid doubles; with a fixed
                               upsampfac the plan is refused with LS_ERR_UNSUPPORTED                        */
    int timing;             /* 1: record CUDA events around each stage of every execute           */
    int device;             /* CUDA device ordinal the plan lives on                              */
    int tile_cells;         /* spreading tile length L in cells: 256, 512 or 1024 (1024: single series only);
                               0 = auto                                                           */
    int batch_chunk;        /* series spread/FFT'd/assembled per pass; 0 = auto (<= 8 GB of grids)  */
    int no_autotune;        /* 1: never time candidate grid sizes at plan time (auto n = power of two) */
    int graph;              /* CUDA-graph replay of the execute sequence (needs timing == 0 and a non-legacy
                               stream): 0 = auto (on; off for good after three consecutive executes
                               with changed buffer pointers), 1 = never, 2 = always                 */
    int fft_impl;           /* 0 = auto: the library's own FFT where it exists (fp64 grids of 2^12..2^24 cells
                               and of 5 x 2^13..5 x 2^16 cells, fp32 grids of 5 x 2^22..5 x 2^25 cells; the powers
                               of two below 2^20 not for large batches), else cuFFT.  For n >= 2^20 the own FFT is a pruned first pass plus ONE
                               persistent kernel for passes 2 + 3 whose intermediate stays in L2.  A batch with
                               shared dy (upsampfac = 0, autotune on) takes a 5 x 2^k grid where one lies
                               between 1.25 Nf and the power of two: two passes, the first pruned, the last
                               fused with the assembly.  An fp32 plan of up to 8 transforms takes a grid of
                               5 x 2^k cells, k = 22..25, where one lies in that range: three passes, the first
                               pruned (ls_fft_f32.cu).  1 = cuFFT plan.  2 = own FFT,
                               three launches, the h transforms' last pass fused with deconvolution +
                               assembly (fp64 with shared dy; otherwise the same as 3).  3 = own FFT as three separate pass kernels and a separate
                               assembly (same arithmetic as auto; kept for comparison).  2 and 3 give
                               LS_ERR_UNSUPPORTED where the own FFT does not exist                   */
    int no_floating_mean;   /* 0: floating mean, six sums (default; north_star).  1: the fixed-mean form of
                               PAPER.md:17 ("four weighted trigonometric sums"): y centred by its weighted
                               mean, sinusoid model without an offset term                          */
    int normalization;      /* LS_NORM_STANDARD (default), _MODEL, _LOG, _PSD            */
    int t_is_dtype;         /* 0: t is double[Nd] (default, recommended: A9).  1 with LS_F32: t is float[Nd]; it is
                               promoted exactly to double on the device before anything else reads it  */
    int reserved[2];        /* zero in production.  Kernel variants kept for comparison and test knobs:
                               reserved[0] = 1: round-1 kernels (per-thread-load FFT passes 2 + 3; one spreading CTA per
                               tile on the cuFFT path), 2: three consumer groups in the FFT kernel / the zero-fill
                               sweep forced on the cuFFT path; reserved[1] = queue lag of the fused FFT passes (1..8) */
} ls_opts;

/* ls_plan — choose (sigma, w, beta, n) from eps ("width and fine grid size are
 * carefully chosen to match the user tolerance"; A10), build the deconvolution table
 * 1/psihat(k') ("diagonal rescaling"), the cuFFT plan and all scratch buffers.
 *   Nd >= 1 points, Nf >= 1 frequencies, f0 >= 0 and df > 0 finite (cycles per unit of t),
 *   eps in [1e-14, 1e-1] for LS_F64 / [1e-6, 1e-1] for LS_F32, 1 <= batch <= 65535 (a grid dimension
 *   of the per-series kernels).
 * Errors: LS_ERR_INVALID_VALUE for anything outside those ranges or out == NULL;
 * LS_ERR_UNSUPPORTED if the fine grid needs n >= 2^31 cells, or a fixed upsampfac needs a kernel wider than 20
 * cells for eps; LS_ERR_ALLOC / _CUDA / _CUFFT. */
int ls_plan(ls_plan_t* out, int64_t Nd, int64_t Nf, double f0, double df, double eps,
            int dtype, int batch, const ls_opts* opts /* NULL ok */);

/* ls_execute — one pass of the whole hot path (§8(a) K1..K6 + cuFFT) for `batch` series.
 *   t      device, const double[Nd]  (const float[Nd] with opts.t_is_dtype on an LS_F32 plan)
 *   y      device, const dtype[batch][Nd]
 *   dy     device, const dtype[Nd] (or [batch][Nd] with opts.dy_per_series)
 *   power  device, dtype[batch][Nf]   (written)
 *   cuda_stream  cudaStream_t to enqueue on.
 * Asynchronous; errors of earlier asynchronous work may surface here as LS_ERR_CUDA. */
int ls_execute(ls_plan_t plan, const void* t, const void* y, const void* dy, void* power,
               void* cuda_stream);

/* ls_execute_host — the same with HOST buffers: copies t, y, dy to plan-owned device staging
 * buffers, executes, copies power back and synchronises the stream before returning.  Pinned
 * host memory makes the copies asynchronous with respect to each other, pageable memory works.
 * Outputs of 8 MB and more leave the device piece by piece on a plan-owned second stream while the
 * next piece is computed: a batch pass by pass (so a batch_chunk below the batch size hides the
 * kernels behind the copy-out; one pass cannot), one long series (Nf >= 2^22) in frequency
 * quarters of the assembly.  `power` is complete, and both streams idle, when the call returns. */
int ls_execute_host(ls_plan_t plan, const void* t, const void* y, const void* dy, void* power,
                    void* cuda_stream);

/* Parameters the plan chose.  Any out-pointer may be NULL.
 *   sigma = n/Nf realised, w = kernel width, beta = ES shape parameter, n = fine-grid cells,
 *   M = transforms per execute (batch + 2 with shared dy; 3*batch with per-series dy),
 *   model_bytes = algorithmic HBM bytes per execute excluding the FFT. */
int ls_get_info(ls_plan_t plan, double* sigma, int* w, double* beta, int64_t* n, int* M,
                double* model_bytes);

/* Device bytes the plan allocated (grids + mode array + FFT work area + tables + scratch). */
size_t ls_workspace_bytes(ls_plan_t plan);

/* ls_set_workspace — run the plan's large buffers (fine grids, compact mode array, cuFFT work area)
 * inside caller-owned device memory, e.g. a torch allocation: `dptr` must be 256-byte aligned and hold
 * at least ls_workspace_bytes(plan) bytes (more than the three buffers need, so that size always
 * suffices).  The plan frees its own copies; the caller keeps ownership of `dptr` and must keep it alive
 * until ls_destroy or the next ls_set_workspace.  Not to be called while an execute is in flight.
 * Errors: LS_ERR_INVALID_VALUE (NULL plan or pointer, misaligned, too small), LS_ERR_CUFFT. */
int ls_set_workspace(ls_plan_t plan, void* dptr, size_t bytes);

/* Milliseconds per stage of the most recent execute (needs opts.timing = 1; synchronises on the
 * recorded events).  ms[LS_NUM_STAGES]; n_stages entries are written.  LS_ERR_NOT_READY if no
 * timed execute has run. */
int ls_get_stage_ms(ls_plan_t plan, float* ms, int n_stages);

/* Number of kernels (own + cuFFT exec calls) one ls_execute enqueues: own_kernels counts the
 * library's own __global__ launches, fft_execs the cufftExec calls. */
int ls_get_launch_counts(ls_plan_t plan, int* own_kernels, int* fft_execs);

/* Test hooks: read intermediates of the most recent execute (synchronises the device).
 *   ls_debug_modes: the deconvolved NUFFT outputs g_k of series `series` at the K indices
 *     kidx[] (host) -> out[K][6] (host, double) = (Sh, Ch, S, C, S2, C2) as the assembly saw them.
 *     Only valid when the plan runs the batch in one pass (batch_chunk >= M) .
 *   ls_debug_stats: out[3*batch] (host) = (W, ybar, YY) per series. */
int ls_debug_modes(ls_plan_t plan, int series, int64_t K, const int64_t* kidx, double* out);
int ls_debug_stats(ls_plan_t plan, double* out);

/* Stage pins (SURVEY.md §8(c) "Stage pins for GPU kernels"): intermediates of single stages, all HOST output buffers,
 * all synchronise the device.  Layouts are those of the kernels and may change with them.
 *   ls_debug_points: the bin-sorted point records of the most recent execute, point set 0 (x1 = n df t) or 1
 *     (x2 = 2 x1): out[Nd][4] = (eta, l0, q_re, q_im); l0 = first fine-grid cell the point touches (unfolded),
 *     eta = 2 (l0 - u) + (w - 1) in [-1, 1) with u the point's grid coordinate; q = w_j e^{2 pi i f_c t_j} (x1) or
 *     w_j e^{4 pi i f_c t_j} (x2) when dy is shared by the batch, the unit phasor otherwise.
 *   ls_debug_bins: out[nbins + 1] = first sorted slot of every sort bin of 64 cells (nbins = ceil(n / 64)).
 *   ls_debug_grid: runs K1..K4 on (t, y, dy) (device pointers, legacy stream) and returns fine grid `slot` as the
 *     spreading kernel left it: out[n][2].  LS_ERR_UNSUPPORTED where empty tiles are not written (own FFT, n >= 2^20).
 *   ls_debug_dinv: out[i] = 1 / psihat(k') at |k'| = kabs[i] <= Nf / 2 (the P0 table).
 *   ls_debug_assemble: K6 alone (no plan): power of K frequencies from sums[K][6] = (Sh, Ch, S, C, S2, C2).
 *   ls_debug_guards: with the environment variable LS_B200_GUARD set when the plan was made, every plan-owned device
 *     allocation sits between two 256-byte guard zones; returns how many guard bytes any kernel has overwritten since
 *     (0 = no out-of-bounds write).  LS_ERR_NOT_READY for a plan made without the variable. */
int ls_debug_points(ls_plan_t plan, int set, double* out);
int ls_debug_bins(ls_plan_t plan, int set, int* out);
int ls_debug_grid(ls_plan_t plan, const void* t, const void* y, const void* dy, int slot, double* out);
int ls_debug_dinv(ls_plan_t plan, int64_t K, const int64_t* kabs, double* out);
int ls_debug_assemble(int64_t K, const double* sums, double YY, double W, int no_floating_mean, int normalization,
                      double* out);
int ls_debug_guards(ls_plan_t plan, int64_t* damaged_bytes);

/* ls_direct_power — verification path, NOT part of ls_execute: the six sums of
 * Eq. 1 evaluated by brute force, O(Nd K), for the K consecutive frequencies
 * f0 + (k0 + i) df, i = 0..K-1, of ONE fp64 series, then the same power assembly.  The kind of direct
 * evaluator the paper measures its errors against and compares with; it lets
 * the NUFFT path be checked on frequency ranges the CPU oracle cannot cover.
 *   t, y, dy  device, const double[Nd];   power  device, double[K] (written).
 * Allocates 40 Nd bytes of scratch, enqueues on `cuda_stream` and SYNCHRONISES it before returning.
 * Errors: LS_ERR_INVALID_VALUE, LS_ERR_ALLOC, LS_ERR_CUDA. */
int ls_direct_power(int64_t Nd, double f0, double df, int64_t k0, int64_t K, const void* t, const void* y,
                    const void* dy, void* power, void* cuda_stream);

/* ls_direct_sums — the same brute-force evaluation, but returning the six sums themselves and NOT the power:
 *   sums  device, double[K][6] = (Sh, Ch, S, C, S2, C2) of frequency f0 + (k0 + i) df (written).
 * None of the library's assembly arithmetic (tau, CC, SS) is involved, so a test can put these sums through the
 * ORACLE's assembly and check the NUFFT path's K6 independently of ls_power.cuh.  Same scratch, stream and error
 * behaviour as ls_direct_power. */
int ls_direct_sums(int64_t Nd, double f0, double df, int64_t k0, int64_t K, const void* t, const void* y,
                   const void* dy, void* sums, void* cuda_stream);

/* ls_direct_power_noalloc — ls_direct_power for callers that cannot allocate (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): same arguments, same kernels, same power, but the scratch (the
 * statistics and 40 bytes per point) is a fixed device array inside the library instead of a cudaMalloc per call.
 *   t, y, dy  device (on the CURRENT device), const double[Nd];   power  device, double[K] (written).
 *   Nd <= LS_NOALLOC_MAX_ND, else LS_ERR_TOO_LARGE (nothing is enqueued).
 * Calls no cudaMalloc / cudaFree and no allocating library routine; the first call on a device resolves the array's
 * device address (cudaGetSymbolAddress: make that call before a capture starts).  ASYNCHRONOUS, unlike ls_direct_power:
 * it enqueues one memset and three kernels on `cuda_stream` and returns; `power` is complete when the stream reaches
 * that point.  The array (256 + 40 LS_NOALLOC_MAX_ND bytes = 2.6 MB) is held by every GPU that loads the library until
 * the process exits, and is SHARED by all calls: calls that overlap on the GPU (two streams, two host threads) race on
 * it — serialise them on one stream or with events.
 * Errors: LS_ERR_INVALID_VALUE, LS_ERR_TOO_LARGE, LS_ERR_CUDA. */
#define LS_NOALLOC_MAX_ND 65536
int ls_direct_power_noalloc(int64_t Nd, double f0, double df, int64_t k0, int64_t K, const void* t, const void* y,
                            const void* dy, void* power, void* cuda_stream);

const char* ls_strerror(int code);

/* Frees everything the plan allocated.  NULL is accepted. */
int ls_destroy(ls_plan_t plan);

#ifdef __cplusplus
}
#endif
#endif /* LS_B200_H */
