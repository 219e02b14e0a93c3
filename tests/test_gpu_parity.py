"""-m gpu parity tests: the CUDA path (through the C-ABI binding) against the CPU oracle, element by
element on the same seeded inputs.

Gate (BASELINE.json north_star, reading A8): E_inf = max|P_gpu - P_or| / max P_or
  <= 1e-8 (fp64, eps 1e-9)   <= 1e-4 (fp32, eps 1e-5).
Pointwise statistics (the paper's metric) are asserted against the band the paper
reports for nifty-ls itself (median <= 1e-8, 99th percentile <= 1e-6 in fp64).
"""
import numpy as np
import pytest

from gpu_util import GATE_F32, GATE_F64, errors, gpu_power, oracle_power
from paper_2409_08090_b200.workloads import Workload, compare_indices, make_workload, scaled_workload

pytestmark = pytest.mark.gpu


def _custom(t, y, dy, f0, df, Nf, dtype="f64", eps=1e-9, name="custom"):
    t = np.ascontiguousarray(t, dtype=np.float64)
    npd = np.float64 if dtype == "f64" else np.float32
    y = np.atleast_2d(np.asarray(y, dtype=npd))
    dy = np.asarray(dy, dtype=npd)
    return Workload(name, t, np.ascontiguousarray(y), np.ascontiguousarray(dy), float(f0), float(df), int(Nf), dtype, eps)


def _check64(e, pointwise=True):
    assert e["Einf"] <= GATE_F64, e
    if pointwise:
        assert e["median"] <= 1e-8 and e["p99"] <= 1e-6, e


# ------------------------------------------------------------------ the five configs
def test_cfg1_full_grid():
    w = make_workload(1)
    Pg, ex = gpu_power(w, return_plan_info=True)
    Po = oracle_power(w)
    e = errors(Pg[0], Po)
    _check64(e)
    assert int(np.argmax(Pg[0])) == int(np.argmax(Po))
    assert ex["launches"][0] > 0 and ex["launches"][1] == 0            # our kernels ran, own FFT included (n = 2^14)
    assert ex["info"]["M"] == 3 and ex["info"]["n"] >= 1.25 * w.Nf


def test_cfg2_full_grid_unsorted_times():
    w = make_workload(2)
    Pg = gpu_power(w)
    e = errors(Pg[0], oracle_power(w, fast=True))
    _check64(e)
    ks = compare_indices(w, 512)
    _check64(errors(Pg[0][ks], oracle_power(w, ks=ks)), pointwise=False)   # strict direct evaluation on a subset


def test_cfg3_headline_size_sampled_frequencies():
    """Full size (N_d = 1e6, N_f = 1.25e7, n = 2.5e7) in the launch configuration bench.py times;
    compared on sampled k the oracle evaluates one by one (seam, edges and the injected peak included)."""
    w = make_workload(3)
    Pg = gpu_power(w)
    assert np.all(np.isfinite(Pg)) and Pg.min() >= -1e-12 and Pg.max() <= 1 + 1e-9
    ks = compare_indices(w, 2048)                                      # K = 2 048 at config 3
    Po = oracle_power(w, ks=ks)
    e = errors(Pg[0][ks], Po)
    _check64(e)
    assert e["max"] <= 1e-6, e                                         # pointwise MAX too (north_star "max relative error")
    kpk = ks[np.argmax(Po)]
    lo, hi = max(0, kpk - 50), min(w.Nf, kpk + 51)
    assert lo + int(np.argmax(Pg[0][lo:hi])) == kpk
    # the launch configuration bench.py times: a side stream, the captured graph replayed (n = 2^24), then a new
    # output buffer (re-capture): the same numbers as the direct launches above
    Pr = gpu_power(w, side_stream=True, repeat=3)
    assert np.max(np.abs(Pr - Pg)) <= 1e-13


def test_cfg3_own_fft_against_cufft_full_grid():
    """The library's own three-pass FFT (pruned first pass, compact mode output; ls_fft.cu) against the cuFFT
    path on the FULL grid of the headline config, and both against the oracle's direct sums on sampled k."""
    import oracle
    w = make_workload(3)
    ks = compare_indices(w, 256)
    P_own, ex_own = gpu_power(w, fft_impl=2, return_plan_info=True, debug_modes=(0, ks))
    P_cu, ex_cu = gpu_power(w, fft_impl=1, return_plan_info=True, debug_modes=(0, ks))
    assert ex_own["info"]["n"] == ex_cu["info"]["n"] == 1 << 24
    assert ex_own["launches"][1] == 0 and ex_cu["launches"][1] == 1      # cuFFT execs per execute
    assert np.max(np.abs(P_own - P_cu)) / P_cu.max() <= 1e-11            # same spreading, two FFTs
    assert np.max(np.abs(gpu_power(w, fft_impl=3) - P_own)) <= 1e-13     # unfused assembly: same arithmetic
    _, sums, _ = oracle.direct(w.t, w.y[0], w.dy, w.f0, w.df, w.Nf, k=ks, return_sums=True)
    for g in (ex_own["modes"], ex_cu["modes"]):
        for a, b in ((0, 1), (2, 3), (4, 5)):
            num = np.sqrt(np.sum((g[:, a] - sums[:, a]) ** 2 + (g[:, b] - sums[:, b]) ** 2))
            den = np.sqrt(np.sum(sums[:, a] ** 2 + sums[:, b] ** 2))
            assert num / den <= w.eps, (a, num / den)


@pytest.mark.parametrize("fft_impl", [0, 2])
def test_own_fft_batch_in_two_passes_at_headline_size(fft_impl):
    """Batch of 3 at n = 2^24 (own FFT, 512-cell tiles, liveness masks reused by the second pass; fft_impl 2: third
    FFT pass fused with the assembly): every series must equal its own single-series execute."""
    w = make_workload(3)
    y = np.stack([w.y[0], 2.5 * w.y[0] + 7.0, w.y[0] + np.sin(2 * np.pi * w.t / 3.3)])
    wb = Workload("cfg3_batch3", w.t, np.ascontiguousarray(y), w.dy, w.f0, w.df, w.Nf, "f64", w.eps)
    Pb, ex = gpu_power(wb, batch_chunk=2, fft_impl=fft_impl, return_plan_info=True)
    assert ex["info"]["n"] == 1 << 24 and ex["info"]["M"] == 5 and ex["launches"][1] == 0
    P0 = gpu_power(w)[0]
    assert np.max(np.abs(Pb[0] - P0)) <= 1e-12
    assert np.max(np.abs(Pb[1] - P0)) <= 1e-11           # power is invariant to scaling and shifting y
    w2 = Workload("cfg3_third", w.t, np.ascontiguousarray(y[2:3]), w.dy, w.f0, w.df, w.Nf, "f64", w.eps)
    assert np.max(np.abs(Pb[2] - gpu_power(w2)[0])) <= 1e-12
    ks = compare_indices(w, 128)
    _check64(errors(Pb[2][ks], oracle_power(w2, ks=ks)))


@pytest.mark.parametrize("p", [12, 13, 14, 15, 16, 17, 18, 19, 20, 21, 22, 23])
def test_own_fft_other_power_of_two_grids(p):
    """n = 2^p: two passes R1 x 256 (p = 12..16), three passes with a first radix of 2, 4, 8 (p = 17..19) or of
    16..128 with pruning (p = 20..23), against cuFFT on the full grid and against the oracle on sampled k."""
    rng = np.random.default_rng(400 + p)
    Nf = int(0.7 * (1 << p))
    Nd = max(200, Nf // 12)
    t = rng.uniform(0, 2000.0, Nd)
    dy = rng.uniform(0.5, 1.5, Nd)
    df = 1.0 / (5 * (t.max() - t.min()))
    kg = Nf // 3
    y = np.sin(2 * np.pi * (df + kg * df) * t + 0.4) + rng.normal(0, 1.0, Nd)
    w = _custom(t, y, dy, df, df, Nf)
    P_own, ex = gpu_power(w, fft_impl=2, no_autotune=1, return_plan_info=True)
    assert ex["info"]["n"] == 1 << p and ex["launches"][1] == 0
    P_cu = gpu_power(w, fft_impl=1, no_autotune=1)
    assert np.max(np.abs(P_own - P_cu)) / P_cu.max() <= 1e-11
    ks = np.unique(np.concatenate([compare_indices(w, 200), np.arange(kg - 3, kg + 4)]))
    _check64(errors(P_own[0][ks], oracle_power(w, ks=ks)))
    assert int(np.argmax(P_own[0])) == kg


@pytest.mark.parametrize("k", [13, 14, 15, 16])
def test_own_fft_grids_of_5_times_a_power_of_two(k):
    """n = 5 x 2^k (two passes: 80 RM x 256 with a 16 x RM x 5 first pass, RM = 2 .. 16; ls_fft_cols5_kernel), asked for
    with upsampfac: against cuFFT on the same grid (full frequency grid, a batch of 3 with the assembly fused into the last
    pass and as its own kernel) and against the oracle on sampled k."""
    n = 5 << k
    rng = np.random.default_rng(500 + k)
    Nf = int(n / 1.3107)                                 # upsampfac 1.3108 -> ceil -> next 2,3,5-smooth even size = n
    Nd = max(200, Nf // 12)
    t = rng.uniform(0, 2000.0, Nd)
    dy = rng.uniform(0.5, 1.5, Nd)
    df = 1.0 / (5 * (t.max() - t.min()))
    kg = Nf // 3
    y0 = np.sin(2 * np.pi * (df + kg * df) * t + 0.4) + rng.normal(0, 1.0, Nd)
    y = np.stack([y0, 2.0 * y0 - 1.0, y0 + np.cos(2 * np.pi * t / 11.0)])
    w = Workload(f"n5_{k}", t, np.ascontiguousarray(y), dy, df, df, Nf, "f64", 1e-9)
    up = n / Nf * (1 - 1e-9)
    P_own, ex = gpu_power(w, fft_impl=2, upsampfac=up, return_plan_info=True)
    assert ex["info"]["n"] == n and ex["launches"][1] == 0
    P_cu, exc = gpu_power(w, fft_impl=1, upsampfac=up, return_plan_info=True)
    assert exc["info"]["n"] == n and exc["launches"][1] == 1
    assert np.max(np.abs(P_own - P_cu)) / P_cu.max() <= 1e-11
    assert np.max(np.abs(gpu_power(w, fft_impl=3, upsampfac=up) - P_own)) <= 1e-13
    ks = np.unique(np.concatenate([compare_indices(w, 200), np.arange(kg - 3, kg + 4)]))
    for b in range(3):
        _check64(errors(P_own[b][ks], oracle_power(w, b=b, ks=ks)))
    assert int(np.argmax(P_own[0])) == kg


@pytest.mark.parametrize("p,batch", [(20, 1), (21, 3), (22, 1), (23, 2)])
def test_own_fft_fused_passes_match_separate_passes(p, batch):
    """n = 2^p >= 2^20, default plan: FFT passes 2 + 3 run as one persistent kernel whose intermediate stays in L2
    (tile queue, slab completion signals, L2 discard).  Same arithmetic as the three separate pass kernels
    (fft_impl = 3), so the powers must agree to rounding — also on replays (the queue resets itself) — and match the
    oracle on sampled k."""
    rng = np.random.default_rng(900 + p)
    Nf = int(0.7 * (1 << p))
    Nd = max(500, Nf // 10)
    t = rng.uniform(0, 3000.0, Nd)
    dy = rng.uniform(0.5, 1.5, Nd)
    df = 1.0 / (5 * (t.max() - t.min()))
    kg = Nf // 4
    y = np.stack([np.sin(2 * np.pi * (df + (kg + 10 * b) * df) * t + 0.3 * b) + rng.normal(0, 1.0, Nd) for b in range(batch)])
    w = Workload(f"fused23_p{p}", t, y, dy, df, df, Nf, "f64", 1e-9)
    P_f, ex = gpu_power(w, no_autotune=1, return_plan_info=True, side_stream=True, repeat=3)
    assert ex["info"]["n"] == 1 << p and ex["launches"][1] == 0
    P_s, ex_s = gpu_power(w, no_autotune=1, fft_impl=3, return_plan_info=True)
    assert ex_s["launches"][0] == ex["launches"][0] + 1                 # one launch fewer than the separate passes
    assert np.max(np.abs(P_f - P_s)) <= 1e-13                           # (the statistics' atomic sums are unordered)
    ks = np.unique(np.concatenate([compare_indices(w, 150), np.arange(kg - 3, kg + 4)]))
    for b in range(batch):
        wb = Workload(w.name, t, np.ascontiguousarray(y[b:b + 1]), dy, df, df, Nf, "f64", 1e-9)
        _check64(errors(P_f[b][ks], oracle_power(wb, ks=ks)))


def test_own_fft_per_series_dy_and_dense_points():
    """Own FFT (n = 2^20) with per-series dy (slots [w2_s ...][(w_s, h_s) ...], liveness masks of both point sets) and
    more points than a spreading chunk holds per tile (several 256-candidate chunks per tile)."""
    rng = np.random.default_rng(77)
    Nf = int(0.7 * (1 << 20)); Nd = 400_000                        # ~1.9 points per cell in the occupied fifth
    t = rng.uniform(0, 1000.0, Nd)
    df = 1.0 / (5 * (t.max() - t.min()))
    y = np.stack([np.sin(2 * np.pi * (df + 50_000 * df) * t) + rng.normal(0, 1, Nd),
                  0.5 * np.cos(2 * np.pi * (df + 300_000 * df) * t) + rng.normal(0, 1, Nd)])
    dy = rng.uniform(0.5, 1.5, (2, Nd))
    w = Workload("own_fft_per_series", t, np.ascontiguousarray(y), np.ascontiguousarray(dy), df, df, Nf, "f64", 1e-9)
    Pg, ex = gpu_power(w, no_autotune=1, return_plan_info=True)
    assert ex["info"]["n"] == 1 << 20 and ex["info"]["M"] == 6 and ex["launches"][1] == 0
    for b, kg in ((0, 50_000), (1, 300_000)):
        ks = np.unique(np.concatenate([compare_indices(w, 150), np.arange(kg - 3, kg + 4)]))
        _check64(errors(Pg[b][ks], oracle_power(w, b, ks=ks)))
        assert int(np.argmax(Pg[b])) == kg


def test_own_fft_rejected_where_unsupported():
    from gpu_util import require_cuda
    require_cuda()
    from paper_2409_08090_b200 import binding as B
    with pytest.raises(B.LsError) as ei:
        B.Plan(1000, 12500, 0.1, 0.1, 1e-5, B.LS_F32, 1, fft_impl=2)     # fp32 grid
    assert ei.value.code == 5
    with pytest.raises(B.LsError) as ei:
        B.Plan(1000, 12500, 0.1, 0.1, 1e-9, B.LS_F64, 1, fft_impl=2, upsampfac=1.5)   # n = 18750, not a power of two
    assert ei.value.code == 5
    with pytest.raises(B.LsError) as ei:
        B.Plan(100, 1000, 0.1, 0.1, 1e-9, B.LS_F64, 1, fft_impl=3)       # n = 2048 < 2^12
    assert ei.value.code == 5
    with pytest.raises(B.LsError) as ei:
        B.Plan(1000, 12500, 0.1, 0.1, 1e-9, B.LS_F64, 1, fft_impl=4)
    assert ei.value.code == 1


def test_cfg3_time_shift_invariance_full_grid():
    """A property that holds at any size (north_star: invariance of power to shifting t), on the FULL
    grid of the headline config: P(t + Delta) == P(t) up to the perturbation rounding t + Delta makes."""
    w = make_workload(3)
    P0 = gpu_power(w)[0]
    w2 = _custom(w.t + 4096.0, w.y, w.dy, w.f0, w.df, w.Nf)
    P1 = gpu_power(w2)[0]
    # fl(t + 4096) moves t by <= 2^-40 day; at f_max = 250/day that is a 2e-10-cycle phase change per point
    assert np.max(np.abs(P1 - P0)) / P0.max() <= 1e-8


def test_cfg4_scaled_batch_full_grid():
    w = scaled_workload(4, 2000, batch=37)
    Pg, ex = gpu_power(w, return_plan_info=True)
    assert ex["info"]["M"] == 39
    for b in (0, 1, 17, 36):
        _check64(errors(Pg[b], oracle_power(w, b)))


def test_cfg4_full_size_batch_1000():
    w = make_workload(4)
    Pg = gpu_power(w)
    assert Pg.shape == (1000, 125_000) and np.all(np.isfinite(Pg))
    ks = compare_indices(w, 48)[:96]
    worst = 0.0
    for b in range(w.batch):                                           # every series on a small subset
        e = errors(Pg[b][ks], oracle_power(w, b, ks=ks))
        worst = max(worst, e["Einf"])
    assert worst <= GATE_F64, worst
    ks = compare_indices(w, 1024)
    for b in (0, 333, 999):                                            # a few series on a large subset
        _check64(errors(Pg[b][ks], oracle_power(w, b, ks=ks)))
    for b in (1, 250, 500, 998):                                       # four series on the FULL grid, against
        _check64(errors(Pg[b], oracle_power(w, b, fast=True)))         # the phase-winding evaluator (pinned to direct at 1e-12)


def test_cfg5_scaled_fp32_clustered():
    w = scaled_workload(5, 100_000)
    Pg = gpu_power(w)
    ks = compare_indices(w, 2048)
    e = errors(Pg[0][ks], oracle_power(w, ks=ks))
    assert e["Einf"] <= GATE_F32, e
    assert e["median"] <= 1e-4, e


def test_zero_fill_sweep_and_tile_lists_on_the_cufft_path():
    """cuFFT path with the sweep kernel that zero-fills empty tiles and lists occupied ones (what config 5 runs at full
    size), forced at small sizes (opts.reserved[0] = 2): fp32 clustered, fp64 non-power-of-two grid, a batch in passes,
    per-series dy, a grid so small that every tile wraps; replays must agree (the lists are rebuilt per execute)."""
    w = scaled_workload(5, 100_000)
    ks = compare_indices(w, 1024)
    Pg = gpu_power(w, reserved=(2, 0), side_stream=True, repeat=2)
    e = errors(Pg[0][ks], oracle_power(w, ks=ks))
    assert e["Einf"] <= GATE_F32, e
    w2 = scaled_workload(2, 3000)
    _check64(errors(gpu_power(w2, fft_impl=1, upsampfac=1.5, reserved=(2, 0))[0], oracle_power(w2, fast=True)), pointwise=False)
    wb = scaled_workload(4, 1500, batch=7)
    P_ref = gpu_power(wb, fft_impl=1, reserved=(1, 0))
    for chunk in (0, 3):
        assert np.max(np.abs(gpu_power(wb, fft_impl=1, reserved=(2, 0), batch_chunk=chunk) - P_ref)) <= 1e-12
    wb.dy = np.ascontiguousarray(np.random.default_rng(3).uniform(0.5, 1.5, (7, wb.Nd)))
    Pp = gpu_power(wb, fft_impl=1, reserved=(2, 0), batch_chunk=2)
    for b in (0, 6):
        _check64(errors(Pp[b], oracle_power(wb, b)))
    rng = np.random.default_rng(8)
    t = rng.uniform(-50.0, 150.0, 400); y = rng.normal(0, 1, 400); dy = rng.uniform(0.5, 1.5, 400)
    ww = _custom(t, y, dy, f0=0.05, df=0.0131, Nf=700)
    _check64(errors(gpu_power(ww, fft_impl=1, reserved=(2, 0))[0], oracle_power(ww)), pointwise=False)


@pytest.mark.parametrize("k", [22, 23, 24])
def test_own_fp32_fft_grids_of_5_times_a_power_of_two(k):
    """fp32, n = 5 x 2^k (three passes 80 RM x 256 x 512, RM = 2, 4, 8; ls_fft_f32.cu; RM = 16 is config 5 itself, below):
    clustered sampling as in config 5, so that most spreading tiles are empty and the first pass prunes; against cuFFT on
    the same grid over the whole frequency grid and against the oracle on sampled k."""
    n = 5 << k
    w0 = scaled_workload(5, 150_000)
    Nf = int(n / 1.3107)
    w = _custom(w0.t, w0.y[0], w0.dy, w0.f0, w0.df, Nf, dtype="f32", eps=1e-5, name=f"f32_n5_{k}")
    w.seed, w.injected = w0.seed, w0.injected
    up = n / Nf * (1 - 1e-9)
    P_own, ex = gpu_power(w, upsampfac=up, return_plan_info=True)
    assert ex["info"]["n"] == n and ex["launches"][1] == 0
    P_cu, exc = gpu_power(w, upsampfac=up, fft_impl=1, return_plan_info=True)
    assert exc["info"]["n"] == n and exc["launches"][1] == 1
    assert np.all(np.isfinite(P_own))
    assert np.max(np.abs(P_own - P_cu)) / P_cu.max() <= 2e-5         # two fp32 FFTs of the same grids
    ks = compare_indices(w, 300)
    e = errors(P_own[0][ks], oracle_power(w, ks=ks))
    assert e["Einf"] <= GATE_F32 and e["median"] <= 1e-4, e
    assert abs(int(np.argmax(P_own[0])) - int(np.argmax(P_cu[0]))) <= 1


def test_own_fp32_fft_batches_variants_and_mode_hook():
    """The fp32 own-FFT path (n = 5 x 2^22) beyond one series: a batch of 3 with shared dy in one pass and in chunks of 2
    (pass 1 reuses the liveness masks), per-series dy (M = 6), the fixed-mean pair of transforms, and the mode debug hook
    on the compact fp32 mode array — each against the oracle on sampled k, the batch also against its single-series runs."""
    import oracle
    from oracle import variants
    n = 5 << 22
    w0 = scaled_workload(5, 60_000)
    Nf = int(n / 1.3107)
    up = n / Nf * (1 - 1e-9)
    rng = np.random.default_rng(91)
    y = np.stack([w0.y[0], 0.5 * w0.y[0] + 3.0, w0.y[0] + np.sin(2 * np.pi * w0.t / 2.7).astype(np.float32)])
    wb = _custom(w0.t, y, w0.dy, w0.f0, w0.df, Nf, dtype="f32", eps=1e-5, name="f32_n5_batch")
    wb.seed, wb.injected = w0.seed, w0.injected
    ks = compare_indices(wb, 200)
    P1, ex = gpu_power(wb, upsampfac=up, return_plan_info=True, debug_modes=(2, ks))
    assert ex["info"]["n"] == n and ex["info"]["M"] == 5 and ex["launches"][1] == 0
    P2 = gpu_power(wb, upsampfac=up, batch_chunk=2)
    assert np.max(np.abs(P1 - P2)) <= 1e-6
    for b in range(3):
        e = errors(P1[b][ks], oracle_power(wb, b=b, ks=ks))
        assert e["Einf"] <= GATE_F32 and e["median"] <= 1e-4, (b, e)
    _, sums, _ = oracle.direct(wb.t, wb.y[2], wb.dy, wb.f0, wb.df, wb.Nf, k=ks, return_sums=True)
    g = ex["modes"]
    for a, b in ((0, 1), (2, 3), (4, 5)):                              # the three type-1 transforms, fp32: <~ eps
        num = np.sqrt(np.sum((g[:, a] - sums[:, a]) ** 2 + (g[:, b] - sums[:, b]) ** 2))
        assert num / np.sqrt(np.sum(sums[:, a] ** 2 + sums[:, b] ** 2)) <= 3e-5, (a, num)
    wp = _custom(w0.t, y[:2], rng.uniform(0.5, 2.0, (2, w0.Nd)), w0.f0, w0.df, Nf, dtype="f32", eps=1e-5, name="f32_n5_per")
    Pp, exp_ = gpu_power(wp, upsampfac=up, return_plan_info=True)
    assert exp_["info"]["M"] == 6 and exp_["launches"][1] == 0
    for b in range(2):
        Po = oracle.direct(wp.t, wp.y[b], wp.dy[b], wp.f0, wp.df, wp.Nf, k=ks)
        assert np.max(np.abs(Pp[b][ks] - Po)) / Po.max() <= GATE_F32, b
    Pf, exf = gpu_power(wb, upsampfac=up, no_floating_mean=1, return_plan_info=True)
    assert exf["info"]["M"] == 4 and exf["launches"][1] == 0
    Pc = gpu_power(wb, upsampfac=up, no_floating_mean=1, fft_impl=1)   # same variant through cuFFT on the same grid
    assert np.max(np.abs(Pf - Pc)) / Pc.max() <= 2e-5
    Po = variants.power(wb.t, wb.y[1], wb.dy, wb.f0, wb.df, wb.Nf, k=ks, fit_mean=False)
    assert np.max(np.abs(Pf[1][ks] - Po)) / Po.max() <= GATE_F32


def test_cfg5_full_size_fp32_sampled_frequencies():
    w = make_workload(5)
    Pg, ex = gpu_power(w, return_plan_info=True)
    assert ex["info"]["n"] == 5 << 25 and ex["launches"][1] == 0       # the own fp32 transform (RM = 16), no cuFFT
    assert np.all(np.isfinite(Pg))
    ks = compare_indices(w, 256)                                       # K = 256 at config 5
    e = errors(Pg[0][ks], oracle_power(w, ks=ks))
    assert e["Einf"] <= GATE_F32, e
    assert e["median"] <= 1e-4, e


# ------------------------------------------------------------------ stage pins (debug exports)
def test_stats_and_nufft_contract():
    """K1 against the oracle's statistics; the three type-1 transforms against the oracle's direct
    sums: ||g~ - g||_2 / ||g||_2 <~ eps."""
    import oracle
    w = make_workload(2)
    ks = compare_indices(w, 1500)
    Pg, ex = gpu_power(w, return_plan_info=True, debug_modes=(0, ks))
    W, ybar, YY = oracle.stats(w.y[0], w.dy)
    assert abs(ex["stats"][0, 0] - W) <= 1e-12 * W
    assert abs(ex["stats"][0, 1] - ybar) <= 1e-13
    assert abs(ex["stats"][0, 2] - YY) <= 1e-12 * YY
    _, sums, _ = oracle.direct(w.t, w.y[0], w.dy, w.f0, w.df, w.Nf, k=ks, return_sums=True)
    g = ex["modes"]
    for a, b in ((0, 1), (2, 3), (4, 5)):                              # (Sh,Ch), (S,C), (S2,C2)
        num = np.sqrt(np.sum((g[:, a] - sums[:, a]) ** 2 + (g[:, b] - sums[:, b]) ** 2))
        den = np.sqrt(np.sum(sums[:, a] ** 2 + sums[:, b] ** 2))
        assert num / den <= w.eps, (a, num / den)


# ------------------------------------------------------------------ options and layouts
@pytest.mark.parametrize("opts", [dict(tile_cells=256), dict(tile_cells=512), dict(kernel_width=10),
                                  dict(upsampfac=1.25), dict(kernel_width=16, upsampfac=1.25)])
def test_plan_options(opts):
    w = scaled_workload(2, 3000)
    Pg = gpu_power(w, **opts)
    e = errors(Pg[0], oracle_power(w, fast=True))
    _check64(e, pointwise=False)


@pytest.mark.parametrize("tile", [256, 512, 1024])
@pytest.mark.parametrize("p", [15, 20])
def test_every_accepted_tile_length(tile, p):
    """every tile_cells the plan accepts has an instantiated kernel, on the cuFFT path (forced), the small
    own FFT (n = 2^15) and the pruned own FFT (n = 2^20: a pass-1 tile of 128 columns lies inside ONE spreading tile)."""
    rng = np.random.default_rng(50 + p)
    Nf = int(0.7 * (1 << p)); Nd = max(300, Nf // 10)
    t = rng.uniform(0, 900.0, Nd); dy = rng.uniform(0.5, 1.5, Nd)
    df = 1.0 / (5 * (t.max() - t.min()))
    y = np.sin(2 * np.pi * (df + (Nf // 3) * df) * t) + rng.normal(0, 1.0, Nd)
    w = _custom(t, y, dy, df, df, Nf)
    ks = compare_indices(w, 300)
    Po = oracle_power(w, ks=ks)
    for fft_impl in (0, 1):
        Pg, ex = gpu_power(w, tile_cells=tile, no_autotune=1, fft_impl=fft_impl, return_plan_info=True)
        assert ex["info"]["n"] == 1 << p
        _check64(errors(Pg[0][ks], Po))
    wb = Workload("tiles_batch", t, np.stack([y, 2 * y + 1]), dy, df, df, Nf, "f64", 1e-9)
    if tile <= 512:
        Pb = gpu_power(wb, tile_cells=tile, no_autotune=1)
        assert np.max(np.abs(Pb[0][ks] - Po)) / Po.max() <= GATE_F64


def test_rejected_tile_lengths_and_widths():
    from gpu_util import require_cuda
    require_cuda()
    from paper_2409_08090_b200 import binding as B
    for bad in (64, 128, 320, 768, 2048):
        with pytest.raises(B.LsError) as ei:
            B.Plan(1000, 12500, 0.1, 0.1, 1e-9, B.LS_F64, 1, tile_cells=bad)
        assert ei.value.code == 1, bad
    with pytest.raises(B.LsError) as ei:
        B.Plan(1000, 12500, 0.1, 0.1, 1e-9, B.LS_F64, 2, tile_cells=1024)      # a batch has two cells per thread
    assert ei.value.code == 1
    # eps = 1e-13 at sigma = 1.25 needs more than the 20 cells the kernels hold: refused, not silently clamped ...
    with pytest.raises(B.LsError) as ei:
        B.Plan(1000, 12500, 0.1, 0.1, 1e-13, B.LS_F64, 1, upsampfac=1.25)
    assert ei.value.code == 5
    # ... and in automatic mode the grid doubles instead (Nf = 12 500: 2^14 has sigma 1.31, needs 25 cells)
    with B.Plan(1000, 12500, 0.1, 0.1, 1e-13, B.LS_F64, 1) as plan:
        assert plan.info["n"] == 1 << 15 and plan.info["w"] <= 20


def test_batch_chunking_matches_single_pass():
    w = scaled_workload(4, 1500, batch=11)
    P_one = gpu_power(w, batch_chunk=11)
    for chunk in (1, 3, 4, 10):
        P_c = gpu_power(w, batch_chunk=chunk)
        assert np.max(np.abs(P_c - P_one)) <= 1e-12
    for b in (0, 10):
        _check64(errors(P_one[b], oracle_power(w, b)))


def test_per_series_dy():
    w = scaled_workload(4, 1200, batch=5)
    rng = np.random.default_rng(7)
    w.dy = np.ascontiguousarray(rng.uniform(0.5, 1.5, (5, w.Nd)))
    for chunk in (0, 2):
        Pg = gpu_power(w, batch_chunk=chunk)
        for b in range(5):
            _check64(errors(Pg[b], oracle_power(w, b)))


def test_caller_owned_workspace():
    """ls_set_workspace: grids, mode array and FFT work area inside a torch allocation; same results."""
    import torch
    from paper_2409_08090_b200 import binding as B
    w = scaled_workload(2, 3000)
    P_ref = gpu_power(w)
    dev = torch.device("cuda:0")
    t = torch.from_numpy(w.t).to(dev); y = torch.from_numpy(w.y).to(dev); dy = torch.from_numpy(w.dy).to(dev)
    P = torch.empty((1, w.Nf), dtype=torch.float64, device=dev)
    with B.Plan(w.Nd, w.Nf, w.f0, w.df, w.eps, B.LS_F64, 1) as plan:
        nbytes = plan.workspace_bytes()
        ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=dev)
        off = (-ws.data_ptr()) % 256
        with pytest.raises(B.LsError):
            plan.set_workspace(ws.data_ptr() + off, nbytes // 2)         # too small
        with pytest.raises(B.LsError):
            plan.set_workspace(ws.data_ptr() + off + 8, nbytes)          # misaligned
        plan.set_workspace(ws.data_ptr() + off, nbytes)
        plan.execute(t, y, dy, P, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
    assert np.max(np.abs(P.cpu().numpy() - P_ref)) <= 1e-13


def test_execute_host_matches_device():
    w = scaled_workload(2, 2500)
    Pd = gpu_power(w)
    Ph = gpu_power(w, host=True)
    assert np.max(np.abs(Pd - Ph)) <= 1e-12
    w5 = scaled_workload(5, 30_000)
    assert np.max(np.abs(gpu_power(w5) - gpu_power(w5, host=True))) <= 1e-5


def test_execute_host_overlapped_copy_out():
    """Outputs of >= 8 MB leave the device piece by piece on a second stream while the next piece is computed
    (ls.h, ls_execute_host): a long single series in frequency quarters (own FFT), and a batch pass by pass
    (shared and per-series dy, batch_chunk forcing several passes with a ragged last one).  The kernels are the
    device path's: same numbers — bit for bit where no atomics' order is involved in the sums."""
    w = scaled_workload(3, 400_000)                     # Nf = 5e6: four assembly launches of 1.25e6 frequencies
    assert w.Nf * 8 >= 8 << 20 and w.Nf >= 1 << 22
    Pd, Ph = gpu_power(w), gpu_power(w, host=True)
    assert np.all(np.isfinite(Ph)) and np.max(np.abs(Pd - Ph)) <= 1e-11
    wb = scaled_workload(4, 4000, batch=23)             # 23 x 50 000 x 8 B = 9.2 MB
    assert wb.batch * wb.Nf * 8 >= 8 << 20
    Pd = gpu_power(wb, batch_chunk=5)
    Ph = gpu_power(wb, host=True, batch_chunk=5)        # 5 passes, the last of 3 series
    assert np.all(np.isfinite(Ph)) and np.max(np.abs(Pd - Ph)) <= 1e-11
    rng = np.random.default_rng(3)
    wp = Workload(wb.name, wb.t, wb.y, rng.uniform(0.5, 1.5, wb.y.shape), wb.f0, wb.df, wb.Nf, "f64", wb.eps)
    assert np.max(np.abs(gpu_power(wp, batch_chunk=7) - gpu_power(wp, host=True, batch_chunk=7))) <= 1e-11


def test_graph_replay_matches_direct_launches():
    """opts.graph = 2 on a side stream: capture once, replay, re-capture when a buffer changes; identical
    to direct launches (graph = 1)."""
    w = scaled_workload(2, 3000)
    P_direct = gpu_power(w, graph=1, side_stream=True)
    P_graph = gpu_power(w, graph=2, side_stream=True, repeat=3)
    assert np.max(np.abs(P_graph - P_direct)) <= 1e-13
    P_auto_legacy = gpu_power(w)                       # auto mode on the legacy default stream: direct launches
    assert np.max(np.abs(P_auto_legacy - P_direct)) <= 1e-13
    _check64(errors(P_graph[0], oracle_power(w, fast=True)), pointwise=False)
    wb = scaled_workload(4, 1200, batch=5)              # batch path through a graph
    assert np.max(np.abs(gpu_power(wb, graph=2, side_stream=True, repeat=2) - gpu_power(wb, graph=1))) <= 1e-13


def test_autotuned_grid_size():
    """N_f just above a power of two / 1.6: the plan times candidate grid sizes and may take a
    non-power-of-two n; whatever it takes must meet the gate, and no_autotune must give the power of two."""
    rng = np.random.default_rng(77)
    Nd, Nf = 20_000, 650_000                            # 1.25 Nf = 812 500 -> 2^20 has sigma 1.61
    t = rng.uniform(0, 500, Nd)
    dy = rng.uniform(0.5, 1.5, Nd)
    df = 1.0 / (5 * (t.max() - t.min()))
    y = np.sin(2 * np.pi * 40000.3 * df * t) + rng.normal(0, 0.5, Nd)
    w = _custom(t, y, dy, df, df, Nf)
    ks = np.unique(np.concatenate([compare_indices(w, 600), np.arange(39990, 40010)]))   # incl. the peak
    Po = oracle_power(w, ks=ks)
    Pa, exa = gpu_power(w, return_plan_info=True)
    Pp, exp_ = gpu_power(w, return_plan_info=True, no_autotune=1)
    assert exp_["info"]["n"] == 1 << 20
    assert 1.25 * Nf <= exa["info"]["n"] <= 1 << 20 and exa["info"]["n"] % 4 == 0
    _check64(errors(Pa[0][ks], Po))
    _check64(errors(Pp[0][ks], Po))


def test_repeat_execute_is_stable():
    """Tile-owner spreading uses no floating-point atomics on the grid: repeated executes of one plan
    agree to rounding of the (atomic) statistics sums."""
    w = scaled_workload(3, 20_000)
    a = gpu_power(w)
    b = gpu_power(w)
    assert np.max(np.abs(a - b)) <= 1e-13


# ------------------------------------------------------------------ edge cases
def test_periodic_wrap_when_points_exceed_the_period():
    """df*T > 1/2: the x2 = 2 x1 point set (and here x1 too) wraps around the periodic fine grid (A6)."""
    rng = np.random.default_rng(3)
    Nd, Nf = 400, 700
    t = rng.uniform(-50.0, 150.0, Nd)
    y = np.sin(2 * np.pi * 0.31 * t) + rng.normal(0, 0.2, Nd)
    dy = rng.uniform(0.5, 1.5, Nd)
    w = _custom(t, y, dy, f0=0.05, df=0.0131, Nf=Nf)                   # df*T = 2.6 periods
    _check64(errors(gpu_power(w)[0], oracle_power(w)), pointwise=False)


@pytest.mark.parametrize("Nf", [1, 2, 3, 17, 1001])
def test_small_and_odd_Nf(Nf):
    rng = np.random.default_rng(100 + Nf)
    Nd = 50
    t = np.sort(rng.uniform(0, 20, Nd)); y = rng.normal(0, 1, Nd); dy = rng.uniform(0.5, 1.5, Nd)
    w = _custom(t, y, dy, f0=0.02, df=0.011, Nf=Nf)
    _check64(errors(gpu_power(w)[0], oracle_power(w)), pointwise=False)


def _sums_close(w, tol):
    """The three transforms themselves (well-conditioned even when the power is not), against the
    NUFFT contract |g~_k - g_k| <= tol * sum_j |c_j| (eps is relative to the strengths)."""
    import oracle
    ks = np.arange(w.Nf)
    _, ex = gpu_power(w, debug_modes=(0, ks))
    _, sums, _ = oracle.direct(w.t, w.y[0], w.dy, w.f0, w.df, w.Nf, return_sums=True)
    wn = w.dy.astype(np.float64) ** -2.0
    wn /= wn.sum()
    l1_h = np.sum(np.abs(wn * (w.y[0] - np.sum(wn * w.y[0]))))           # sum |h_j|; sum |w_j| = 1
    scale = np.array([l1_h, l1_h, 1.0, 1.0, 1.0, 1.0])
    assert np.max(np.abs(ex["modes"] - sums) / scale) <= tol


@pytest.mark.parametrize("Nd", [3, 4, 33, 257])
def test_tiny_Nd(Nd):
    rng = np.random.default_rng(Nd)
    t = rng.uniform(0, 10, Nd); y = rng.normal(0, 1, Nd); dy = rng.uniform(0.5, 1.5, Nd)
    w = _custom(t, y, dy, f0=0.013, df=0.017, Nf=200)
    Pg, Po = gpu_power(w)[0], oracle_power(w)
    _sums_close(w, 1e-9)
    if Nd == 3:
        # 3 points, 3 parameters: the model interpolates, P = 1; CC, SS are differences of O(1) numbers
        # that nearly cancel, which amplifies the NUFFT's 1e-12 error in the sums (ill-conditioned)
        good = np.abs(Po - 1) < 1e-9
        assert good.sum() > 100 and np.max(np.abs(Pg[good] - 1)) < 1e-4
        assert np.median(np.abs(Pg[good] - 1)) < 1e-8
    elif Nd == 4:
        # one degree of freedom left: still close to singular at some frequencies
        assert np.max(np.abs(Pg - Po)) <= 1e-6 and np.median(np.abs(Pg - Po)) <= 1e-9
    else:
        assert np.max(np.abs(Pg - Po)) <= 1e-8


def test_all_points_in_one_cell_and_duplicates():
    """Degenerate clustering: every point inside one fine-grid cell (one sort bin takes everything).
    All phases coincide to 1e-9 cycle, so CC*SS - CS^2 -> 0 and the POWER is ill-conditioned at any
    precision; what the kernels must get right here are the transforms, which are compared tightly."""
    rng = np.random.default_rng(9)
    Nd = 5000
    t = 100.0 + rng.uniform(0, 1e-7, Nd)
    t[::7] = t[0]                                                     # exact duplicates
    y = rng.normal(0, 1, Nd); dy = rng.uniform(0.5, 1.5, Nd)
    w = _custom(t, y, dy, f0=0.01, df=0.01, Nf=300)
    Pg = gpu_power(w)[0]
    assert np.all(np.isfinite(Pg))
    _sums_close(w, 1e-9)


def test_f0_zero_convention():
    """f0 = 0: k = 0 is the zero frequency, where the sine term vanishes (reading A14: that term is
    dropped, P = 0 — parity unpinned for that one value); every k >= 1 must match the oracle."""
    rng = np.random.default_rng(12)
    Nd = 300
    t = rng.uniform(0, 50, Nd); y = rng.normal(1.0, 1, Nd); dy = rng.uniform(0.5, 1.5, Nd)
    w = _custom(t, y, dy, f0=0.0, df=0.004, Nf=900)
    Pg, Po = gpu_power(w)[0], oracle_power(w)
    assert np.max(np.abs(Pg[1:] - Po[1:])) / Po[1:].max() <= GATE_F64
    assert np.isfinite(Pg[0]) and abs(Pg[0]) <= 1e-6


def test_noiseless_sinusoid_peaks_at_one():
    rng = np.random.default_rng(41)
    Nd, Nf = 3000, 20000
    t = rng.uniform(0, 200, Nd); dy = rng.uniform(0.5, 1.5, Nd)
    df = 1.0 / (5 * (t.max() - t.min())); kg = 7777
    y = 3.1 + 1.3 * np.sin(2 * np.pi * (df + kg * df) * t + 0.9)
    Pg = gpu_power(_custom(t, y, dy, df, df, Nf))[0]
    assert int(np.argmax(Pg)) == kg and abs(1.0 - Pg[kg]) <= 1e-8


def test_dy_scale_invariance():
    w = scaled_workload(2, 4000)
    P0 = gpu_power(w)[0]
    w2 = _custom(w.t, w.y, 4.0 * w.dy, w.f0, w.df, w.Nf)
    assert np.max(np.abs(gpu_power(w2)[0] - P0)) <= 1e-12


def test_invalid_arguments_are_rejected():
    from gpu_util import require_cuda
    require_cuda()
    from paper_2409_08090_b200 import binding as B
    bad = [dict(Nd=0), dict(Nf=0), dict(df=0.0), dict(df=float("nan")), dict(f0=-1.0), dict(eps=1e-16),
           dict(eps=0.5), dict(dtype=7), dict(batch=0)]
    base = dict(Nd=100, Nf=1000, f0=0.1, df=0.1, eps=1e-9, dtype=B.LS_F64, batch=1)
    for b in bad:
        kw = dict(base, **b)
        with pytest.raises(B.LsError) as ei:
            B.ls_plan(**kw)
        assert ei.value.code == 1, (b, ei.value.code)
    with pytest.raises(B.LsError) as ei:
        B.ls_plan(100, 1000, 0.1, 0.1, 1e-7, B.LS_F32, 1)              # eps below the fp32 floor
    assert ei.value.code == 1
    with pytest.raises(B.LsError) as ei:
        B.ls_plan(100, 2_000_000_000, 0.1, 0.1, 1e-9, B.LS_F64, 1)     # n >= 2^31
    assert ei.value.code == 5
    h = B.ls_plan(**base)
    with pytest.raises(B.LsError):
        B.ls_execute(h, 0, 0, 0, 0, 0)                                 # NULL buffers
    with pytest.raises(B.LsError) as ei:
        B.ls_get_stage_ms(h)                                           # timing not enabled
    assert ei.value.code == 6
    B.ls_destroy(h)
    B.ls_destroy(None)                                                 # NULL accepted


def test_times_given_in_float32():
    """opts.t_is_dtype on an fp32 plan: t is float[Nd], promoted exactly on the device; the oracle gets the same
    rounded times."""
    import torch
    from paper_2409_08090_b200 import binding as B
    w = scaled_workload(5, 20_000)
    tf = w.t.astype(np.float32)
    w32 = Workload(w.name + "_t32", tf.astype(np.float64), w.y, w.dy, w.f0, w.df, w.Nf, "f32", w.eps)
    dev = torch.device("cuda:0")
    P = torch.empty((1, w.Nf), dtype=torch.float32, device=dev)
    with B.Plan(w.Nd, w.Nf, w.f0, w.df, w.eps, B.LS_F32, 1, t_is_dtype=1) as plan:
        plan.execute(torch.from_numpy(tf).to(dev), torch.from_numpy(w.y).to(dev), torch.from_numpy(w.dy).to(dev), P,
                     torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
    Pg = P.cpu().numpy()[0].astype(np.float64)
    assert np.max(np.abs(Pg - gpu_power(w32)[0])) <= 1e-6             # same as handing the promoted doubles
    ks = compare_indices(w32, 1024)
    e = errors(Pg[ks], oracle_power(w32, ks=ks))
    assert e["Einf"] <= GATE_F32, e
