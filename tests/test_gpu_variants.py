"""-m gpu parity of the periodogram variants (fixed mean = the "four sums" of PAPER.md:17, and the
normalisations of the Astropy interface) against oracle/variants.py, on the cuFFT path, on the own-FFT
path with the fused last pass, and for a batch."""
import numpy as np
import pytest

from gpu_util import gpu_power
from oracle import variants
from paper_2409_08090_b200.workloads import Workload, compare_indices, scaled_workload

pytestmark = pytest.mark.gpu
NORM = {"standard": 0, "model": 1, "log": 2, "psd": 3}


def _rel(Pg, Po):
    return float(np.max(np.abs(Pg - Po)) / np.max(np.abs(Po)))


@pytest.mark.parametrize("fit_mean", [True, False])
@pytest.mark.parametrize("norm", ["standard", "model", "log", "psd"])
def test_variants_small_grid_cufft_path(fit_mean, norm):
    w = scaled_workload(2, 3000)
    Pg = gpu_power(w, no_floating_mean=0 if fit_mean else 1, normalization=NORM[norm])[0]
    Po = variants.power(w.t, w.y[0], w.dy, w.f0, w.df, w.Nf, fit_mean=fit_mean, normalization=norm)
    assert _rel(Pg, Po) <= 1e-8, (fit_mean, norm, _rel(Pg, Po))


@pytest.mark.parametrize("fit_mean,norm,fft_impl", [(False, "standard", 2), (False, "psd", 0), (True, "log", 2)])
def test_variants_own_fft_paths(fit_mean, norm, fft_impl):
    rng = np.random.default_rng(90)
    Nf = int(0.7 * (1 << 20)); Nd = Nf // 12
    t = rng.uniform(0, 800.0, Nd); dy = rng.uniform(0.5, 1.5, Nd)
    df = 1.0 / (5 * (t.max() - t.min()))
    y = 5.0 + np.sin(2 * np.pi * (df + 40000 * df) * t) + rng.normal(0, 1.0, Nd)
    w = Workload("variants_p20", t, np.ascontiguousarray(y[None]), dy, df, df, Nf, "f64", 1e-9)
    Pg, ex = gpu_power(w, no_autotune=1, no_floating_mean=0 if fit_mean else 1, normalization=NORM[norm],
                       fft_impl=fft_impl, return_plan_info=True)
    assert ex["launches"][1] == 0                                   # own FFT, no cuFFT exec
    ks = np.unique(np.concatenate([compare_indices(w, 300), np.arange(39995, 40006)]))
    Po = variants.power(w.t, w.y[0], w.dy, w.f0, w.df, w.Nf, k=ks, fit_mean=fit_mean, normalization=norm)
    assert _rel(Pg[0][ks], Po) <= 1e-8


def test_variants_batch_shared_and_per_series_dy():
    w = scaled_workload(4, 1500, batch=6)
    for per in (False, True):
        if per:
            w.dy = np.ascontiguousarray(np.random.default_rng(5).uniform(0.5, 1.5, (6, w.Nd)))
        Pg = gpu_power(w, no_floating_mean=1, normalization=NORM["model"])
        for b in (0, 5):
            dyb = w.dy[b] if per else w.dy
            Po = variants.power(w.t, w.y[b], dyb, w.f0, w.df, w.Nf, fit_mean=False, normalization="model")
            assert _rel(Pg[b], Po) <= 1e-8, (per, b)


def test_fixed_mean_is_a_pair_of_transforms():
    """opts.no_floating_mean runs the paper's "pair of NUFFTs": w at x2 and h at x1 — the w transform at
    x1 is neither spread nor transformed (M = batch + 1 with shared dy, 2 batch with per-series dy); batch passes,
    the fused last pass and the mode debug hook keep working on the shorter slot layout."""
    import oracle
    w = scaled_workload(4, 1500, batch=5)
    for chunk in (0, 2):
        Pg, ex = gpu_power(w, no_floating_mean=1, batch_chunk=chunk, return_plan_info=True,
                           debug_modes=(3, np.arange(0, w.Nf, 7)) if chunk == 0 else None)
        assert ex["info"]["M"] == 6
        for b in (0, 3, 4):
            Po = variants.power(w.t, w.y[b], w.dy, w.f0, w.df, w.Nf, fit_mean=False)
            assert _rel(Pg[b], Po) <= 1e-8, (chunk, b)
        if chunk == 0:
            _, sums, _ = oracle.direct(w.t, w.y[3], w.dy, w.f0, w.df, w.Nf, k=np.arange(0, w.Nf, 7), return_sums=True)
            g = ex["modes"]
            assert np.max(np.abs(g[:, [0, 1, 4, 5]] - sums[:, [0, 1, 4, 5]])) <= 1e-9       # (Sh, Ch) and (S2, C2)
    wp = scaled_workload(4, 1500, batch=3)
    wp.dy = np.ascontiguousarray(np.random.default_rng(6).uniform(0.5, 1.5, (3, wp.Nd)))
    Pg, ex = gpu_power(wp, no_floating_mean=1, return_plan_info=True)
    assert ex["info"]["M"] == 6
    for b in range(3):
        assert _rel(Pg[b], variants.power(wp.t, wp.y[b], wp.dy[b], wp.f0, wp.df, wp.Nf, fit_mean=False)) <= 1e-8
    assert gpu_power(scaled_workload(2, 2000), no_floating_mean=1, return_plan_info=True)[1]["info"]["M"] == 2


def test_astropy_style_front_end():
    import torch
    from paper_2409_08090_b200.lombscargle import LombScargle
    w = scaled_workload(2, 2000)
    ls = LombScargle(w.t, w.y[0], w.dy, fit_mean=False, normalization="psd")
    f0, df, Nf = ls.autofrequency(samples_per_peak=5, nyquist_factor=3)
    T = w.t.max() - w.t.min()
    assert df == pytest.approx(1 / (5 * T)) and f0 == pytest.approx(df / 2) and Nf > 1000
    freq, P = ls.autopower(samples_per_peak=5, nyquist_factor=3)
    torch.cuda.synchronize()
    assert P.shape == (Nf,) and freq.shape == (Nf,) and float(freq[1] - freq[0]) == pytest.approx(df)
    Po = variants.power(w.t, w.y[0], w.dy, f0, df, Nf, fit_mean=False, normalization="psd")
    assert _rel(P.cpu().numpy(), Po) <= 1e-8
    P2 = ls.power_grid(w.f0, w.df, w.Nf)                           # explicit grid, replaces the cached plan
    torch.cuda.synchronize()
    assert _rel(P2.cpu().numpy(), variants.power(w.t, w.y[0], w.dy, w.f0, w.df, w.Nf, fit_mean=False,
                                                 normalization="psd")) <= 1e-8
    ls.close()
    with pytest.raises(ValueError):
        LombScargle(w.t, w.y[0], w.dy, normalization="nope")
