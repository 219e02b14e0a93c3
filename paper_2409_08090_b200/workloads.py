"""Seeded synthetic workloads (the five BASELINE.json configs) — input generation ONLY.

This module is shared by the CPU oracle's tests and by the CUDA path's tests / bench, and
therefore holds none of the method's arithmetic: it draws times, values and uncertainties,
and derives the frequency grid (f0, df, N_f) exactly as BASELINE.json `configs` states it
("astropy-style grid: df = 1/(5T), T = max t - min t, f0 = df, N_f = round(12.5 N_d)").
It imports numpy only (no torch, no oracle, no CUDA binding).

Recipe: SURVEY.md §8(d) table "Synthetic inputs" (seed, draw order, derived quantities);
the paper's own workload is synthetic too (§2 "a double-precision time series
with N_d in [1e2, 1e6]" and "the default Astropy N_f ~ 12 N_d").

All draws are made in fp64 with numpy `default_rng(seed)` (PCG64) in the order listed in each
builder; `y` and `dy` are cast to the config's dtype afterwards; `t` always stays fp64
(reading A9).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

__all__ = ["Workload", "make_workload", "scaled_workload", "CONFIG_NAMES", "compare_indices"]

CONFIG_NAMES = {
    1: "cfg1_single_Nd1e3_f64",
    2: "cfg2_single_Nd1e4_f64",
    3: "cfg3_single_Nd1e6_f64",
    4: "cfg4_batch1000_Nd1e4_f64",
    5: "cfg5_clustered_Nd1e7_f32",
}

_SEEDS = {1: 24090801, 2: 24090802, 3: 24090803, 4: 24090804, 5: 24090805}


@dataclass
class Workload:
    """One problem instance handed unchanged to both the oracle and the CUDA path."""

    name: str
    t: np.ndarray            # [Nd] float64
    y: np.ndarray            # [batch, Nd] dtype
    dy: np.ndarray           # [Nd] dtype (shared by the batch)
    f0: float
    df: float
    Nf: int
    dtype: str               # "f64" | "f32"
    eps: float
    injected: list = field(default_factory=list)   # injected signal frequencies (cycles/day)
    seed: int = 0

    @property
    def Nd(self) -> int:
        return int(self.t.shape[0])

    @property
    def batch(self) -> int:
        return int(self.y.shape[0])

    @property
    def np_dtype(self):
        return np.float64 if self.dtype == "f64" else np.float32


def _grid(t: np.ndarray, Nd: int):
    """df = 1/(5T), f0 = df, Nf = round(12.5 Nd)   (BASELINE.json configs)."""
    T = float(t.max() - t.min())
    df = 1.0 / (5.0 * T)
    return df, df, int(round(12.5 * Nd))


def _cfg1(Nd=1000, seed=_SEEDS[1]):
    rng = np.random.default_rng(seed)
    t = np.sort(rng.uniform(0.0, 1000.0, Nd))
    noise = rng.normal(0.0, 0.3, Nd)
    dy = rng.uniform(0.5, 1.5, Nd)
    y = np.sin(2 * np.pi * t / 7.3) + noise
    f0, df, Nf = _grid(t, Nd)
    return Workload(CONFIG_NAMES[1], t, y[None, :], dy, f0, df, Nf, "f64", 1e-9, [1 / 7.3], seed)


def _cfg2(Nd=10_000, seed=_SEEDS[2]):
    rng = np.random.default_rng(seed)
    phi = rng.uniform(0.0, 2 * np.pi)
    t = rng.uniform(0.0, 3650.0, Nd)
    noise = rng.normal(0.0, 0.5, Nd)
    dy = rng.uniform(0.2, 1.0, Nd)
    y = 0.8 * np.sin(2 * np.pi * t / 23.1 + phi) + noise
    f0, df, Nf = _grid(t, Nd)
    return Workload(CONFIG_NAMES[2], t, y[None, :], dy, f0, df, Nf, "f64", 1e-9, [1 / 23.1], seed)


def _cfg3(Nd=1_000_000, seed=_SEEDS[3]):
    rng = np.random.default_rng(seed)
    t = rng.uniform(0.0, 1.0e4, Nd)
    noise = rng.normal(0.0, 1.0, Nd)
    dy = rng.uniform(0.5, 1.5, Nd)
    y = np.sin(2 * np.pi * t / 1.7) + noise
    f0, df, Nf = _grid(t, Nd)
    return Workload(CONFIG_NAMES[3], t, y[None, :], dy, f0, df, Nf, "f64", 1e-9, [1 / 1.7], seed)


def _cfg4(Nd=10_000, batch=1000, seed=_SEEDS[4]):
    rng = np.random.default_rng(seed)
    t = rng.uniform(0.0, 3650.0, Nd)
    dy = rng.uniform(0.5, 1.5, Nd)
    y = np.empty((batch, Nd), dtype=np.float64)
    inj = []
    for b in range(batch):
        A = rng.uniform(0.0, 2.0)
        P = float(np.exp(rng.uniform(np.log(0.5), np.log(500.0))))
        phi = rng.uniform(0.0, 2 * np.pi)
        noise = rng.normal(0.0, 1.0, Nd)
        y[b] = A * np.sin(2 * np.pi * t / P + phi) + noise
        inj.append(1.0 / P)
    f0, df, Nf = _grid(t, Nd)
    return Workload(CONFIG_NAMES[4], t, y, dy, f0, df, Nf, "f64", 1e-9, inj, seed)


def _cfg5(Nd=10_000_000, n_nights=3650, seed=_SEEDS[5]):
    """Strongly clustered sampling: nightly 0.3-day windows over n_nights days,
    nights with (index mod 365) >= 219 dropped (contiguous 40 % seasonal gap), per-night
    counts ~ Multinomial(Nd; equal p) (= independent Poissons conditioned on the total)."""
    rng = np.random.default_rng(seed)
    nights = np.arange(n_nights)
    kept = nights[(nights % 365) < 219]
    counts = rng.multinomial(Nd, np.full(kept.size, 1.0 / kept.size))
    t = np.repeat(kept.astype(np.float64), counts) + rng.uniform(0.0, 0.3, Nd)
    noise = rng.normal(0.0, 1.0, Nd)
    dy = rng.uniform(0.5, 2.0, Nd)
    y = np.sin(2 * np.pi * t / 0.9137) + 0.3 * np.sin(2 * np.pi * t / 365.25) + noise
    f0, df, Nf = _grid(t, Nd)
    return Workload(CONFIG_NAMES[5], t, y.astype(np.float32)[None, :], dy.astype(np.float32),
                    f0, df, Nf, "f32", 1e-5, [1 / 0.9137, 1 / 365.25], seed)


_BUILDERS = {1: _cfg1, 2: _cfg2, 3: _cfg3, 4: _cfg4, 5: _cfg5}


def make_workload(cfg: int) -> Workload:
    """Full-size BASELINE.json config `cfg` (1..5)."""
    return _BUILDERS[cfg]()


def scaled_workload(cfg: int, Nd: int, batch: int | None = None, seed: int | None = None) -> Workload:
    """Same recipe as config `cfg` at a different N_d (and batch): used for parity cases the
    oracle finishes in seconds.  The time span is kept, so the point density changes."""
    kw = {"Nd": Nd}
    if seed is not None:
        kw["seed"] = seed
    if cfg == 4 and batch is not None:
        kw["batch"] = batch
    w = _BUILDERS[cfg](**kw)
    w.name = f"{w.name}@Nd{Nd}" + (f"xB{w.batch}" if cfg == 4 else "")
    return w


def compare_indices(w: Workload, K: int, seed_offset: int = 1000) -> np.ndarray:
    """Frequency indices on which configs too large for a full-grid direct evaluation are compared
    (SURVEY §8(d) "Compared frequencies"): K seeded random k, plus always k in {0,1,2}, the
    mode-wrap seam floor(Nf/2)-1..+1, {Nf-2, Nf-1}, and +-3 bins around each injected frequency
    (at most the first 8 injected ones), so that max_k P over the subset is the true peak."""
    Nf = w.Nf
    rng = np.random.default_rng(w.seed + seed_offset)
    ks = set(int(k) for k in rng.integers(0, Nf, size=min(K, Nf)))
    fixed = [0, 1, 2, Nf // 2 - 1, Nf // 2, Nf // 2 + 1, Nf - 2, Nf - 1]
    for fi in w.injected[:8]:
        kc = int(round((fi - w.f0) / w.df))
        fixed.extend(range(kc - 3, kc + 4))
    ks.update(k for k in fixed if 0 <= k < Nf)
    return np.array(sorted(ks), dtype=np.int64)
