"""Pins for the CPU oracle (oracle/ls_oracle.c) against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each pin is chosen so that a plausible mistake in the
oracle (dropped term, wrong sign or index, transposed operand, lost phase precision) fails it:
  worked example (golden, 50 digits) .......... every step O1..O6, end to end
  mpmath brute force, N_d <= 64 ............... Eq. 1 sums incl. huge time offsets
  scipy.signal.lombscargle .................... independent library implementation
  chi2 definition vs tau formulas ............. assembly, floating mean
  equispaced t -> DFT, Parseval ............... Eq. 1 reduces to an exact DFT
  noiseless sinusoid -> P = 1 at f_g .......... whole path
  time-shift / dy-scale invariance ............ phase reduction, weight normalisation
  phase precision at config-3 range ........... O3/O4 double-double phases (PAPER.md:71 floor)
  phase winding vs direct ....... O-fast
"""
import os

import mpmath as mp
import numpy as np
import pytest

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden", "worked_example.txt")


def _gold():
    d = {}
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        k, v = line.split("=", 1)
        vals = [float(x) for x in v.split()]
        d[k.strip()] = vals[0] if len(vals) == 1 else np.array(vals)
    return d


# ---------------------------------------------------------------- worked example (golden file)
def test_worked_example_end_to_end():
    g = _gold()
    P, sums, aux = oracle.direct(g["t"], g["y"], g["dy"], g["f0"], g["df"], int(g["Nf"]), return_sums=True)
    assert np.max(np.abs(P - g["P"])) < 1e-14
    assert np.max(np.abs(sums[0] - g["sums_k0"])) < 1e-14
    assert np.max(np.abs(sums[3] - g["sums_k3"])) < 1e-14
    assert abs(aux[0, 0] - g["tan_k0"]) < 1e-13 and abs(aux[3, 0] - g["tan_k3"]) < 1e-13
    assert np.max(np.abs(aux[:, 1] - g["P"])) < 1e-13          # tau-free form agrees
    W, ybar, YY = oracle.stats(g["y"], g["dy"])
    assert abs(W - g["W"]) < 1e-13 and abs(ybar - g["ybar"]) < 1e-15 and abs(YY - g["YY"]) < 1e-15
    for variant in ("strict", "double-angle"):
        assert np.max(np.abs(oracle.direct(g["t"], g["y"], g["dy"], g["f0"], g["df"], 8, variant=variant) - g["P"])) < 1e-14
    assert np.max(np.abs(oracle.chi2(g["t"], g["y"], g["dy"], g["f0"], g["df"], 8) - g["P"])) < 1e-14
    assert np.max(np.abs(oracle.winding(g["t"], g["y"], g["dy"], g["f0"], g["df"], 0, 8) - g["P"])) < 1e-14


def test_assembly_alone_against_golden_sums():
    g = _gold()
    P, aux = oracle.assemble(np.stack([g["sums_k0"], g["sums_k3"]]), g["YY"])
    assert abs(P[0] - g["P"][0]) < 1e-14 and abs(P[1] - g["P"][3]) < 1e-14
    assert abs(aux[0, 0] - g["tan_k0"]) < 1e-13 and abs(aux[1, 0] - g["tan_k3"]) < 1e-13


# ---------------------------------------------------------------- mpmath brute force on tiny inputs
def _mp_reference(t, y, dy, f0, df, ks, dps=40):
    """Independent high-precision evaluation: trig sums by Eq. 1 AND the periodogram
    from its definition P = 1 - chi2_min/chi2_0 via a 3x3 weighted least-squares solve."""
    mp.mp.dps = dps
    t = [mp.mpf(float(v)) for v in t]; y = [mp.mpf(float(v)) for v in y]; dy = [mp.mpf(float(v)) for v in dy]
    w = [1 / (d * d) for d in dy]; W = mp.fsum(w); w = [v / W for v in w]
    ybar = mp.fsum(wi * yi for wi, yi in zip(w, y))
    chi0 = mp.fsum(wi * (yi - ybar) ** 2 for wi, yi in zip(w, y))
    out_P, out_sums = [], []
    for k in ks:
        f = mp.mpf(float(f0)) + int(k) * mp.mpf(float(df))
        c = [mp.cos(2 * mp.pi * f * tj) for tj in t]; s = [mp.sin(2 * mp.pi * f * tj) for tj in t]
        c2 = [mp.cos(4 * mp.pi * f * tj) for tj in t]; s2 = [mp.sin(4 * mp.pi * f * tj) for tj in t]
        h = [wi * (yi - ybar) for wi, yi in zip(w, y)]
        out_sums.append([mp.fsum(a * b for a, b in zip(h, s)), mp.fsum(a * b for a, b in zip(h, c)),
                         mp.fsum(a * b for a, b in zip(w, s)), mp.fsum(a * b for a, b in zip(w, c)),
                         mp.fsum(a * b for a, b in zip(w, s2)), mp.fsum(a * b for a, b in zip(w, c2))])
        B = [c, s, [mp.mpf(1)] * len(t)]
        A = mp.matrix(3, 3); r = mp.matrix(3, 1)
        for a in range(3):
            for b in range(3):
                A[a, b] = mp.fsum(wi * u * v for wi, u, v in zip(w, B[a], B[b]))
            r[a] = mp.fsum(wi * u * yi for wi, u, yi in zip(w, B[a], y))
        x = mp.lu_solve(A, r)
        chi = mp.fsum(wi * (yi - (x[0] * ci + x[1] * si + x[2])) ** 2 for wi, yi, ci, si in zip(w, y, c, s))
        out_P.append(1 - chi / chi0)
    return np.array([float(p) for p in out_P]), np.array([[float(v) for v in row] for row in out_sums])


@pytest.mark.parametrize("seed,Nd,Nf,offset", [(11, 64, 96, 0.0), (12, 37, 64, 0.0), (13, 48, 64, 2.45e6), (14, 5, 40, -733.25)])
def test_bruteforce_mpmath(seed, Nd, Nf, offset):
    rng = np.random.default_rng(seed)
    t = np.sort(rng.uniform(0, 40, Nd)) + offset
    y = rng.normal(0.3, 1.0, Nd) + np.sin(2 * np.pi * 0.37 * t)
    dy = rng.uniform(0.3, 2.0, Nd)
    f0, df = 0.013, 0.0171
    P_ref, S_ref = _mp_reference(t, y, dy, f0, df, range(Nf))
    P, sums, aux = oracle.direct(t, y, dy, f0, df, Nf, return_sums=True)
    assert np.max(np.abs(sums - S_ref)) < 5e-15
    # the power is a ratio of small differences at a few frequencies: 1e-12 absolute on P in [0,1]
    assert np.max(np.abs(P - P_ref)) < 1e-12
    assert np.max(np.abs(oracle.direct(t, y, dy, f0, df, Nf, variant="double-angle") - P_ref)) < 1e-12
    assert np.max(np.abs(oracle.chi2(t, y, dy, f0, df, Nf) - P_ref)) < 1e-11
    # subset indexing returns the same numbers as the full grid
    ks = np.array([0, 3, Nf - 1, 7])
    assert np.array_equal(oracle.direct(t, y, dy, f0, df, Nf, k=ks), P[ks])


def test_phase_precision_at_config3_range():
    """f*t up to 2.5e6 cycles (config 3: f_max ~ 250/day, t up to 1e4 days): a plain-double phase is
    off by ~1e-9 there (error floor N_f eps_mach); the oracle's double-double phase
    must stay at the 1e-15 level."""
    rng = np.random.default_rng(5)
    Nd = 24
    t = rng.uniform(0, 1.0e4, Nd); y = rng.normal(0, 1, Nd); dy = rng.uniform(0.5, 1.5, Nd)
    df = 1.0 / (5 * (t.max() - t.min())); f0 = df
    ks = np.array([12_499_999, 12_345_678, 6_250_001, 9_999_999, 1], dtype=np.int64)
    P_ref, S_ref = _mp_reference(t, y, dy, f0, df, ks)
    P, sums, _ = oracle.direct(t, y, dy, f0, df, 12_500_000, k=ks, return_sums=True)
    assert np.max(np.abs(sums - S_ref)) < 5e-15
    assert np.max(np.abs(P - P_ref)) < 1e-12
    # and the naive phase really is worse (so this pin has teeth)
    f = f0 + ks[:, None] * df
    naive = np.sum((1 / dy**2 / np.sum(1 / dy**2)) * np.sin(2 * np.pi * f * t[None, :]), axis=1)
    assert np.max(np.abs(naive - S_ref[:, 2])) > 1e-12


# ---------------------------------------------------------------- library routine
def test_against_scipy_lombscargle():
    from scipy.signal import lombscargle
    rng = np.random.default_rng(21)
    Nd, Nf = 200, 500
    t = np.sort(rng.uniform(0, 100, Nd)); dy = rng.uniform(0.5, 1.5, Nd)
    y = 1.7 + np.sin(2 * np.pi * 0.21 * t + 0.4) + rng.normal(0, 0.5, Nd)
    f0, df = 0.002, 0.002
    f = f0 + df * np.arange(Nf)
    ref = lombscargle(t, y, 2 * np.pi * f, normalize=True, weights=dy**-2.0, floating_mean=True)
    P = oracle.direct(t, y, dy, f0, df, Nf)
    assert np.max(np.abs(P - ref)) < 1e-11


# ---------------------------------------------------------------- second definition
@pytest.mark.parametrize("seed", [31, 32, 33])
def test_chi2_definition_equals_tau_formulas(seed):
    rng = np.random.default_rng(seed)
    Nd = int(rng.integers(8, 65))
    t = rng.uniform(0, 30, Nd); y = rng.normal(2.0, 1.0, Nd); dy = rng.uniform(0.2, 2.0, Nd)
    P, sums, aux = oracle.direct(t, y, dy, 0.01, 0.013, 300, return_sums=True)
    assert np.max(np.abs(P - oracle.chi2(t, y, dy, 0.01, 0.013, 300))) < 1e-12
    assert np.max(np.abs(P - aux[:, 1])) < 1e-11
    assert P.min() >= -1e-15 and P.max() <= 1 + 1e-15


# ---------------------------------------------------------------- closed form: equispaced -> DFT
@pytest.mark.parametrize("N", [33, 64, 101])
def test_equispaced_reduces_to_dft(N):
    rng = np.random.default_rng(N)
    Delta = 0.75
    t = Delta * np.arange(N); y = rng.normal(0.5, 1.0, N); dy = np.full(N, 0.8)
    f1 = 1.0 / (N * Delta)
    kmax = (N - 1) // 2
    P, sums, _ = oracle.direct(t, y, dy, f1, f1, kmax, return_sums=True)      # f_k = (k+1)/(N Delta)
    yc = y - y.mean()
    Y = np.fft.fft(yc)                                                        # sum yc e^{-2 pi i k j/N}
    k = np.arange(1, kmax + 1)
    assert np.max(np.abs(sums[:, 1] - Y.real[k] / N)) < 5e-15                 # Ch = Re sum h cos, h = yc/N
    assert np.max(np.abs(sums[:, 0] + Y.imag[k] / N)) < 5e-15                 # Sh = +sum h sin = -Im Y / N
    assert np.max(np.abs(sums[:, 2:])) < 5e-15                                # S = C = S2 = C2 = 0
    assert np.max(np.abs(P - 2 * np.abs(Y[k]) ** 2 / (N * np.sum(yc**2)))) < 1e-13
    if N % 2 == 1:
        assert abs(P.sum() - 1.0) < 1e-13                                     # Parseval


# ---------------------------------------------------------------- special case: noiseless sinusoid
def test_noiseless_sinusoid_power_is_one():
    rng = np.random.default_rng(41)
    Nd, Nf = 300, 2000
    t = rng.uniform(0, 200, Nd); dy = rng.uniform(0.5, 1.5, Nd)
    df = 1.0 / (5 * (t.max() - t.min())); f0 = df
    kg = 777
    fg = f0 + kg * df
    y = 3.1 + 1.3 * np.sin(2 * np.pi * fg * t + 0.9)
    P = oracle.direct(t, y, dy, f0, df, Nf)
    assert int(np.argmax(P)) == kg
    assert 1.0 - P[kg] < 1e-12


# ---------------------------------------------------------------- invariants
def test_time_shift_invariance():
    rng = np.random.default_rng(51)
    Nd, Nf = 2000, 5000
    t = rng.uniform(0, 3650, Nd); dy = rng.uniform(0.2, 1.0, Nd)
    y = 0.8 * np.sin(2 * np.pi * t / 23.1) + rng.normal(0, 0.5, Nd)
    df = 1.0 / (5 * (t.max() - t.min())); f0 = df
    P0 = oracle.direct(t, y, dy, f0, df, Nf)
    P1 = oracle.direct(t + 1825.0, y, dy, f0, df, Nf)       # t + 1825 rounds t: a 2e-13-day perturbation
    assert np.max(np.abs(P1 - P0)) / P0.max() < 1e-12
    P2 = oracle.direct(t - 4096.0, y, dy, f0, df, Nf)
    assert np.max(np.abs(P2 - P0)) / P0.max() < 1e-12


def test_dy_scale_invariance():
    rng = np.random.default_rng(52)
    Nd, Nf = 500, 800
    t = rng.uniform(0, 100, Nd); dy = rng.uniform(0.2, 1.0, Nd); y = rng.normal(0, 1, Nd)
    P0 = oracle.direct(t, y, dy, 0.01, 0.01, Nf)
    assert np.array_equal(oracle.direct(t, y, 4.0 * dy, 0.01, 0.01, Nf), P0)      # power of two: bit-identical
    assert np.max(np.abs(oracle.direct(t, y, 3.7 * dy, 0.01, 0.01, Nf) - P0)) < 1e-13


# ---------------------------------------------------------------- phase winding
def test_winding_matches_direct():
    rng = np.random.default_rng(61)
    Nd, Nf = 1000, 12500
    t = np.sort(rng.uniform(0, 1000, Nd)); dy = rng.uniform(0.5, 1.5, Nd)
    y = np.sin(2 * np.pi * t / 7.3) + rng.normal(0, 0.3, Nd)
    df = 1.0 / (5 * (t.max() - t.min())); f0 = df
    P = oracle.direct(t, y, dy, f0, df, Nf)
    Pw = oracle.winding(t, y, dy, f0, df, 0, Nf, reseed=64)
    assert np.max(np.abs(Pw - P)) / P.max() < 1e-12
    k0 = 5000
    assert np.max(np.abs(oracle.winding(t, y, dy, f0, df, k0, 300, reseed=7) - P[k0:k0 + 300])) / P.max() < 1e-12
    Pd = oracle.direct(t, y, dy, f0, df, Nf, variant="double-angle")
    assert np.max(np.abs(Pd - P)) / P.max() < 1e-13
