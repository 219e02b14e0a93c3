"""-m gpu tests of the brute-force GPU evaluator (ls_direct_power) and, through it, of the NUFFT
path on frequency ranges the CPU oracle cannot cover.

1. ls_direct_power against the CPU oracle (configs 1 and 2): it is a verification tool, so it is itself checked first.
2. ls_execute (own FFT, fused) against ls_direct_power on 1.3 million frequencies of config 3 — contiguous slabs at
   both ends of the grid, across the mode-wrap seam and around the injected peak — where the oracle can only sample."""
import numpy as np
import pytest

from gpu_util import GATE_F64, errors, gpu_power, oracle_power, require_cuda
from paper_2409_08090_b200.workloads import make_workload

pytestmark = pytest.mark.gpu


def _direct(w, k0, K):
    torch = require_cuda()
    from paper_2409_08090_b200 import binding as B
    dev = torch.device("cuda:0")
    t = torch.from_numpy(w.t).to(dev); y = torch.from_numpy(np.ascontiguousarray(w.y[0])).to(dev)
    dy = torch.from_numpy(w.dy).to(dev)
    P = torch.full((K,), float("nan"), dtype=torch.float64, device=dev)
    B.ls_direct_power(w.Nd, w.f0, w.df, k0, K, t, y, dy, P, torch.cuda.current_stream().cuda_stream)
    return P.cpu().numpy()


def test_direct_against_oracle_cfg1_full_grid():
    w = make_workload(1)
    Pd = _direct(w, 0, w.Nf)
    Po = oracle_power(w)
    e = errors(Pd, Po)
    assert e["Einf"] <= 1e-12 and e["max"] <= 1e-9, e          # direct vs direct: rounding only


def test_direct_against_oracle_cfg2_offset_range_and_ragged_tail():
    w = make_workload(2)
    k0, K = 100_003, 24_997                                     # not a multiple of the 8 frequencies per thread
    Pd = _direct(w, k0, K)
    Po = oracle_power(w, fast=True)[k0:k0 + K]
    e = errors(Pd, Po)
    assert e["Einf"] <= 1e-12 and e["max"] <= 1e-8, e
    ks = np.arange(k0, k0 + K, 97)
    assert np.max(np.abs(Pd[ks - k0] - oracle_power(w, ks=ks))) <= 1e-12


def test_cfg3_nufft_power_against_direct_sums_through_the_oracles_assembly():
    """ls_direct_power shares the K6 arithmetic (ls_power.cuh) with the NUFFT path, so an error there would cancel in
    the comparison above.  Here the brute-force SUMS (ls_direct_sums: no assembly) go through the ORACLE's assembly, on
    2^17 frequencies of config 3 across the mode-wrap seam: K6 of the NUFFT path is checked by independent code."""
    import oracle
    torch = require_cuda()
    from paper_2409_08090_b200 import binding as B
    w = make_workload(3)
    Pg = gpu_power(w)[0]
    dev = torch.device("cuda:0")
    t = torch.from_numpy(w.t).to(dev); y = torch.from_numpy(np.ascontiguousarray(w.y[0])).to(dev)
    dy = torch.from_numpy(w.dy).to(dev)
    K = 1 << 17
    k0 = w.Nf // 2 - K // 2
    S = torch.empty((K, 6), dtype=torch.float64, device=dev)
    B.ls_direct_sums(w.Nd, w.f0, w.df, k0, K, t, y, dy, S, torch.cuda.current_stream().cuda_stream)
    sums = S.cpu().numpy()
    ks = k0 + np.arange(0, K, 4096)
    _, so, _ = oracle.direct(w.t, w.y[0], w.dy, w.f0, w.df, w.Nf, k=ks, return_sums=True)
    assert np.max(np.abs(sums[ks - k0] - so)) <= 1e-13           # direct vs direct sums (|sums| <= 1)
    _, _, YY = oracle.stats(w.y[0], w.dy)
    Po = oracle.assemble(sums, YY)[0]
    e = errors(Pg[k0:k0 + K], Po)
    assert e["Einf"] <= GATE_F64 and e["median"] <= 1e-8 and e["p99"] <= 1e-6, e


def test_direct_rejects_bad_arguments():
    require_cuda()
    from paper_2409_08090_b200 import binding as B
    with pytest.raises(B.LsError):
        B.ls_direct_power(0, 0.1, 0.1, 0, 10, 1, 1, 1, 1)
    with pytest.raises(B.LsError):
        B.ls_direct_power(10, 0.1, 0.0, 0, 10, 1, 1, 1, 1)
    with pytest.raises(B.LsError):
        B.ls_direct_power(10, 0.1, 0.1, 0, 10, 0, 1, 1, 1)      # NULL t


def test_cfg3_nufft_path_against_direct_on_wide_ranges():
    """Headline size, launch configuration of bench.py (auto plan: n = 2^24, own FFT)."""
    w = make_workload(3)
    Pg = gpu_power(w)[0]
    half = w.Nf // 2
    kpk = int(round((1 / 1.7 - w.f0) / w.df))
    slabs = [(0, 1 << 18), (half - (1 << 17), 1 << 18), (w.Nf - (1 << 18), 1 << 18), (3_000_000, 1 << 18),
             (9_000_001, (1 << 18) + 5)]                      # the first slab holds the injected peak (k ~ 29 400)
    assert 0 <= kpk < (1 << 18)
    pmax = Pg.max()
    worst, rel = 0.0, []
    for k0, K in slabs:
        Pd = _direct(w, k0, K)
        d = np.abs(Pg[k0:k0 + K] - Pd)
        worst = max(worst, float(d.max()))
        rel.append(d / np.maximum(Pd, 1e-300))
    rel = np.concatenate(rel)
    assert worst / pmax <= GATE_F64, worst / pmax
    assert np.median(rel) <= 1e-8 and np.percentile(rel, 99) <= 1e-6, (np.median(rel), np.percentile(rel, 99))
    assert int(np.argmax(Pg)) == kpk or abs(int(np.argmax(Pg)) - kpk) <= 1


def test_cfg5_fp32_path_against_direct_on_ranges():
    """Config 5 at full size (fp32 grids, autotuned n): three slabs of 2^15 frequencies against the fp64 brute force
    evaluated on the same (exactly promoted) fp32 inputs; gate of the fp32 config (north_star: <= 1e-4)."""
    from gpu_util import GATE_F32
    w = make_workload(5)
    Pg = gpu_power(w)[0]
    w64 = type(w)(w.name, w.t, w.y.astype(np.float64), w.dy.astype(np.float64), w.f0, w.df, w.Nf, "f64", w.eps)
    kpk = int(round((1 / 0.9137 - w.f0) / w.df))
    pmax = float(Pg.max())
    worst, rel = 0.0, []
    for k0 in (0, max(0, kpk - (1 << 14)), w.Nf // 2 - (1 << 14), w.Nf - (1 << 15)):
        Pd = _direct(w64, k0, 1 << 15)
        d = np.abs(Pg[k0:k0 + (1 << 15)] - Pd)
        worst = max(worst, float(d.max()))
        rel.append(d / np.maximum(Pd, 1e-300))
    rel = np.concatenate(rel)
    assert worst / pmax <= GATE_F32, worst / pmax
    assert np.median(rel) <= 1e-4, np.median(rel)


def test_cfg3_julian_date_sized_time_offset_against_direct_and_oracle():
    """Config 3 with t + 2 450 000.5 (Julian-date-sized times: f t reaches 6e8 cycles, the regime that needs the
    (cell, fraction) double-double coordinates): NUFFT path vs brute force on two slabs, and both vs the
    CPU oracle on sampled frequencies of those slabs."""
    w = make_workload(3)
    w2 = type(w)(w.name + "_jd", w.t + 2450000.5, w.y, w.dy, w.f0, w.df, w.Nf, "f64", w.eps)
    Pg = gpu_power(w2)[0]
    pmax = float(Pg.max())
    for k0 in (0, w.Nf - (1 << 17)):
        K = 1 << 17
        Pd = _direct(w2, k0, K)
        assert np.max(np.abs(Pg[k0:k0 + K] - Pd)) / pmax <= GATE_F64
        ks = k0 + np.arange(0, K, 2048)
        Po = oracle_power(w2, ks=ks)
        assert np.max(np.abs(Pd[ks - k0] - Po)) / pmax <= 1e-11           # direct vs direct
        assert np.max(np.abs(Pg[ks] - Po)) / pmax <= GATE_F64
