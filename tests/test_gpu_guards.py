"""-m gpu: out-of-bounds WRITE check of every kernel through guard zones (compute-sanitizer is closed on this GPU
pool: profiles/r2_checks.md).  With LS_B200_GUARD in the environment every plan-owned device buffer sits between two
256-byte zones of 0xA5; after the executes no guard byte may have changed, on every code path the five configs take:
small and pruned own FFT, cuFFT, batches in several passes, per-series dy, fp32, the host-buffer entry point."""
import numpy as np
import pytest

from gpu_util import require_cuda
from paper_2409_08090_b200.workloads import Workload, make_workload, scaled_workload

pytestmark = pytest.mark.gpu


def _run(w, monkeypatch, host=False, repeat=2, expect=None, **opts):
    torch = require_cuda()
    from paper_2409_08090_b200 import binding as B
    monkeypatch.setenv("LS_B200_GUARD", "1")
    dev = torch.device("cuda:0")
    tdt = torch.float64 if w.dtype == "f64" else torch.float32
    per = 1 if w.dy.ndim == 2 else 0
    with B.Plan(w.Nd, w.Nf, w.f0, w.df, w.eps, B.LS_F64 if w.dtype == "f64" else B.LS_F32, w.batch, dy_per_series=per, **opts) as plan:
        s = torch.cuda.Stream()
        if expect is not None:                       # (n, cuFFT execs per execute) the case is meant to exercise
            assert plan.info["n"] == expect[0], plan.info
        if host:
            P = np.empty((w.batch, w.Nf), dtype=w.np_dtype)
            for _ in range(repeat):
                plan.execute_host(np.ascontiguousarray(w.t), np.ascontiguousarray(w.y), np.ascontiguousarray(w.dy), P, s.cuda_stream)
        else:
            t = torch.from_numpy(np.ascontiguousarray(w.t)).to(dev); y = torch.from_numpy(np.ascontiguousarray(w.y)).to(dev)
            dy = torch.from_numpy(np.ascontiguousarray(w.dy)).to(dev)
            P = torch.empty((w.batch, w.Nf), dtype=tdt, device=dev)
            for _ in range(repeat):
                plan.execute(t, y, dy, P, s.cuda_stream)
            torch.cuda.synchronize()
            assert bool(torch.isfinite(P).all())
        if expect is not None:
            assert plan.launch_counts()[1] == expect[1]
        return B.ls_debug_guards(plan.handle)


def _p20(batch=1):
    rng = np.random.default_rng(33)
    Nf = int(0.7 * (1 << 20)); Nd = 60_000
    t = rng.uniform(0, 700.0, Nd); dy = rng.uniform(0.5, 1.5, Nd)
    df = 1.0 / (5 * (t.max() - t.min()))
    y = np.stack([np.sin(2 * np.pi * 3.3 * t + b) + rng.normal(0, 1, Nd) for b in range(batch)])
    return Workload("guards_p20", t, y, dy, df, df, Nf, "f64", 1e-9)


def _resized(w, Nf):
    return Workload(w.name + "_resized", w.t, w.y, w.dy, w.f0, w.df, Nf, w.dtype, w.eps)


def test_no_kernel_writes_outside_its_buffers(monkeypatch):
    assert _run(make_workload(1), monkeypatch) == 0                                 # n = 2^14, own two-pass FFT
    assert _run(make_workload(2), monkeypatch) == 0                                 # n = 2^18, own FFT, small first radix
    assert _run(make_workload(2), monkeypatch, fft_impl=1, host=True) == 0          # cuFFT path, host buffers
    assert _run(_p20(), monkeypatch, no_autotune=1) == 0                            # pruned pass 1 + TMA passes 2 + 3
    assert _run(_p20(), monkeypatch, no_autotune=1, fft_impl=2) == 0                # last pass fused with the assembly
    assert _run(_p20(3), monkeypatch, no_autotune=1, batch_chunk=2) == 0            # batch in two passes, own FFT
    w4 = scaled_workload(4, 1500, batch=7)
    assert _run(w4, monkeypatch, batch_chunk=3) == 0                                # batch, cuFFT or small own FFT
    w4.dy = np.ascontiguousarray(np.random.default_rng(1).uniform(0.5, 1.5, (7, w4.Nd)))
    assert _run(w4, monkeypatch) == 0                                               # per-series dy
    assert _run(w4, monkeypatch, no_floating_mean=1) == 0                           # fixed mean: shorter slot layout
    assert _run(scaled_workload(5, 60_000), monkeypatch) == 0                       # fp32, clustered
    assert _run(scaled_workload(5, 60_000), monkeypatch, t_is_dtype=0, tile_cells=256) == 0
    # the round-2 transforms on grids of 5 x 2^k cells: fp64 two passes (a batch: pruned first pass, fused last pass; and
    # one series through the unfused kernels), fp32 three passes (pruned first pass, liveness masks of 2 x 128 x 5 words)
    w5 = scaled_workload(4, 1500, batch=9)
    n5 = 5 << 13
    assert _run(_resized(w5, int(n5 / 1.3107)), monkeypatch, expect=(n5, 0), upsampfac=n5 / int(n5 / 1.3107) * (1 - 1e-9)) == 0
    assert _run(_resized(scaled_workload(2, 3000), int((5 << 14) / 1.3107)), monkeypatch, expect=(5 << 14, 0), fft_impl=3,
                upsampfac=(5 << 14) / int((5 << 14) / 1.3107) * (1 - 1e-9)) == 0
    wf = scaled_workload(5, 60_000)
    nf = 5 << 22
    assert _run(_resized(wf, int(nf / 1.3107)), monkeypatch, expect=(nf, 0), upsampfac=nf / int(nf / 1.3107) * (1 - 1e-9), tile_cells=512) == 0


def test_guards_need_the_environment_variable(monkeypatch):
    """A plan made without LS_B200_GUARD has no guard zones: the hook says so instead of reporting a clean bill."""
    torch = require_cuda()
    from paper_2409_08090_b200 import binding as B
    monkeypatch.delenv("LS_B200_GUARD", raising=False)
    with B.Plan(100, 1000, 0.1, 0.1, 1e-9, B.LS_F64, 1) as plan:
        with pytest.raises(B.LsError) as ei:
            B.ls_debug_guards(plan.handle)                                           # made without the variable
        assert ei.value.code == 6
