"""-m gpu test of ls_direct_power_noalloc (include/ls.h): the brute-force evaluator with its scratch in a fixed device
array inside the library instead of a cudaMalloc per call, for callers that cannot allocate.  Collected last on purpose
(the file name): the suite runs with pytest -x.

The new entry point against the existing one (ls_direct_power) on the same inputs, on two calls in a row that share the
array — a larger problem first, then a smaller one, so that stale sums or stale points of the first call would show in the
second — plus the size limit.  Tolerance: the one tests/test_gpu_direct.py uses for direct against direct (1e-12 of a
power in [0, 1]: the statistics are accumulated with atomics, so two runs differ in the last bits)."""
import numpy as np
import pytest

from gpu_util import require_cuda
from paper_2409_08090_b200.workloads import make_workload, scaled_workload

pytestmark = pytest.mark.gpu


def _both(w, k0, K):
    torch = require_cuda()
    from paper_2409_08090_b200 import binding as B
    dev = torch.device("cuda:0")
    t = torch.from_numpy(np.ascontiguousarray(w.t)).to(dev)
    y = torch.from_numpy(np.ascontiguousarray(w.y[0])).to(dev)
    dy = torch.from_numpy(np.ascontiguousarray(w.dy)).to(dev)
    stream = torch.cuda.current_stream().cuda_stream
    P_ref = torch.full((K,), float("nan"), dtype=torch.float64, device=dev)
    B.ls_direct_power(w.Nd, w.f0, w.df, k0, K, t, y, dy, P_ref, stream)              # allocates, synchronises
    P_new = torch.full((K,), float("nan"), dtype=torch.float64, device=dev)
    B.ls_direct_power_noalloc(w.Nd, w.f0, w.df, k0, K, t, y, dy, P_new, stream)      # asynchronous
    torch.cuda.synchronize()
    return P_new.cpu().numpy(), P_ref.cpu().numpy()


def test_no_alloc_entry_point_matches_the_allocating_one_on_two_calls_in_a_row():
    w2 = make_workload(2)                                  # N_d = 10 000, a ragged range of frequencies
    Pn, Pr = _both(w2, 100_003, 24_997)
    assert np.all(np.isfinite(Pn)) and np.max(np.abs(Pn - Pr)) <= 1e-12
    w1 = make_workload(1)                                  # N_d = 1 000: the array still holds config 2's sums and points
    Pn, Pr = _both(w1, 0, w1.Nf)
    assert np.all(np.isfinite(Pn)) and np.max(np.abs(Pn - Pr)) <= 1e-12
    assert int(np.argmax(Pn)) == int(np.argmax(Pr))
    Pn2, _ = _both(w1, 0, w1.Nf)                           # and once more with the same inputs
    assert np.max(np.abs(Pn2 - Pn)) <= 1e-12


def test_no_alloc_entry_point_size_limit():
    torch = require_cuda()
    from paper_2409_08090_b200 import binding as B
    wmax = scaled_workload(3, B.LS_NOALLOC_MAX_ND)         # exactly the maximum: accepted
    assert wmax.Nd == B.LS_NOALLOC_MAX_ND
    Pn, Pr = _both(wmax, wmax.Nf // 2 - 100, 203)
    assert np.all(np.isfinite(Pn)) and np.max(np.abs(Pn - Pr)) <= 1e-12
    dev = torch.device("cuda:0")
    Nd = B.LS_NOALLOC_MAX_ND + 1                           # one more: refused, nothing enqueued, output untouched
    t = torch.linspace(0.0, 100.0, Nd, dtype=torch.float64, device=dev)
    y = torch.sin(t)
    dy = torch.ones_like(t)
    P = torch.full((16,), -7.0, dtype=torch.float64, device=dev)
    with pytest.raises(B.LsError) as ei:
        B.ls_direct_power_noalloc(Nd, 0.01, 0.01, 0, 16, t, y, dy, P, torch.cuda.current_stream().cuda_stream)
    assert ei.value.code == B.LS_ERR_TOO_LARGE and "LS_NOALLOC_MAX_ND" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((P == -7.0).all())
