"""Host-side logic of the N > 1 bench path on CPU: two processes, gloo backend, world size 2.

The hot path has no exchange step: ranks run independent series and only their TIMINGS meet
(max over ranks).  This checks that each rank draws its own series, that the max-reduction and the whole-job
value are right, and that rendezvous over 127.0.0.1 works the way bench.py does it under torchrun."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = bench.rank_workload(1, rank)
        # pretend rank r took (10 + 5 r) ms on the device leg and (20 - 3 r) ms end to end
        dev_ms, e2e_ms = bench.max_over_ranks([10.0 + 5 * rank, 20.0 - 3 * rank], torch.device("cpu"), world)
        ms_per_step, value = bench.whole_job_value(dev_ms, steps=5, batch=w.batch, world=world)
        dist.barrier()
        out.put((rank, float(w.t[0]), float(w.y[0, 0]), w.Nd, w.Nf, dev_ms, e2e_ms, ms_per_step, value))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo_weak_scaling_logic():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, t0, y0, Nd0, Nf0, d0, e0, s0, v0), (r1, t1, y1, Nd1, Nf1, d1, e1, s1, v1) = res
    assert (Nd0, Nf0) == (Nd1, Nf1) == (1000, 12500)            # same shape on every rank (weak scaling)
    assert t0 != t1 and y0 != y1                                # ... but each rank has its own series
    assert d0 == d1 == 15.0 and e0 == e1 == 20.0                # max over ranks, identical on both
    assert s0 == pytest.approx(3.0) and v0 == pytest.approx(1.5)  # 15 ms / 5 steps; / (1 series x 2 ranks)


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([1.5, 2.5], torch.device("cpu"), 1) == [1.5, 2.5]
    assert bench.whole_job_value(10.0, 5, 4, 1) == (2.0, 0.5)
    w0, w1 = bench.rank_workload(2, 0), bench.rank_workload(2, 3)
    assert w0.Nd == w1.Nd and not np.array_equal(w0.t, w1.t)
