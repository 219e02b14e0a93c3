"""Helpers for the -m gpu parity tests: run a Workload through the C-ABI binding and compare with the
oracle.  Marshalling and error statistics only — no method arithmetic lives here."""
from __future__ import annotations

import numpy as np

# Gates (BASELINE.json north_star; DESIGN.md §3 reading A8): E_inf = max_k |P_gpu - P_or| / max_k P_or
GATE_F64 = 1e-8      # eps = 1e-9, fp64
GATE_F32 = 1e-4      # eps = 1e-5, fp32


def require_cuda():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("GPU test selected without a CUDA device (the library has no CPU fallback)")
    return torch


def gpu_power(w, host=False, return_plan_info=False, debug_modes=None, side_stream=False, repeat=1, **opts):
    """P[batch, Nf] (float64 numpy) of Workload `w` via ls_plan / ls_execute(/_host) / ls_destroy."""
    torch = require_cuda()
    from paper_2409_08090_b200 import binding as B
    dev = torch.device("cuda:0")
    tdt = torch.float64 if w.dtype == "f64" else torch.float32
    dy_per = 1 if (w.dy.ndim == 2) else 0
    plan = B.Plan(w.Nd, w.Nf, w.f0, w.df, w.eps, B.LS_F64 if w.dtype == "f64" else B.LS_F32, w.batch,
                  dy_per_series=dy_per, **opts)
    try:
        sobj = torch.cuda.Stream() if side_stream else torch.cuda.current_stream()
        stream = sobj.cuda_stream
        if host:
            P = np.empty((w.batch, w.Nf), dtype=w.np_dtype)
            plan.execute_host(np.ascontiguousarray(w.t), np.ascontiguousarray(w.y), np.ascontiguousarray(w.dy), P, stream)
            out = P.astype(np.float64)
        else:
            t = torch.from_numpy(np.ascontiguousarray(w.t)).to(dev)
            y = torch.from_numpy(np.ascontiguousarray(w.y)).to(dev)
            dy = torch.from_numpy(np.ascontiguousarray(w.dy)).to(dev)
            P = torch.full((w.batch, w.Nf), float("nan"), dtype=tdt, device=dev)
            torch.cuda.synchronize()
            for _ in range(repeat):                      # same buffers: a graph plan replays its capture
                plan.execute(t, y, dy, P, stream)
            if repeat > 1:                               # new output buffer: the plan must notice and re-capture
                P = torch.full((w.batch, w.Nf), float("nan"), dtype=tdt, device=dev)
                torch.cuda.synchronize()
                plan.execute(t, y, dy, P, stream)
            torch.cuda.synchronize()
            out = P.cpu().numpy().astype(np.float64)
        extra = {}
        if return_plan_info:
            extra["info"] = plan.info
            extra["launches"] = plan.launch_counts()
            extra["stats"] = B.ls_debug_stats(plan.handle, w.batch)
        if debug_modes is not None:
            series, ks = debug_modes
            extra["modes"] = B.ls_debug_modes(plan.handle, series, ks)
    finally:
        plan.close()
    return (out, extra) if (return_plan_info or debug_modes is not None) else out


def errors(Pg, Po):
    """Norm-wise gate value and the paper's pointwise statistics."""
    d = np.abs(Pg - Po)
    rel = d / np.maximum(Po, 1e-300)
    return {"Einf": float(d.max() / Po.max()), "median": float(np.median(rel)),
            "p99": float(np.percentile(rel, 99)), "max": float(rel.max())}


def oracle_power(w, b=0, ks=None, fast=False):
    """Oracle P of series b at indices ks (default full grid).  fast=True uses the phase-winding
    evaluator (pinned to the direct one at <= 1e-12 in test_oracle_pins.py)."""
    import oracle
    dy = w.dy[b] if w.dy.ndim == 2 else w.dy
    if ks is None and fast:
        return oracle.winding(w.t, w.y[b], dy, w.f0, w.df, 0, w.Nf)
    return oracle.direct(w.t, w.y[b], dy, w.f0, w.df, w.Nf, k=ks)
