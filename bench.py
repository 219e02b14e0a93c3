#!/usr/bin/env python
"""bench.py — ms per periodogram / NU points per second of the Lomb-Scargle hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

One "step" = one pass of the whole hot path (K1 stats, K3 bin-sort, K2 premultiply, K4 spread, cuFFT,
K5+K6 deconvolve + assemble) over one synthetic series set of the chosen BASELINE.json
config (default: config 3, N_d = 1e6, N_f = 1.25e7, fp64, eps = 1e-9 — the one `metric` is quoted on).
Prints ONE JSON line (rank 0).  See DESIGN.md §8 for every field.

  value        ms per periodogram, device-timed (CUDA events on the launching stream), inputs resident
               in HBM, L2 flushed between steps; whole job: max-over-ranks time / periodograms of all ranks
  e2e          same through ls_execute_host with pinned HOST buffers (H2D of t, y, dy and D2H of power
               inside the timed region)
  roofline     dominant own kernel (stage timers inside the library, CUDA events) vs measured HBM peak
  path_roofline  the north_star figure: model bytes of spread + deconvolve + assembly path (everything
               except the cuFFT) / (t_total - t_fft)
  cpu_baseline the oracle as it stands on this box's host cores, bounded frequency sample

`--impl reference` times the CPU oracle (this tier's reference arm) on a bounded sample per step.
Multi-GPU (torchrun): the path has no exchange step — each rank runs its own series ("weak").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "ms/periodogram"
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback ("of fallback")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-freqs", type=int, default=0, help="oracle sample size (0 = auto)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (tuning runs)")
    ap.add_argument("--parity-k", type=int, default=64, help="frequencies of the timed plan's output checked against "
                    "the oracle after the timed loop (0 = skip)")
    # plan tuning knobs (ls_opts); 0 = the library's automatic choice
    ap.add_argument("--tile-cells", type=int, default=0)
    ap.add_argument("--upsampfac", type=float, default=0.0)
    ap.add_argument("--kernel-width", type=int, default=0)
    ap.add_argument("--batch-chunk", type=int, default=0)
    ap.add_argument("--fft-impl", type=int, default=0, help="0 auto, 1 cuFFT, 2 own FFT with the last pass fused into the assembly, 3 own FFT unfused")
    ap.add_argument("--graph", type=int, default=0, help="0 auto, 1 never, 2 always (user-facing plan)")
    ap.add_argument("--traffic-from", default="", help="CPU-side helper: turn `ncu -i REP --page raw --csv` output into "
                    "profiles/r2_traffic.csv (needs --traffic-meta workload,n,w and --traffic-command)")
    ap.add_argument("--traffic-meta", default="cfg3_single_Nd1e6_f64,16777216,17")
    ap.add_argument("--traffic-command", default="")
    ap.add_argument("--variant", type=int, default=0, help="ls_opts.reserved[0]: kernel variant kept for comparison")
    ap.add_argument("--lag", type=int, default=0, help="ls_opts.reserved[1]: queue lag of the fused FFT kernels (0 = default)")
    return ap.parse_args()


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (profiling recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "25"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
                for nm, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


# ----------------------------------------------------------------------------- workloads
def rank_workload(cfg: int, rank: int):
    """Config `cfg`; ranks > 0 draw their own series (same recipe, different seed): the path has no
    exchange step, so multi-GPU is weak scaling over independent periodograms."""
    from paper_2409_08090_b200.workloads import _BUILDERS, _SEEDS, make_workload
    if rank == 0:
        return make_workload(cfg)
    return _BUILDERS[cfg](seed=_SEEDS[cfg] + 1000 * rank)


def oracle_sample(w, K):
    """Frequency indices of the bounded oracle sample: K seeded random k of the Nf."""
    rng = np.random.default_rng(w.seed + 77)
    return np.sort(rng.choice(w.Nf, size=min(K, w.Nf), replace=False)).astype(np.int64)


def auto_cpu_freqs(w, cores, target_s=15.0):
    # direct evaluation costs ~ Nd * K * batch point-frequency pairs at ~2e7 pairs/s/core (strict variant, measured on the GPU box's 16 cores)
    pairs = target_s * 2.0e7 * max(cores, 1)
    return int(max(8, min(w.Nf, pairs / (w.Nd * min(w.batch, 4)))))


def time_oracle(w, K):
    """The oracle as it stands (oracle.direct, strict variant), on K sampled frequencies of up to 4
    series; returns (seconds for the sample, extrapolated ms per full periodogram, series used)."""
    import oracle
    ks = oracle_sample(w, K)
    nser = min(w.batch, 4)
    t0 = time.perf_counter()
    for b in range(nser):
        oracle.direct(w.t, w.y[b], w.dy, w.f0, w.df, w.Nf, k=ks)
    dt = time.perf_counter() - t0
    ms_full = dt / nser * (w.Nf / ks.size) * 1e3          # cost is exactly linear in the number of frequencies
    return dt, ms_full, nser, int(ks.size)


def config_dict(w, extra=None):
    d = {"workload": w.name, "Nd": w.Nd, "Nf": w.Nf, "batch": w.batch, "eps": w.eps,
         "l2": "flushed between steps (write of a 512 MiB buffer, > the 126 MB L2)"}
    if extra:
        d.update(extra)
    return d


# ----------------------------------------------------------------------------- reference arm
def run_reference(args):
    """This tier's reference arm = the CPU oracle, timed as it stands on the host cores.  Rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    w = rank_workload(args.config, 0)
    cores = oracle.num_threads()
    K = args.cpu_freqs or max(8, auto_cpu_freqs(w, cores, target_s=3.0))
    for _ in range(args.warmup):
        time_oracle(w, max(8, K // 8))
    tot_s, ms_acc = 0.0, 0.0
    for _ in range(args.steps):
        dt, ms_full, nser, kk = time_oracle(w, K)
        tot_s += dt; ms_acc += ms_full
    ms = ms_acc / args.steps
    sample = (f"{kk} of {w.Nf} frequencies x {nser} of {w.batch} series per step (oracle.direct, strict), "
              f"time extrapolated linearly to the full grid")
    line = {"impl": "reference", "metric": METRIC, "value": ms, "unit": "ms", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": tot_s / args.steps * 1e3,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(w), "gpu_launches": 0,
            "nu_pts_per_s": 3.0 * w.Nd * w.batch / (ms * 1e-3),
            "cpu_baseline": {"value": ms, "unit": "ms", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": ms, "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------- multi-rank host logic
def max_over_ranks(values, device, world):
    """Element-wise MAX over all ranks of a list of per-rank timings (the contract's max-over-ranks);
    identity at world size 1.  Works on any backend (NCCL on the GPU box, gloo in the CPU tests)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_value(total_ms, steps, batch, world):
    """(ms per step, ms per periodogram) of the WHOLE job: every rank runs `batch` periodograms per step
    (weak scaling: no exchange step), all ranks' periodograms divide the slowest rank's time."""
    ms_per_step = total_ms / steps
    return ms_per_step, ms_per_step / (batch * world)


# ----------------------------------------------------------------------------- our arm
STAGE_BYTES_DOC = "DESIGN.md §6"


def occupied_tile_rows(w, info, L):
    """(tiles holding points) x (transforms of that point set), summed over the two point sets — what the
    spreading kernel writes and the first FFT pass reads when the own FFT is used (empty tiles are never
    written).  Host-side count from the inputs; plain doubles are ample for counting tiles."""
    n, wd = info["n"], info["w"]
    ntiles = (n + L - 1) // L
    u1 = np.mod(n * w.df * w.t, n)
    out = 0
    for u, rows in ((u1, 1 + w.batch), (np.mod(2.0 * u1, n), 1)):
        lo = np.floor((u - wd / 2 - 1) / L).astype(np.int64) % ntiles
        hi = np.floor((u + wd / 2 + 1) / L).astype(np.int64) % ntiles
        out += np.union1d(lo, hi).size * rows
    return out


def stage_model_bytes(w, info, own_fft, L):
    """Algorithmic HBM bytes per execute of each own kernel: every
    intermediate written once and read once, nothing counted for re-reads or halo candidates.  With the
    own FFT the fine grids are sparse (only tiles that hold points exist), so the grid term of the
    spreading kernel and of the first FFT pass's reads is the occupied part, not M n."""
    B = 8 if w.dtype == "f64" else 4
    Nd, Nf, n, M, batch = w.Nd, w.Nf, info["n"], info["M"], w.batch
    nbins = n // 64
    rec = 4 * B                                           # one bin-sorted point record (32 B fp64 / 16 B fp32)
    rows = M * Nd * B                                     # real strengths, one row per transform
    grid = M * n * 2 * B
    n5 = n % 5 == 0 and (n // 5) & (n // 5 - 1) == 0
    pruned = own_fft and (n >= 1 << 20 or n5)             # tiles without points are neither written nor read
    written = occupied_tile_rows(w, info, L) * L * 2 * B if pruned else grid
    d = {
        "stats": 8 * Nd + batch * Nd * B + Nd * B + 2 * 4 * nbins,
        "sort": 3 * 2 * 4 * nbins,
        "premul": 8 * Nd + batch * Nd * B + Nd * B + 2 * Nd * rec + rows + (0 if batch == 1 else 2 * 4 * Nd),
        "spread": written + 2 * Nd * rec + rows,
        "assemble": M * Nf * 2 * B + batch * Nf * B + (Nf // 2 + 1) * 8,
    }
    if own_fft:
        d.update({"fft_pass1": written + grid, "fft_pass2": 2 * grid, "fft_pass3": grid + M * Nf * 2 * B,
                  # passes 2 + 3 as one kernel, intermediate in L2 and discarded: grid in, kept modes out
                  "fft_pass23": grid + M * Nf * 2 * B})
    return d


TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r2_traffic.csv")
KERNEL_STAGE = {"ls_stats_count_kernel": "stats", "ls_premultiply_kernel": "premul", "ls_spread_tile_kernel": "spread",
                "ls_fft_pass1_kernel": "fft_pass1", "ls_fft_pass23_tma_kernel": "fft_pass23", "ls_fft_pass23_kernel": "fft_pass23",
                "ls_assemble_kernel": "assemble", "ls_assemble_shared_kernel": "assemble", "ls_fft_cols_kernel": "fft_pass2",
                "ls_fft_rows_kernel": "fft_pass3", "ls_bin_scan_totals_kernel": "sort", "ls_bin_scan_apply_kernel": "sort",
                "ls_tile_list_kernel": "sort", "ls_rows_kernel": "premul"}


def source_hash():
    """sha256 prefix over the library's CUDA sources: ties a committed ncu capture to the kernels it measured."""
    import glob, hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_2409_08090_b200", "csrc")
    for f in sorted(glob.glob(os.path.join(csrc, "*.cu")) + glob.glob(os.path.join(csrc, "*.cuh")) + glob.glob(os.path.join(csrc, "*.h"))):
        with open(f, "rb") as fh:
            h.update(os.path.basename(f).encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


def write_traffic(raw_csv, meta, command):
    """`ncu -i X.ncu-rep --page raw --csv` output -> profiles/r2_traffic.csv (per-launch means of every own kernel),
    stamped with the hash of the sources it was captured from.  Runs on the CPU box; no GPU needed."""
    import csv
    workload, n, wd = meta.split(",")
    with open(raw_csv) as f:
        rows = list(csv.reader(f))
    hdr = rows[0]
    ik, it = hdr.index("Kernel Name"), hdr.index("gpu__time_duration.sum")
    ir, iw = hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
    units = rows[1]
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "ns": 1e-3, "us": 1.0, "ms": 1e3, "usecond": 1.0, "nsecond": 1e-3, "msecond": 1e3}
    acc = {}
    for r in rows[2:]:
        name = next((k for k in KERNEL_STAGE if k in r[ik]), None)
        if name is None:
            continue
        a = acc.setdefault(name, [0, 0.0, 0.0, 0.0])
        a[0] += 1
        a[1] += float(r[it].replace(",", "")) * scale[units[it]]
        a[2] += float(r[ir].replace(",", "")) * scale[units[ir]]
        a[3] += float(r[iw].replace(",", "")) * scale[units[iw]]
    with open(TRAFFIC_FILE, "w") as f:
        f.write("# dram__bytes_read.sum / dram__bytes_write.sum per launch (mean over the captured launches) of every own kernel\n")
        f.write(f"# command: {command}\n")
        f.write(f"# source_hash: {source_hash()}\n")
        f.write("stage,kernel,workload,n,w,launches,time_us,dram_read_bytes,dram_write_bytes\n")
        for name, a in acc.items():
            f.write(f"{KERNEL_STAGE[name]},{name},{workload},{n},{wd},{a[0]},{a[1] / a[0]:.1f},{a[2] / a[0]:.0f},{a[3] / a[0]:.0f}\n")
    print(f"wrote {TRAFFIC_FILE} ({len(acc)} kernels, source_hash {source_hash()})")


def measured_traffic(kernel_stage, w, info):
    """(dram__bytes_read.sum + dram__bytes_write.sum per launch of the stage's kernels, capture record) from the
    committed ncu --set full capture profiles/r2_traffic.csv; the record says which sources the capture saw and whether
    they are the sources of this run (`stale`).  (None, None) when the capture does not cover this workload / plan."""
    try:
        with open(TRAFFIC_FILE) as f:
            lines = [l.strip() for l in f if l.strip()]
        cap_hash = next((l.split(":", 1)[1].strip() for l in lines if l.startswith("# source_hash:")), None)
        rows = [l.split(",") for l in lines if not l.startswith("#")]
        hdr, rows = rows[0], rows[1:]
        tot = None
        for r in rows:
            d = dict(zip(hdr, r))
            if d["stage"] == kernel_stage and d["workload"] == w.name and int(d["n"]) == info["n"] and int(d["w"]) == info["w"]:
                tot = (tot or 0.0) + float(d["dram_read_bytes"]) + float(d["dram_write_bytes"])
        if tot is None:
            return None, None
        return tot, {"file": "profiles/r2_traffic.csv", "source_hash": cap_hash, "stale": cap_hash != source_hash()}
    except Exception:
        return None, None


def run_ours(args):
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the library has no CPU fallback")
    from paper_2409_08090_b200 import binding as B
    from paper_2409_08090_b200.build import build
    build()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    w = rank_workload(args.config, rank)
    tdt = torch.float64 if w.dtype == "f64" else torch.float32
    t = torch.from_numpy(w.t).to(dev); y = torch.from_numpy(w.y).to(dev); dy = torch.from_numpy(w.dy).to(dev)
    P = torch.empty((w.batch, w.Nf), dtype=tdt, device=dev)
    # pinned host buffers for the e2e leg
    ht = torch.from_numpy(w.t).pin_memory(); hy = torch.from_numpy(w.y).pin_memory()
    hdy = torch.from_numpy(w.dy).pin_memory()
    hP = torch.empty((w.batch, w.Nf), dtype=tdt).pin_memory()
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    popts = dict(device=local, tile_cells=args.tile_cells, upsampfac=args.upsampfac,
                 kernel_width=args.kernel_width, batch_chunk=args.batch_chunk, fft_impl=args.fft_impl)
    if args.variant or args.lag:
        popts["reserved"] = (args.variant, args.lag)
    ldt = B.LS_F64 if w.dtype == "f64" else B.LS_F32
    # Two plans: `plan` is what a user runs (no stage events; small problems replay a CUDA graph; with the own FFT
    # the last pass is fused with the assembly) and gives `value`; `plan_t` records CUDA events around every
    # stage and gives stage_ms / the roofline legs — same n, w and FFT, but with the assembly as its own kernel
    # (fft_impl 3) so that "fft" and "assemble" are cleanly separated as north_star asks.
    plan = B.Plan(w.Nd, w.Nf, w.f0, w.df, w.eps, ldt, w.batch, timing=0, graph=args.graph, **popts)
    info = plan.info
    if not args.upsampfac:
        popts["upsampfac"] = info["n"] / w.Nf * (1 - 1e-12) if info["n"] & (info["n"] - 1) else 0.0   # same n as `plan`
    plan_t = None
    n5 = info["n"] % 5 == 0 and (info["n"] // 5) & (info["n"] // 5 - 1) == 0       # 5 x 2^k: own two-pass FFT, fused for batches
    if popts["fft_impl"] == 2 or (popts["fft_impl"] == 0 and n5):
        try:
            plan_t = B.Plan(w.Nd, w.Nf, w.f0, w.df, w.eps, ldt, w.batch, timing=1, no_autotune=1,
                            **dict(popts, fft_impl=3))
        except B.LsError:                             # own FFT not available for this grid: cuFFT plan
            plan_t = None
    if plan_t is None:
        plan_t = B.Plan(w.Nd, w.Nf, w.f0, w.df, w.eps, ldt, w.batch, timing=1, no_autotune=1, **popts)
    assert plan_t.info["n"] == info["n"] and plan_t.info["w"] == info["w"], (plan_t.info, info)
    side = torch.cuda.Stream(device=dev)             # a capturable (non-legacy) stream; all timed work runs on it
    stream = side.cuda_stream

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    with torch.cuda.stream(side):
        for _ in range(max(args.warmup, 3)):
            plan.execute(t, y, dy, P, stream)
            plan_t.execute(t, y, dy, P, stream)
    torch.cuda.synchronize()
    own, ffts = plan.launch_counts()

    # ---- device-resident leg: K steps, each bracketed by events on the launching stream, L2 flushed in between
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    stage_acc = {k: 0.0 for k in B.STAGES}
    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    wall0 = time.perf_counter()
    with torch.cuda.stream(side):
        for i in range(args.steps):
            flush.fill_(i & 0xFF)
            ev[i][0].record()
            plan.execute(t, y, dy, P, stream)
            ev[i][1].record()
    barrier()
    wall = time.perf_counter() - wall0
    step_ms = [a.elapsed_time(b) for a, b in ev]
    dev_ms = float(np.sum(step_ms))
    # stage timers: the same K steps through the event-recording plan (not part of `value`)
    with torch.cuda.stream(side):
        for i in range(args.steps):
            flush.fill_(i & 0xFF)
            plan_t.execute(t, y, dy, P, stream)
            side.synchronize()
            for k, v in plan_t.stage_ms().items():
                stage_acc[k] += v
    barrier()

    # ---- e2e leg: host buffers through ls_execute_host (H2D + D2H inside the timed region)
    # A batch that the device-timed plan runs in one pass goes through a second plan with batch_chunk = batch / 8 here:
    # ls_execute_host copies a pass's power to the host while the next pass is computed (ls.h), which one pass cannot.
    plan_e, e2e_plan = plan, "the timed plan"
    if not args.no_e2e and w.batch >= 64 and not args.batch_chunk:
        ck = -(-w.batch // 8)
        plan_e = B.Plan(w.Nd, w.Nf, w.f0, w.df, w.eps, ldt, w.batch, timing=0, graph=args.graph, no_autotune=1,
                        **dict(popts, batch_chunk=ck))   # popts pins the timed plan's n
        e2e_plan = f"own plan, batch_chunk={ck} ({-(-w.batch // ck)} passes: the copy-out of a pass overlaps the next pass)"
    for _ in range(0 if args.no_e2e else 2):
        plan_e.execute_host(ht, hy, hdy, hP, stream)
    e2e_ms = 0.0
    barrier()
    for i in range(0 if args.no_e2e else args.steps):
        flush.fill_(i & 0xFF)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        plan_e.execute_host(ht, hy, hdy, hP, stream)     # synchronises the stream before returning
        e2e_ms += (time.perf_counter() - t0) * 1e3
    barrier()
    e2e_diff = None
    if not args.no_e2e:                                  # the host leg's output against the device leg's (same inputs)
        e2e_diff = float((hP.to(dev) - P).abs().max().item())
    if plan_e is not plan:
        plan_e.close()
    clocks = sampler.stop() if rank == 0 else None      # sampled over both timed legs

    dev_ms, e2e_ms = max_over_ranks([dev_ms, e2e_ms], dev, world)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    n_periodograms = w.batch * world                      # per step, all ranks
    ms_per_step, value = whole_job_value(dev_ms, args.steps, w.batch, world)
    stage = {k: v / args.steps for k, v in stage_acc.items()}
    peak, peak_src = measured_peak()
    own_fft = ffts == 0
    L = args.tile_cells or (1024 if w.batch == 1 else 512)
    sbytes = stage_model_bytes(w, info, own_fft, L)
    fused23 = own_fft and info["n"] >= 1 << 20 and stage["fft_pass3"] == 0.0 and stage["fft_pass2"] > 0.0 and w.dtype == "f64"
    if fused23:                                           # the library reports the fused kernel's time as pass 2
        stage["fft_pass23"] = stage.pop("fft_pass2")
        stage.pop("fft_pass3")
    two_pass = own_fft and (info["n"] <= 65536 or (n5 and info["n"] <= 5 << 16))      # R1 x 256: there is no middle pass
    fft_stages = ["fft_pass1", "fft_pass23"] if fused23 else ["fft_pass1", "fft_pass3"] if two_pass else ["fft_pass1", "fft_pass2", "fft_pass3"]
    own_stages = ["stats", "sort", "premul", "spread", "assemble"] + (fft_stages if own_fft else [])
    dom = max(own_stages, key=lambda k: stage[k])      # the dominant OWN kernel (cuFFT, when used, is a library)
    ach = sbytes[dom] / (stage[dom] * 1e-3) / 1e9
    path_ms = stage["total"] - stage["fft"]
    path_ach = info["model_bytes"] / (path_ms * 1e-3) / 1e9
    path_sparse = info["model_bytes"] - (info["M"] * info["n"] * 2 * (8 if w.dtype == "f64" else 4) - (sbytes["spread"] - 2 * w.Nd * 4 * (8 if w.dtype == "f64" else 4) - info["M"] * w.Nd * (8 if w.dtype == "f64" else 4)))
    traffic, traffic_cap = measured_traffic(dom, w, info)
    Bi = ht.numel() * ht.element_size() + hy.numel() * hy.element_size() + hdy.numel() * hdy.element_size()
    Bo = hP.numel() * hP.element_size()
    line = {
        "metric": METRIC, "value": value, "unit": "ms", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": w.dtype, "data": "synthetic",
        "config": config_dict(w, {"sigma": info["sigma"], "w": info["w"], "n": info["n"], "M": info["M"]}),
        "nu_pts_per_s": info["M"] * w.Nd * world / (stage["spread"] * 1e-3),
        "nu_pts_per_s_whole": info["M"] * w.Nd * world / (ms_per_step * 1e-3),
        "freqs_per_s": w.Nf * n_periodograms / (ms_per_step * 1e-3),
        "stage_ms": stage, "wall_ms_per_step_incl_flush": wall / args.steps * 1e3,
        "step_ms_min": float(np.min(step_ms)), "step_ms_median": float(np.median(step_ms)),
        "roofline": {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                     "traffic": traffic, "traffic_capture": traffic_cap, "peak_source": peak_src, "algorithmic_bytes": sbytes[dom],
                     "kernel_ms": stage[dom],
                     "per_kernel": {k: {"ms": stage[k], "algorithmic_bytes": sbytes[k],
                                        "frac": sbytes[k] / (stage[k] * 1e-3) / 1e9 / peak if stage[k] > 0 else None}
                                    for k in own_stages},
                     **({"note": "fft_pass23 = FFT passes 2 + 3 fused through L2 (TMA tile loads, mbarrier ring): its algorithmic "
                                 "bytes are half of the two separate passes' (the intermediate never reaches HBM); the kernel "
                                 "is bound by its consumers' shared-memory traffic (profiles/r2_cfg3.md, r2_experiments.md); "
                                 "stage times come from a second, event-recording plan with the same kernels (direct launches), "
                                 "`value` from graph replay of the user-facing plan"} if fused23 else {})},
        "path_roofline": {"what": "the north_star figure: spread + deconvolve + assembly path = all own kernels except the FFT "
                                  "(total - fft).  HEADLINE = for the bytes actually moved (bytes_moved: inputs, sort permutation, "
                                  "the spreading tiles that hold points, kept modes, power); the dense streaming model of "
                                  + STAGE_BYTES_DOC + " (every grid cell written once) is the labelled secondary figure",
                          "ms": path_ms, "unit": "GB/s",
                          "bytes_moved": path_sparse, "achieved": path_sparse / (path_ms * 1e-3) / 1e9,
                          "frac_bytes_moved_of_measured": path_sparse / (path_ms * 1e-3) / 1e9 / peak,
                          "frac_bytes_moved_of_8TBs": path_sparse / (path_ms * 1e-3) / 1e9 / 8000.0,
                          "target_50pct_met": bool(path_sparse / (path_ms * 1e-3) / 1e9 / peak >= 0.5),
                          "dense_model": {"bytes": info["model_bytes"], "achieved": path_ach, "frac_of_measured": path_ach / peak,
                                          "frac_of_8TBs": path_ach / 8000.0}},
        "fft_ms": stage["fft"],
        "fft": {"impl": "cuFFT" if ffts else "own three radix-256 passes (first pruned by the spreading kernel's "
                                             "liveness masks)" + ("; in `value` the last is fused with the assembly"
                                                                if args.fft_impl == 2 else "")
                                             + ("; passes 2 + 3 are one persistent kernel whose intermediate stays in "
                                                "L2 and is discarded, not written back" if fused23 else ""),
                "ms": stage["fft"], "grid_bytes": info["M"] * info["n"] * 2 * (8 if w.dtype == "f64" else 4),
                "grid_passes_at_measured_peak": stage["fft"] * 1e-3 * peak * 1e9
                / (2.0 * info["M"] * info["n"] * 2 * (8 if w.dtype == "f64" else 4))},
        "e2e": {"value": e2e_ms / args.steps / n_periodograms, "unit": "ms", "h2d_bytes_per_step": Bi,
                "d2h_bytes_per_step": Bo, "plan": e2e_plan, "max_abs_diff_vs_device_leg": e2e_diff},
        "gpu_launches": own * args.steps, "own_kernels_per_step": own, "cufft_execs_per_step": ffts,
        "clocks": clocks,
    }
    if args.parity_k > 0:
        # The output of the plan that was TIMED (same launch configuration: side stream, graph replay), checked after the
        # timed loop against the oracle's direct sums on sampled frequencies (peak and seam included): the paper's error
        # metric (pointwise relative error, median / 99th percentile) next to the gate's E_inf (A8).
        import oracle
        from paper_2409_08090_b200.workloads import compare_indices
        P.fill_(float("nan"))
        with torch.cuda.stream(side):
            plan.execute(t, y, dy, P, stream)
        side.synchronize()
        ks = compare_indices(w, args.parity_k)
        nser = min(w.batch, 2)
        Pg = P[:nser].cpu().numpy().astype(np.float64)[:, ks]
        Po = np.stack([oracle.direct(w.t, w.y[b], w.dy, w.f0, w.df, w.Nf, k=ks) for b in range(nser)])
        d = np.abs(Pg - Po)
        rel = d / np.maximum(Po, 1e-300)
        gate = 1e-8 if w.dtype == "f64" else 1e-4
        line["parity"] = {"against": "oracle.direct (strict)", "K": int(ks.size), "series": nser,
                          "Einf": float((d.max(axis=1) / Po.max(axis=1)).max()), "median": float(np.median(rel)),
                          "p99": float(np.percentile(rel, 99)), "max": float(rel.max()), "gate_Einf": gate,
                          "ok": bool((d.max(axis=1) / Po.max(axis=1)).max() <= gate and np.all(np.isfinite(Pg)))}
    if not args.no_cpu_baseline and world == 1:
        import oracle
        cores = oracle.num_threads()
        K = args.cpu_freqs or auto_cpu_freqs(w, cores)
        dt, ms_full, nser, kk = time_oracle(w, K)
        line["cpu_baseline"] = {"value": ms_full, "unit": "ms", "cores": cores, "kind": "oracle",
                                "sample": f"{kk} of {w.Nf} frequencies x {nser} of {w.batch} series in {dt:.1f} s "
                                          f"(oracle.direct, strict), extrapolated linearly to the full grid"}
    print(json.dumps(line), flush=True)
    plan.close()
    plan_t.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.traffic_from:
        write_traffic(a.traffic_from, a.traffic_meta, a.traffic_command)
    elif a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
