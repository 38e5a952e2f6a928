#!/usr/bin/env python
"""bench.py -- headline metric of BASELINE.json on one node.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config 4]

metric: "PSF-conv metric applies/s at 4096^2 (8192^2 padded)".  A step is one fused PSF-convolution
metric apply y = s . C(s . x) ("L1 apply") on BASELINE.json configs[3] (4096^2 single
channel) -- three kernels (row R2C, column FFT.W.iFFT, row C2R).  The same run also times the latent
metric apply, one energy+gradient and a CG iteration (reported under "extra"), the dominant kernel
alone for the roofline, the end-to-end call with host buffers, and the fp64 oracle on the host cores.
Single-channel configs do not shard: --gpus N runs N independent replicas.
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

METRIC = "PSF-conv metric applies/s at 4096^2 (8192^2 padded)"
UNIT = "applies/s"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def bytes_l1(ny, nx, nchan=1):
    """Algorithmic bytes of one L1 apply: SURVEY 8(d) table (F1 + F2 + F3), fp32, real W."""
    n2 = ny * nx
    half = ny * (nx + 1) * 8                    # pruned intermediate N (M/2+1) complex64
    what = (2 * ny) * (nx + 1) * 4              # W real M (M/2+1)
    f1 = 2 * n2 * 4 + half
    f2 = half + what + half
    f3 = half + n2 * 4 + n2 * 4
    return nchan * (f1 + f2 + f3), nchan * f2


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "20"], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                mx.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ----------------------------------------------------------------------------------------- oracle arm
def oracle_l1_sample(n_s, reps, seed=0):
    """Time the oracle's L1 apply, as it stands, at n_s x n_s (config-4 recipe at reduced size)."""
    from gen import workloads as wl
    from oracle import frs_oracle as o
    w = wl.make_config(4, n=n_s, seed=seed)
    rng = np.random.default_rng(1)
    s = np.exp(0.5 * rng.normal(size=(1, n_s, n_s)))
    x = rng.normal(size=(1, n_s, n_s))
    o.sky_metric_apply(w.w_half, s, x)
    ts = []
    for _ in range(reps):
        t0 = time.perf_counter()
        o.sky_metric_apply(w.w_half, s, x)
        ts.append(time.perf_counter() - t0)
    return ts


def scale_to_full(n_s, n_full=4096):
    """FFT work ratio between the sample and the full size: N^2 log2(2N)."""
    return (n_full / n_s) ** 2 * np.log2(2 * n_full) / np.log2(2 * n_s)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    total = args.steps + args.warmup
    n_s = 4096 if total <= 40 else (2048 if total <= 160 else (1024 if total <= 600 else 512))
    ts = oracle_l1_sample(n_s, total)
    ts = ts[args.warmup:]
    sc = scale_to_full(n_s)
    t_step = float(np.mean(ts)) * sc
    val = 1.0 / t_step
    cores = 1
    sample = (f"oracle.sky_metric_apply (numpy fp64) at {n_s}^2 (padded {2 * n_s}^2), config-4 recipe; per-step time scaled "
              f"to 4096^2 by the FFT work ratio N^2 log2(2N) = x{sc:.1f}")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t_step * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "config4: 4096x4096 single channel, padded 8192^2 (oracle on a bounded sample)"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------- CUDA arm
def run_cuda(args):
    import torch
    import torch.distributed as dist
    import paper_2406_09144_b200 as frs
    from gen import workloads as wl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    frs.load_library()

    w = wl.make_config(args.config, seed=rank)           # replicas: one independent problem per rank
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a, np.float32)).cuda()  # noqa: E731
    ctx = frs.Context(w.ny, w.nx, w.nchan, device=local)
    ctx.set_psf_weights(dev(w.w_half))
    ctx.set_dirty(dev(w.dirty))
    ctx.set_amplitude(dev(w.amp), w.mu)
    ctx.set_channel_lognu(w.lognu)
    rng = np.random.default_rng(100 + rank)
    xi = dev(0.5 * rng.normal(size=(w.nfield, w.ny, w.nx)))
    ctx.sky_forward(xi)
    xs = [dev(rng.normal(size=(w.nchan, w.ny, w.nx))) for _ in range(2)]
    y = ctx.new_image()

    l_after_warmup = 0

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, warmup):
        for i in range(warmup):
            fn(i)
        barrier()
        nonlocal l_after_warmup
        l_after_warmup = ctx.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(steps):
            fn(i)
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        if world > 1:
            t = torch.tensor([ms], device="cuda", dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms

    step = lambda i: ctx.sky_metric_apply(xs[i & 1], y)  # noqa: E731
    # ---- headline: K L1 applies, inputs resident in HBM
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ms = timed(step, args.steps, args.warmup)
    launches = ctx.launch_count() - l_after_warmup
    clocks = sampler.stop() if rank == 0 else None
    ms_step = ms / args.steps
    value = world * args.steps / (ms * 1e-3)

    # ---- dominant kernel alone (CUDA events around each pass, on the ctx's stream)
    ctx.profile_enable(True)
    for i in range(args.steps):
        step(i)
    prof = ctx.profile_read()
    ctx.profile_enable(False)
    b_l1, b_f2 = bytes_l1(w.ny, w.nx, w.nchan)
    peak, peak_src = peaks()
    f2_ms = prof["conv_cols"][0] / max(1, prof["conv_cols"][1])
    ach = b_f2 / (f2_ms * 1e-3) / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic_conv_cols.json")
    if os.path.exists(tpath):
        traffic = json.load(open(tpath)).get("dram_bytes_per_launch")
    roofline = {"bound": "hbm", "kernel": "conv_cols_kernel (column FFT . W . iFFT)", "achieved": ach, "peak": peak,
                "unit": "GB/s", "frac": ach / peak, "traffic": traffic, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": b_f2, "ms_per_launch": f2_ms,
                "pass_ms": {k: v[0] / max(1, v[1]) for k, v in prof.items() if v[1]}}
    # the co-binding roof of the same kernel: FP32 pipe slots.  One slot = one fp32
    # add / mul / fma per lane (a packed FFMA2 counts two); conv_cols executes 2759 slots per thread and column
    # (SASS count at NF = 4096: 1220 packed + 319 scalar), 256 threads per column; peak = SMs x 128 lanes x clock.
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    fp_peak = sms * 128 * (clocks["sm_mhz"] if clocks and clocks.get("sm_mhz") else 1965.0) * 1e6 / 1e12
    fp_ach = 2759.0 * 256 * (w.nx + 1) * w.nchan * (w.ny / 4096.0) / (f2_ms * 1e-3) / 1e12 if w.ny == 4096 else None
    roofline_fp32 = {"bound": "alu", "kernel": "conv_cols_kernel", "achieved": fp_ach, "peak": fp_peak, "unit": "T fp32 lane-ops/s",
                     "frac": (fp_ach / fp_peak) if fp_ach else None,
                     "peak_source": "148 SMs x 128 fp32 lanes x SM clock sampled during the run (B200_PROFILING.md unit counts)"}
    ach_step = b_l1 / (ms_step * 1e-3) / 1e9
    roofline_step = {"what": "whole L1 apply (3 kernels), minimal 3-pass byte model", "bytes": b_l1, "achieved": ach_step,
                     "unit": "GB/s", "frac_of_measured_peak": ach_step / peak, "frac_of_nominal_8TBs": ach_step / 8000.0}

    # ---- end to end: host buffers, copies inside the timed region
    n_e2e = max(3, min(args.steps, 20))
    xh = [torch.from_numpy(np.ascontiguousarray(x.cpu().numpy())).pin_memory() for x in xs]
    yh = torch.empty_like(xh[0]).pin_memory()
    barrier()
    for i in range(2):
        ctx.sky_metric_apply_host(xh[i & 1], yh)
    barrier()
    t0 = time.perf_counter()
    for i in range(n_e2e):
        ctx.sky_metric_apply_host(xh[i & 1], yh)
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - t0
    if world > 1:
        t = torch.tensor([t_e2e], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        t_e2e = float(t.item())
    nbytes = xs[0].numel() * 4
    e2e = {"value": world * n_e2e / t_e2e, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
           "steps": n_e2e, "call": "frs_sky_metric_apply_host (pinned host buffers)"}

    # ---- the rest of the hot path (extra; same run)
    extra = {}
    if rank == 0:
        v = dev(rng.normal(size=(w.nfield, w.ny, w.nx)))
        out = ctx.new_latent()
        k2 = max(5, args.steps // 4)
        m = timed(lambda i: ctx.metric_apply(v, out, True), k2, 3) if world == 1 else None
        if m is not None:
            extra["latent_metric_apply_ms"] = m / k2
            g = ctx.new_latent()
            m = timed(lambda i: ctx.energy_grad(xi, g, True, host_energy=False), k2, 3)
            extra["energy_grad_ms"] = m / k2
            b = (-g).contiguous()
            sol = torch.zeros_like(b)
            iters = 10
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ctx.cg_solve(b, sol, 2)
            sol.zero_()
            e0.record()
            ctx.cg_solve(b, sol, iters)
            e1.record()
            torch.cuda.synchronize()
            extra["ms_per_cg_iter"] = e0.elapsed_time(e1) / (iters + 1)   # + the initial M x0 apply

    if world > 1:
        dist.barrier()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- oracle on the host cores, bounded sample
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        n_s = w.ny if w.nchan == 1 else 2048
        ts = oracle_l1_sample(n_s, 3)
        sc = scale_to_full(n_s, w.ny)
        tfull = float(np.mean(ts)) * sc
        cpu = {"value": 1.0 / tfull, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"3 oracle L1 applies (numpy fp64, as it stands) at {n_s}^2 (padded {2 * n_s}^2), config-4 recipe, "
                         f"scaled to {w.ny}^2 by N^2 log2(2N) = x{sc:.2f}; host cpu_count={os.cpu_count()}"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": f"config{args.config}: {w.ny}x{w.nx} x{w.nchan}ch, padded {2 * w.ny}x{2 * w.nx}; one step = "
                                   "frs_sky_metric_apply y = s.C(s.x)",
                       "l2": "no flush: a step streams 0.94 GB (inputs 2 x 67 MB rotated, 134 MB spectrum, 134 MB weights) "
                             ">> 126 MB L2",
                       "parallelism": f"replicas x{world} (single-channel path does not shard)"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "roofline_step": roofline_step, "roofline_fp32": roofline_fp32,
            "cpu_baseline": cpu, "extra": extra}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
