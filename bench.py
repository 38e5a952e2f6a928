#!/usr/bin/env python
"""bench.py -- headline metric of BASELINE.json on one node.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config 4]

metric: "PSF-conv metric applies/s at 4096^2 (8192^2 padded)".  A step is one fused PSF-convolution
metric apply y = s . C(s . x) ("L1 apply") on BASELINE.json configs[3] (4096^2 single
channel) -- three kernels (row R2C, column FFT.W.iFFT, row C2R).  The same run also times the latent
metric apply, one energy+gradient and a CG iteration (reported under "extra"), the dominant kernel
alone for the roofline, the end-to-end call with host buffers, and the fp64 oracle on the host cores.
Single-channel configs do not shard: --gpus N runs N independent replicas, one process
per GPU (started here through torch.distributed.run when the caller has not already done so).  The multi-channel
config does shard: `--config 5 --shard channels` times the channel-sharded latent metric apply and CG iteration
(ChannelShard: one NCCL all-reduce per apply), strong scaling.

The timed operator is the N' = R' limit of the paper's Eq. 9 (E = 1/2 s^T C s - j^T s, metric J^T C J, R1);
with the separately fitted noise kernel of Eq. 15-18 (frs_set_noise_kernel + frs_set_likelihood(1)) a latent metric apply
is three convolutions; its time is reported under "extra" (eq9_metric_apply_ms).
"""
from __future__ import annotations

import argparse
import json
import os
import socket
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


def byte_models(ny, nx):
    """Minimal-pass algorithmic bytes of the operators bench.py times beside the headline (single channel, one field, fp32;
    BASELINE.md section 3 derives each).  img = one image, hl = the half spectrum of an UNPADDED image (latent Hartley
    passes), half = the pruned padded spectrum, what = the real PSF weights."""
    img = ny * nx * 4
    hl = ny * (nx // 2 + 1) * 8
    half = ny * (nx + 1) * 8
    what = (2 * ny) * (nx + 1) * 4
    k1 = img + hl                      # .A + first Hartley pass
    k2 = hl + img + half               # second Hartley pass + .s + pad + row R2C
    k3 = 2 * half + what               # column FFT . W . iFFT
    k4 = half + img + hl               # row C2R + crop + .s + first Hartley pass
    k5 = hl + 2 * img                  # second Hartley pass + .A + v
    l2 = k1 + k2 + k3 + k4 + k5
    # Eq. 9 (reading R14): between the two convolutions the periodic N'^-1 on the unpadded grid -- row C2R + crop fused
    # with the N-point row R2C (half -> hl), column FFT . K^-1 . iFFT (2 hl + the real half-plane of K^-1), row C2R fused
    # with pad + row R2C of the second convolution (hl -> half)
    ninv = (half + hl) + (2 * hl + hl // 2) + (hl + half)
    eq9 = k1 + k2 + k3 + ninv + k3 + k4 + k5
    # energy + gradient (mode 0): sky forward (k1, then the second pass writes s and the padded row spectrum), k3,
    # row C2R + (C s - j) . s + first Hartley pass (reads s and j), second pass + .A + xi
    eg = k1 + (hl + img + half) + k3 + (half + 2 * img + hl) + k5
    return {"latent_metric_apply": l2, "ms_per_cg_iter": l2 + 7 * img, "ms_per_cg_iter_plain_launches": l2 + 7 * img,
            "energy_grad": eg, "eq9_metric_apply": eq9,
            # joint (xi, theta): the prologue reads xi beside dxi (A and dA come from a few thousand bins), the
            # epilogue reads xi again for the bin sums of xi . h
            "joint_metric_apply": l2 + 2 * img, "joint_energy_grad": eg + 2 * img,
            # one position of the sample-averaged KL metric: a sky evaluation (k1 + second pass writing s) + an apply
            "kl_metric_apply_per_position": (k1 + hl + img) + l2}


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
            t0 = time.time()                      # nvidia-smi needs a moment to start: wait for its first line
            while not self.lines and time.time() - t0 < 3.0:
                time.sleep(0.01)
            self.n0 = len(self.lines)
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self, load=None, sync=None):
        """load/sync: the timed step and a device synchronise.  The timed region of the default run is shorter than
        a few sampling periods (20 ms), so the very same step loop keeps running, untimed, for another 0.4 s while
        the sampler goes on: the clocks reported are those of this kernel sequence under load."""
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        window = "timed region"
        if load is not None:
            t_end, i = time.time() + 0.4, 0
            while time.time() < t_end:
                for _ in range(16):
                    load(i)
                    i += 1
                sync()
            window = "timed region + 0.4 s of the same step loop (untimed)"
        else:
            time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        for l in self.lines[getattr(self, "n0", 0):]:
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
                "reasons": sorted(reasons), "samples": len(sm), "window": window}


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
    # ---- the timed operator must be the operator: symmetry <x1, A x0> = <A x1, x0> and positivity <x0, A x0> >= 0 of
    # A = s . C (s . ) on this very configuration (the oracle comparison at this size lives in tests/, minutes of CPU)
    y1 = ctx.new_image()
    ctx.sky_metric_apply(xs[0], y)
    ctx.sky_metric_apply(xs[1], y1)
    d01, d10 = float((xs[1].double() * y.double()).sum()), float((y1.double() * xs[0].double()).sum())
    d00 = float((xs[0].double() * y.double()).sum())
    stripped = b"ATTRIBUTION BUILD" in frs.lib().frs_version()     # FRS_STRIP build: wrong results by construction, times only
    assert stripped or (abs(d01 - d10) <= 1e-4 * max(abs(d01), abs(d10), 1e-300) and d00 > 0.0), ("L1 apply not symmetric PSD", d01, d10, d00)
    del y1
    # ---- headline: K L1 applies, inputs resident in HBM
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ms = timed(step, args.steps, args.warmup)
    launches = ctx.launch_count() - l_after_warmup
    clocks = sampler.stop(step, torch.cuda.synchronize) if rank == 0 else None
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
    traffic, traffic_src = None, None
    tpath = os.path.join(ROOT, "profiles", "traffic_conv_cols.json")
    if os.path.exists(tpath) and args.config == 4:
        tj = json.load(open(tpath))
        traffic = tj.get("dram_bytes_per_launch")
        traffic_src = "from " + tj.get("source", "profiles/") + " -- an ncu capture of this kernel, NOT measured in this run"
    roofline = {"bound": "hbm", "kernel": "conv_cols_dif_kernel (column FFT . W . iFFT)", "achieved": ach, "peak": peak,
                "unit": "GB/s", "frac": ach / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": b_f2, "ms_per_launch": f2_ms,
                "pass_ms": {k: v[0] / max(1, v[1]) for k, v in prof.items() if v[1]}}
    # the co-binding roof of the same kernel: FP32 pipe slots.  One slot = one fp32 add / mul /
    # fma per lane (a packed FADD2 / FMUL2 / FFMA2 counts two).  Slots per thread and column: the SASS instruction mix of
    # conv_cols_dif_kernel<4096> kept in profiles/sass_mix_conv_cols.json (cuobjdump count, command inside); 256 threads
    # per column; peak = SMs x 128 lanes x SM clock.
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    fp_peak = sms * 128 * (clocks["sm_mhz"] if clocks and clocks.get("sm_mhz") else 1965.0) * 1e6 / 1e12
    fp_ach, slots = None, None
    spath = os.path.join(ROOT, "profiles", "sass_mix_conv_cols.json")
    if os.path.exists(spath) and w.ny == 4096:
        slots = float(json.load(open(spath))["fp32_lane_ops_per_thread_per_column"])
        fp_ach = slots * 256 * (w.nx + 1) * w.nchan / (f2_ms * 1e-3) / 1e12
    roofline_fp32 = {"bound": "alu", "kernel": "conv_cols_dif_kernel", "achieved": fp_ach, "peak": fp_peak, "unit": "T fp32 lane-ops/s",
                     "frac": (fp_ach / fp_peak) if fp_ach else None, "lane_ops_per_thread_per_column": slots,
                     "peak_source": "148 SMs x 128 fp32 lanes x SM clock sampled during the run (B200_PROFILING.md unit counts)"}
    ach_step = b_l1 / (ms_step * 1e-3) / 1e9
    roofline_step = {"what": "whole L1 apply (3 kernels), minimal 3-pass byte model", "bytes": b_l1, "achieved": ach_step,
                     "unit": "GB/s", "frac_of_measured_peak": ach_step / peak, "frac_of_nominal_8TBs": ach_step / 8000.0}

    # ---- end to end: host buffers, copies inside the timed region.  Two public calls: one apply per call (copy in,
    # three kernels, copy out, synchronise) and the batch call, which overlaps the copies of neighbouring items with the
    # kernels (every item still crosses the bus both ways inside the timed region).  `value` is the batch call.
    n_e2e = max(4, min(args.steps, 20))
    xh = [torch.from_numpy(np.ascontiguousarray(x.cpu().numpy())).pin_memory() for x in xs]
    yh = [torch.empty_like(xh[0]).pin_memory() for _ in range(2)]
    barrier()
    for i in range(2):
        ctx.sky_metric_apply_host(xh[i & 1], yh[0])
    ctx.sky_metric_apply_host_batch([xh[i & 1] for i in range(4)], [yh[i & 1] for i in range(4)])
    assert stripped or (torch.equal(yh[0], yh[1]) is False and torch.isfinite(yh[1]).all())
    ctx.sky_metric_apply_host(xh[1], yh[0])
    assert stripped or torch.equal(yh[0], yh[1]), "batched and single host applies disagree"
    barrier()
    t0 = time.perf_counter()
    for i in range(n_e2e):
        ctx.sky_metric_apply_host(xh[i & 1], yh[0])
    torch.cuda.synchronize()
    t_single = time.perf_counter() - t0
    barrier()
    t0 = time.perf_counter()
    ctx.sky_metric_apply_host_batch([xh[i & 1] for i in range(n_e2e)], [yh[i & 1] for i in range(n_e2e)])
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - t0
    if world > 1:
        t = torch.tensor([t_e2e, t_single], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        t_e2e, t_single = float(t[0].item()), float(t[1].item())
    nbytes = xs[0].numel() * 4
    e2e = {"value": world * n_e2e / t_e2e, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
           "steps": n_e2e, "call": "frs_sky_metric_apply_host_batch (pinned host buffers; copies of neighbouring items overlap the kernels)",
           "one_apply_per_call": {"value": world * n_e2e / t_single, "call": "frs_sky_metric_apply_host"}}

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
            iters = 20
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ctx.cg_solve(b, sol, iters)                                    # warm-up: also builds the iteration graph
            sol.zero_()
            e0.record()
            ctx.cg_solve(b, sol, iters)
            e1.record()
            torch.cuda.synchronize()
            extra["ms_per_cg_iter"] = e0.elapsed_time(e1) / (iters + 1)   # + the initial M x0 apply
            ctx.set_cuda_graphs(False)                                     # the same solve with plain launches
            ctx.cg_solve(b, sol, 2)
            sol.zero_()
            e0.record()
            ctx.cg_solve(b, sol, iters)
            e1.record()
            torch.cuda.synchronize()
            extra["ms_per_cg_iter_plain_launches"] = e0.elapsed_time(e1) / (iters + 1)
            ctx.set_cuda_graphs(True)
            # the paper's literal likelihood (Eq. 9 with the fitted noise kernel): J^T C N'^-1 C J + 1
            ctx.set_noise_kernel(1e-2 * float(np.sum(w.w_half[0][:, 0]) + 2 * np.sum(w.w_half[0][:, 1:-1]) + np.sum(w.w_half[0][:, -1])))
            ctx.set_likelihood(1)
            m = timed(lambda i: ctx.metric_apply(v, out, True), k2, 3)
            extra["eq9_metric_apply_ms"] = m / k2
            ctx.set_likelihood(0)
            if w.nchan == 1:
                # learned amplitude spectrum (NEXT-3, reading R17): joint (xi, theta) energy + gradient and metric apply
                ctx.set_amplitude_model((float(w.mu[0]), 1.0, 0.1, 1.0, 0.3, -3.0, 0.2, 0.5, 0.2, 0.2, 0.1))
                th = dev(0.3 * rng.normal(size=ctx.ntheta))
                gth, oth = torch.empty_like(th), torch.empty_like(th)
                m = timed(lambda i: ctx.energy_grad_joint(xi, th, g, gth, True), k2, 3)
                extra["joint_energy_grad_ms"] = m / k2
                dth = dev(rng.normal(size=ctx.ntheta))
                m = timed(lambda i: ctx.metric_apply_joint(v, dth, out, oth, True), k2, 3)
                extra["joint_metric_apply_ms"] = m / k2
                extra["joint_ntheta"] = int(ctx.ntheta)

                # sample-averaged KL metric (reading R15) on one mirrored sample = two positions, each a sky evaluation + an apply
                ctx.set_amplitude(dev(w.amp), w.mu)
                smp = dev(0.1 * rng.normal(size=(1, w.nfield, w.ny, w.nx)))
                m = timed(lambda i: ctx.kl_metric_apply(xi, smp, v, out, True), k2, 2)
                extra["kl_metric_apply_per_position_ms"] = m / k2 / 2
                ctx.sky_forward(xi)
            if w.nchan == 1 and w.nfield == 1:
                # byte model and fraction of the measured HBM peak beside every time above
                bm = byte_models(w.ny, w.nx)
                for key, nbytes in bm.items():
                    tkey = key if key.startswith("ms_per") else key + "_ms"
                    if tkey in extra:
                        extra[key + "_bytes"] = nbytes
                        extra[key + "_frac_of_measured_peak"] = nbytes / (extra[tkey] * 1e-3) / 1e9 / peak

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
                       "operator": "N' = R' limit of Eq. 9 (E = 1/2 s^T C s - j^T s): one padded PSF convolution per apply",
                       "parallelism": f"replicas x{world} (single-channel path does not shard), one process per GPU"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "roofline_step": roofline_step, "roofline_fp32": roofline_fp32,
            "cpu_baseline": cpu, "extra": extra}
    if stripped:
        line["invalid"] = frs.lib().frs_version().decode() + " -- NOT a bench value: read roofline.pass_ms only"
        line["value"] = None
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ----------------------------------------------------------------------------------------- sharded arm (config 5)
def run_sharded(args):
    """--config 5 --shard channels: the 16 channels are partitioned over the ranks (ChannelShard), the latent vectors are
    replicated, every latent metric apply / CG iteration ends in ONE NCCL all-reduce of a latent-sized vector."""
    import torch
    import torch.distributed as dist
    import paper_2406_09144_b200 as frs
    from paper_2406_09144_b200.parallel import ChannelShard
    from gen import workloads as wl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if not dist.is_initialized():
        if world == 1:
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", str(_free_port()))
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", local))
    frs.load_library()
    w = wl.make_config(5, seed=0)                        # the SAME problem on every rank; each keeps its channels
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a, np.float32)).cuda()  # noqa: E731
    sh = ChannelShard(w.ny, w.nx, w.nchan, w.lognu)
    sh.set_psf_weights(dev(w.w_half))
    sh.set_dirty(dev(w.dirty))
    sh.set_amplitude(dev(w.amp), w.mu)
    rng = np.random.default_rng(100)
    xi = dev(0.5 * rng.normal(size=(w.nfield, w.ny, w.nx)))
    g = torch.empty_like(xi)
    sh.energy_grad(xi, g, True)                          # sets the position
    v, out = dev(rng.normal(size=(w.nfield, w.ny, w.nx))), torch.empty_like(xi)

    def barrier():
        dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, warmup):
        for i in range(warmup):
            fn(i)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(steps):
            fn(i)
        e1.record()
        barrier()
        t = torch.tensor([e0.elapsed_time(e1)], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = sh.ctx.launch_count()
    ms = timed(lambda i: sh.metric_apply(v, out, True), args.steps, args.warmup)
    launches = (sh.ctx.launch_count() - l0) * args.steps // (args.steps + args.warmup)
    clocks = sampler.stop() if rank == 0 else None
    b = (-g).contiguous()
    x = torch.zeros_like(b)
    iters = 10
    ms_cg = timed(lambda i: sh.cg_solve(b, x, iters, True), 2, 1) / (2 * iters)
    if rank == 0:
        line = {"metric": "16-channel latent metric applies/s at 1024^2 (2048^2 padded), channel-sharded", "value": args.steps / (ms * 1e-3),
                "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
                "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": f"config5: {w.nchan} x {w.ny}x{w.nx}, two latent fields; one step = frs_metric_apply on "
                                       f"{len(sh.channels)} of {w.nchan} channels per rank + ONE all-reduce (NCCL) of {w.nfield} x {w.ny}x{w.nx} fp32",
                           "l2": "no flush: a step streams > 1 GB per rank at world 1",
                           "parallelism": f"channels sharded x{world} (ChannelShard), latent vectors replicated"},
                "clocks": clocks, "gpu_launches": int(launches), "extra": {"ms_per_cg_iter": ms_cg}}
        print(json.dumps(line), flush=True)
    dist.destroy_process_group()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher: start N ranks (one process per GPU) through torch.distributed.run,
    exactly as the driver would, and hand its exit code back.  Rank 0 prints the single JSON line."""
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")                         # keep NCCL's communicator log (transport, NVLS) ...
    env.setdefault("NCCL_DEBUG_FILE", os.path.join(ROOT, "gpurun_out", "nccl_%h_%p.log"))   # ... out of the JSON line
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--shard", default="none", choices=["none", "channels"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    if args.impl == "reference":
        run_reference(args)                              # rank 0 alone runs the oracle; other ranks exit 0
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args))
    elif args.shard == "channels":
        if args.config != 5:
            sys.exit("--shard channels needs --config 5 (single-channel configs do not shard, DESIGN.md Multi-GPU)")
        run_sharded(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
