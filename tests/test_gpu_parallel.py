"""The channel-sharded path (paper_2406_09144_b200/parallel.py) with the REAL CUDA context and NCCL, world size 1 on one
GPU: ChannelShard -> Context -> frs_cg_step_begin -> all_reduce (NCCL, on the ctx's stream) -> frs_cg_step_end, against the
fp64 oracle on all channels.  (World size 2 over gloo, against an oracle-backed stand-in: tests/test_parallel_gloo.py.)"""
import os
import socket

import numpy as np
import pytest

from gen import workloads as wl
from oracle import frs_oracle as o

pytestmark = pytest.mark.gpu


def rel(a, b):
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.fixture(scope="module")
def nccl_world1():
    import torch
    import torch.distributed as dist
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    created = False
    if not dist.is_initialized():
        with socket.socket() as s:
            s.bind(("127.0.0.1", 0))
            port = s.getsockname()[1]
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ["MASTER_PORT"] = str(port)
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
        created = True
    yield dist
    if created:
        dist.destroy_process_group()


def test_channel_shard_real_context_nccl_world1(nccl_world1):
    import torch
    import paper_2406_09144_b200 as frs
    from paper_2406_09144_b200.parallel import ChannelShard
    frs.load_library()
    w = wl.make_config(5, n=64, nchan=4)                        # reduced config 5: 4 channels, two latent fields
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a, np.float32)).cuda()  # noqa: E731
    sh = ChannelShard(w.ny, w.nx, w.nchan, w.lognu)
    assert list(sh.channels) == [0, 1, 2, 3] and sh.world == 1
    sh.set_psf_weights(dev(w.w_half))
    sh.set_dirty(dev(w.dirty))
    sh.set_amplitude(dev(w.amp), w.mu)
    xi = (0.3 * np.random.default_rng(3).normal(size=(2, w.ny, w.nx))).astype(np.float32)
    g = torch.empty((2, w.ny, w.nx), device="cuda")
    e = sh.energy_grad(dev(xi), g, with_prior=True)
    e_ref, g_ref = o.energy_grad(w.w_half, w.dirty, w.amp, w.mu, w.lognu, xi, True)
    assert abs(e - e_ref) <= 1e-5 * abs(e_ref)
    assert rel(g.cpu().numpy(), g_ref) <= 1e-5
    v = np.random.default_rng(4).normal(size=(2, w.ny, w.nx)).astype(np.float32)
    out = torch.empty_like(g)
    sh.metric_apply(dev(v), out, with_prior=True)
    s64 = o.sky(xi, w.amp, w.mu, w.lognu)
    ap = lambda u: o.metric_apply(w.w_half, w.amp, w.mu, w.lognu, xi, u, True, s=s64)  # noqa: E731
    assert rel(out.cpu().numpy(), ap(v)) <= 1e-5
    # the split CG iteration with the collective between its halves (multi-channel, two fields: jvp/vjp combine path)
    b = (-g).contiguous()
    x = torch.zeros_like(b)
    rn = sh.cg_solve(b, x, 3, with_prior=True)
    ref = o.cg(ap, b.cpu().numpy().astype(np.float64), max_iter=3)
    assert rel(x.cpu().numpy(), ref["x"]) <= 1e-4
    assert abs(rn - ref["res"][-1]) <= 1e-3 * ref["res"][-1]


def test_sample_shard_real_context_nccl_world1(nccl_world1):
    """MGVI samples over ranks (SampleShard) with the real context and NCCL at world size 1: draw -> KL energy / gradient
    -> all_reduce -> KL metric, against the oracle running on the GPU's noise kernel and the GPU's own samples."""
    import torch
    import paper_2406_09144_b200 as frs
    from paper_2406_09144_b200.parallel import SampleShard
    frs.load_library()
    w = wl.make_config(1, n=64, sigma_rel=0.1)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a, np.float32)).cuda()  # noqa: E731
    ctx = frs.Context(w.ny, w.nx, 1)
    ctx.set_psf_weights(dev(w.w_half))
    ctx.set_dirty(dev(w.dirty))
    ctx.set_amplitude(dev(w.amp), w.mu)
    ctx.set_noise_kernel(1e-2 * float(o.psf_from_weights(w.w_half[0])[0, 0]))
    ctx.set_likelihood(1)
    kern = ctx.get_noise_kernel().cpu().numpy().astype(np.float64)
    rng = np.random.default_rng(11)
    xi = (0.2 * rng.normal(size=(1, w.ny, w.nx))).astype(np.float32)
    ctx.sky_forward(dev(xi))
    nsamp = 2
    eta_xi = rng.normal(size=(nsamp, 1, w.ny, w.nx)).astype(np.float32)
    eta_d = rng.normal(size=(nsamp, 1, w.ny, w.nx)).astype(np.float32)
    sh = SampleShard(ctx, nsamp)
    assert list(sh.mine) == [0, 1]
    samples = sh.draw(dev(eta_xi), dev(eta_d), 30)
    g = ctx.new_latent()
    e = sh.kl_energy_grad(dev(xi), g, True)
    smp = samples.cpu().numpy().astype(np.float64)
    e_ref, g_ref = o.kl_energy_grad_eq9(w.w_half, kern, w.dirty, w.amp, w.mu, w.lognu, xi, smp, True)
    assert abs(e - e_ref) <= 1e-5 * abs(e_ref) and rel(g.cpu().numpy(), g_ref) <= 1e-5
    v = rng.normal(size=xi.shape).astype(np.float32)
    out = ctx.new_latent()
    sh.kl_metric_apply(dev(xi), dev(v), out, True)
    assert rel(out.cpu().numpy(), o.kl_metric_apply_eq9(w.w_half, kern, w.amp, w.mu, w.lognu, xi, smp, v, True)) <= 1e-5


def test_two_devices_if_present():
    """Contexts on two devices in one process (per-device launch caches); skipped on a one-GPU box."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("one GPU")
    import paper_2406_09144_b200 as frs
    w = wl.make_config(1)
    outs = []
    for d in (0, 1):
        with torch.cuda.device(d):
            ctx = frs.Context(w.ny, w.nx, 1, device=d)
            ctx.set_psf_weights(torch.from_numpy(w.w_half).to(f"cuda:{d}"))
            x = torch.from_numpy(w.sky_true.astype(np.float32)).to(f"cuda:{d}")
            y = torch.empty_like(x)
            ctx.psf_apply(x, y)
            outs.append(y.cpu().numpy())
    assert np.array_equal(outs[0], outs[1])
