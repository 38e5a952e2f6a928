"""Host logic of the channel-sharded multi-GPU path (paper_2406_09144_b200/parallel.py), run on CPU
with world_size = 2 over gloo.  The CUDA context is replaced by an oracle-backed stand-in with the same
methods, so what is tested is the partitioning, the placement of the prior terms and the single
all-reduce per operator: the sharded result must equal the oracle evaluated on ALL channels."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from gen import workloads as wl
from oracle import frs_oracle as o
from paper_2406_09144_b200.parallel import ChannelShard, SampleShard, partition_channels


def test_partition_is_a_balanced_cover():
    for nchan in (1, 2, 5, 16, 17):
        for world in (1, 2, 3, 8):
            parts = [partition_channels(nchan, world, r) for r in range(world)]
            assert [c for p in parts for c in p] == list(range(nchan))          # contiguous cover, in order
            sizes = [len(p) for p in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        partition_channels(4, 2, 2)


class OracleCtx:
    """Stand-in for binding.Context on CPU tensors: same methods, arithmetic from the oracle."""

    def __init__(self, ny, nx, nchan):
        self.ny, self.nx, self.nchan = ny, nx, nchan
        self.lognu = np.zeros(nchan)

    def set_psf_weights(self, w):
        self.w = w.numpy().astype(np.float64)

    def set_dirty(self, j):
        self.j = j.numpy().astype(np.float64)

    def set_amplitude(self, amp, mu):
        self.amp, self.mu = amp.numpy().astype(np.float64), np.asarray(mu, np.float64)

    def set_channel_lognu(self, lognu):
        self.lognu = np.asarray(lognu, np.float64)

    def energy_grad(self, xi, grad, with_prior=True):
        self.xi = xi.numpy().astype(np.float64)
        e, g = o.energy_grad(self.w, self.j, self.amp, self.mu, self.lognu, self.xi, with_prior)
        grad.copy_(torch.from_numpy(g).to(grad.dtype))
        return e

    def _m(self, v, with_prior):
        return o.metric_apply(self.w, self.amp, self.mu, self.lognu, self.xi, v, with_prior)

    def metric_apply(self, v, out, with_prior=True):
        out.copy_(torch.from_numpy(self._m(v.numpy().astype(np.float64), with_prior)).to(out.dtype))

    def cg_solve(self, b, x, max_iter, with_prior=True):
        assert max_iter == 0
        self.r = b.clone().double()
        self.p = b.clone().double()
        self.rr = float((self.r * self.r).sum())

    def cg_step_begin(self):
        self.q = torch.from_numpy(self._m(self.p.numpy(), False))
        return self.q

    def cg_step_end(self, x, with_prior=True):
        q = self.q + self.p if with_prior else self.q
        alpha = self.rr / float((self.p * q).sum())
        x.add_((alpha * self.p).to(x.dtype))
        self.r = self.r - alpha * q
        rr_new = float((self.r * self.r).sum())
        self.p = self.r + (rr_new / self.rr) * self.p
        self.rr = rr_new

    def cg_read_state(self):
        return self.r, self.p, self.q, [self.rr]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = wl.make_config(5, n=32, nchan=3, npts=3000)              # 3 channels over 2 ranks: uneven split
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a))      # noqa: E731
        sh = ChannelShard(w.ny, w.nx, w.nchan, w.lognu, make_ctx=OracleCtx)
        sh.set_psf_weights(t(w.w_half))
        sh.set_dirty(t(w.dirty))
        sh.set_amplitude(t(w.amp), [float(m) for m in w.mu])
        xi = (0.3 * np.random.default_rng(3).normal(size=(w.nfield, w.ny, w.nx)))
        g = torch.zeros(w.nfield, w.ny, w.nx, dtype=torch.float64)
        e = sh.energy_grad(t(xi), g, with_prior=True)
        v = np.random.default_rng(4).normal(size=xi.shape)
        mv = torch.zeros_like(g)
        sh.metric_apply(t(v), mv, with_prior=True)
        b = -g.clone()
        x = torch.zeros_like(g)
        rn = sh.cg_solve(b, x, 6, with_prior=True)
        if rank == 0:
            e_ref, g_ref = o.energy_grad(w.w_half, w.dirty, w.amp, w.mu, w.lognu, xi, True)
            mv_ref = o.metric_apply(w.w_half, w.amp, w.mu, w.lognu, xi, v, True)
            sol = o.cg(lambda u: o.metric_apply(w.w_half, w.amp, w.mu, w.lognu, xi, u, True), -g_ref, max_iter=6)
            rel = lambda a, r: float(np.linalg.norm(a - r) / np.linalg.norm(r))   # noqa: E731
            out.put((len(sh.channels), abs(e - e_ref) / abs(e_ref), rel(g.numpy(), g_ref), rel(mv.numpy(), mv_ref),
                     rel(x.numpy(), sol["x"]), rn))
    finally:
        dist.destroy_process_group()


def test_sharded_operators_equal_the_full_oracle_world2():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = out.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    nloc, de, dg, dm, dx, rn = res
    assert nloc == 2                                   # rank 0 owns 2 of the 3 channels
    assert de <= 1e-12 and dg <= 1e-12 and dm <= 1e-12, res
    assert dx <= 1e-9 and rn > 0, res


# ---------------------------------------------------------------------------------- MGVI samples over ranks
class OracleKlCtx:
    """Stand-in with the MGVI methods of binding.Context, arithmetic from the oracle (Eq. 9 likelihood, R14 / R15)."""

    def __init__(self, w, kern):
        self.w, self.kern = w, kern

    def draw_sample(self, eta_xi, eta_d, sample, max_iter, rtol=0.0):
        s = o.draw_sample_eq9(self.w.w_half, self.kern, self.w.amp, self.w.mu, self.w.lognu, self.xi, eta_xi.numpy(), eta_d.numpy(), max_iter)[0]
        sample.copy_(torch.from_numpy(s))

    def kl_energy_grad(self, xi, samples, grad, mirrored=True):
        e, g = o.kl_energy_grad_eq9(self.w.w_half, self.kern, self.w.dirty, self.w.amp, self.w.mu, self.w.lognu, xi.numpy(),
                                    samples.numpy(), mirrored)
        grad.copy_(torch.from_numpy(g))
        return e

    def kl_metric_apply(self, xi, samples, v, out, mirrored=True):
        out.copy_(torch.from_numpy(o.kl_metric_apply_eq9(self.w.w_half, self.kern, self.w.amp, self.w.mu, self.w.lognu, xi.numpy(),
                                                         samples.numpy(), v.numpy(), mirrored)))


def _kl_worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = wl.make_config(1, n=16, seed=2)
        kern = o.noise_kernel_from_psf(w.w_half[0], 1e-2 * float(o.psf_from_weights(w.w_half[0])[0, 0]))[None]
        rng = np.random.default_rng(7)                                  # the same stream on every rank
        xi = 0.2 * rng.normal(size=(1, w.ny, w.nx))
        nsamp = 3                                                       # 3 samples over 2 ranks: uneven split
        eta_xi, eta_d = rng.normal(size=(nsamp, 1, w.ny, w.nx)), rng.normal(size=(nsamp, 1, w.ny, w.nx))
        ctx = OracleKlCtx(w, kern)
        ctx.xi = xi
        sh = SampleShard(ctx, nsamp)
        sh.draw(torch.from_numpy(eta_xi), torch.from_numpy(eta_d), 8)
        g = torch.zeros(1, w.ny, w.nx, dtype=torch.float64)
        e = sh.kl_energy_grad(torch.from_numpy(xi), g, True)
        v = rng.normal(size=xi.shape)
        mv = torch.zeros_like(g)
        sh.kl_metric_apply(torch.from_numpy(xi), torch.from_numpy(v), mv, True)
        if rank == 0:
            full = np.stack([o.draw_sample_eq9(w.w_half, kern, w.amp, w.mu, w.lognu, xi, eta_xi[i], eta_d[i], 8)[0] for i in range(nsamp)])
            e_ref, g_ref = o.kl_energy_grad_eq9(w.w_half, kern, w.dirty, w.amp, w.mu, w.lognu, xi, full, True)
            m_ref = o.kl_metric_apply_eq9(w.w_half, kern, w.amp, w.mu, w.lognu, xi, full, v, True)
            rel = lambda a, r: float(np.linalg.norm(a - r) / np.linalg.norm(r))   # noqa: E731
            out.put((len(sh.mine), abs(e - e_ref) / abs(e_ref), rel(g.numpy(), g_ref), rel(mv.numpy(), m_ref)))
    finally:
        dist.destroy_process_group()


def test_sample_sharded_kl_equals_the_full_oracle_world2():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_kl_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = out.get(timeout=240)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    nloc, de, dg, dm = res
    assert nloc == 2 and de <= 1e-12 and dg <= 1e-12 and dm <= 1e-12, res
