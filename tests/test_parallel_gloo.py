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
from paper_2406_09144_b200.parallel import ChannelShard, partition_channels


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
