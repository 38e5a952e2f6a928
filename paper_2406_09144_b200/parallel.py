"""Channel sharding of the multi-frequency problem over ranks.

Channels are independent through the whole convolution (own PSF spectrum, dirty image and sky), so they
are partitioned over the ranks of a torch.distributed process group (one process per GPU, NCCL over
NVLink; gloo on CPU in the tests).  The latent vectors (xi, v, the CG vectors) are replicated.  The one
exchange step of the path is the sum over channels inside the VJP: every rank applies its own
J_c^T C_c J_c and the results are summed with ONE all-reduce of a latent-sized vector per gradient /
metric apply / CG iteration; the prior term (+xi, +v, 1/2 <xi,xi>) is added by rank 0 only (gradient,
metric apply) or after the sum (CG step), so that the reduced result is exactly the full operator.
Dot products of CG run redundantly on the replicated vectors: no further communication.

This module holds no arithmetic of the method: every operator is a call into the C-ABI library through
`Context` (or any object with the same methods, which is how the CPU tests drive it).
"""
from __future__ import annotations


def partition_channels(nchan: int, world: int, rank: int) -> range:
    """Contiguous, balanced block of channels for `rank` (the first nchan % world ranks get one more)."""
    if not (0 <= rank < world) or nchan < 0:
        raise ValueError("bad rank / world / nchan")
    base, extra = divmod(nchan, world)
    start = rank * base + min(rank, extra)
    return range(start, start + base + (1 if rank < extra else 0))


class ChannelShard:
    """One rank's share of a multi-channel problem.

    make_ctx(ny, nx, nchan_local) -> context object (default: the CUDA `Context`); `group` is a
    torch.distributed process group (None: the default group).  Arrays passed to the setters are the
    FULL multi-channel arrays (every rank sees the same call); the shard slices its channels.
    """

    def __init__(self, ny, nx, nchan, lognu, group=None, make_ctx=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.channels = partition_channels(nchan, self.world, self.rank)
        if len(self.channels) == 0:
            raise ValueError(f"rank {self.rank}: no channels to own ({nchan} channels over {self.world} ranks)")
        if make_ctx is None:
            import torch
            from .binding import Context
            device = torch.cuda.current_device()              # one process per GPU: the rank's own device

            def make_ctx(ny_, nx_, nc_):
                return Context(ny_, nx_, nc_, device=device)
        self.ctx = make_ctx(ny, nx, len(self.channels))
        self.lognu = [float(lognu[c]) for c in self.channels]
        self.first = self.rank == 0                      # the rank that contributes the prior terms

    def _mine(self, a):
        return a[self.channels.start:self.channels.stop].contiguous()

    # ---- setup: every rank keeps its own channels only
    def set_psf_weights(self, w_half):
        self.ctx.set_psf_weights(self._mine(w_half))

    def set_dirty(self, j):
        self.ctx.set_dirty(self._mine(j))

    def set_amplitude(self, amp, mu):
        self.ctx.set_amplitude(amp, mu)
        if len(mu) == 2:
            self.ctx.set_channel_lognu(self.lognu)

    def _sum(self, t):
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)
        return t

    # ---- hot path
    def energy_grad(self, xi, grad, with_prior=True):
        """Total energy and gradient over ALL channels (identical on every rank)."""
        import torch
        e = self.ctx.energy_grad(xi, grad, with_prior=bool(with_prior and self.first))
        et = torch.tensor([e], dtype=torch.float64, device=grad.device)
        self._sum(et)
        self._sum(grad)
        return float(et.item())

    def metric_apply(self, v, out, with_prior=True):
        self.ctx.metric_apply(v, out, with_prior=bool(with_prior and self.first))
        self._sum(out)
        return out

    def cg_solve(self, b, x, max_iter, with_prior=True):
        """max_iter CG iterations on M x = b from x = 0 (x is zeroed).  Returns the final ||r||."""
        x.zero_()
        self.ctx.cg_solve(b, x, 0, with_prior=with_prior)     # r = p = b, rr = <b,b>  (M 0 = 0 on every rank)
        for _ in range(max_iter):
            q = self.ctx.cg_step_begin()                      # local likelihood part, ctx-owned
            self._sum(q)                                      # the exchange step
            self.ctx.cg_step_end(x, with_prior=with_prior)
        r, p, q, sc = self.ctx.cg_read_state()
        return float(sc[0]) ** 0.5


# ---- MGVI samples over ranks (the replica axis of the single-channel configs) ------------------------
def partition_samples(nsamp: int, world: int, rank: int) -> range:
    """Contiguous, balanced block of sample indices for `rank` (same rule as the channels)."""
    return partition_channels(nsamp, world, rank)


class SampleShard:
    """One rank's share of the MGVI samples of a single-channel problem (reading R15).

    Every rank holds the WHOLE problem (PSF spectrum, dirty image, model: replicas) and draws / evaluates only its
    own samples: drawing a sample is an independent CG solve, and the sample-averaged KL, its gradient and its metric
    are means over samples, so the only exchange is ONE all-reduce (sum) of a latent-sized vector (plus the energy
    scalar) per KL evaluation or metric apply; a rank weights its local mean by n_local / n_total before the sum.
    `ctx` is a ready Context (or any object with draw_sample / kl_energy_grad / kl_metric_apply).
    """

    def __init__(self, ctx, nsamp, group=None):
        import torch.distributed as dist
        self.dist, self.group, self.ctx = dist, group, ctx
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.nsamp = int(nsamp)
        self.mine = partition_samples(self.nsamp, self.world, self.rank)
        self.samples = None

    def _sum(self, t):
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)
        return t

    def draw(self, eta_xi, eta_d, max_iter, rtol=0.0):
        """eta_xi [nsamp, nfield, ny, nx], eta_d [nsamp, nchan, ny, nx]: the white-noise inputs of ALL samples (every rank
        sees the same arrays, e.g. from a counter-based generator); the rank solves for its own block only."""
        import torch
        loc = [torch.zeros_like(eta_xi[0]) for _ in self.mine]
        for out, i in zip(loc, self.mine):
            self.ctx.draw_sample(eta_xi[i].contiguous(), eta_d[i].contiguous(), out, max_iter, rtol)
        self.samples = torch.stack(loc) if loc else eta_xi[:0].clone()
        return self.samples

    def kl_energy_grad(self, xi, grad, mirrored=True):
        """KL estimate over ALL samples and its gradient (identical on every rank)."""
        import torch
        n = len(self.mine)
        e = 0.0
        if n:
            e = self.ctx.kl_energy_grad(xi, self.samples, grad, mirrored) * n / self.nsamp
            grad.mul_(n / self.nsamp)
        else:
            grad.zero_()
        et = torch.tensor([e], dtype=torch.float64, device=grad.device)
        self._sum(et)
        self._sum(grad)
        return float(et.item())

    def kl_metric_apply(self, xi, v, out, mirrored=True):
        n = len(self.mine)
        if n:
            self.ctx.kl_metric_apply(xi, self.samples, v, out, mirrored)
            out.mul_(n / self.nsamp)
        else:
            out.zero_()
        self._sum(out)
        return out
