"""Guard-zone sweep: the stand-in for compute-sanitizer memcheck (closed on the GPU pool, profiles/r2_sanitizer.md).
With FRS_GUARD=1 every array a context owns sits between two 4 KB zones of a byte pattern; after a pass over every family of
calls, at square, rectangular, multi-channel and embedded shapes, no zone may have been written to -- and a deliberate
write one element past an array must be caught."""
import os

import numpy as np
import pytest

from gen import workloads as wl
from oracle import frs_oracle as o

pytestmark = pytest.mark.gpu


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


@pytest.fixture()
def guarded(monkeypatch):
    import torch
    assert torch.cuda.is_available()
    import paper_2406_09144_b200 as frs
    frs.load_library()
    monkeypatch.setenv("FRS_GUARD", "1")
    return frs


def _exercise(frs, w, eq9=True):
    import torch
    ctx = frs.Context(w.ny, w.nx, w.nchan)
    ctx.set_psf_weights(dev(w.w_half))
    ctx.set_dirty(dev(w.dirty))
    ctx.set_amplitude(dev(w.amp), w.mu)
    ctx.set_channel_lognu(w.lognu)
    rng = np.random.default_rng(0)
    xi = dev(0.3 * rng.normal(size=(w.nfield, w.ny, w.nx)))
    x = dev(rng.normal(size=(w.nchan, w.ny, w.nx)))
    y = ctx.new_image()
    ctx.psf_apply(x, y)
    ctx.sky_forward(xi)
    ctx.sky_metric_apply(x, y)
    g = ctx.new_latent()
    for mode in ((0, 1) if eq9 else (0,)):
        if mode == 1:
            ctx.set_noise_kernel(1e-2 * float(o.psf_from_weights(w.w_half[0])[0, 0]))
            ctx.set_likelihood(1)
        ctx.energy_grad(xi, g, with_prior=True)
        out = ctx.new_latent()
        ctx.metric_apply(g, out, with_prior=True)
        b = (-g).contiguous()
        sol = torch.zeros_like(b)
        ctx.cg_solve(b, sol, 4)
        ctx.cg_solve(b, sol, 20, rtol=1e-1)
        ctx.cg_step(sol)
        if mode == 1 and w.nchan == 1:
            smp = ctx.new_latent()
            ctx.draw_sample(dev(rng.normal(size=(w.nfield, w.ny, w.nx))), dev(rng.normal(size=(w.nchan, w.ny, w.nx))), smp, 3)
            ctx.kl_energy_grad(xi, smp[None].contiguous(), g, True)
            ctx.kl_metric_apply(xi, smp[None].contiguous(), b, out, True)
    xh = torch.from_numpy(rng.normal(size=(w.nchan, w.ny, w.nx)).astype(np.float32)).pin_memory()
    yh = [torch.empty_like(xh).pin_memory() for _ in range(2)]
    ctx.set_likelihood(0)
    ctx.sky_metric_apply_host(xh, yh[0])
    ctx.sky_metric_apply_host_batch([xh, xh, xh], [yh[0], yh[1], yh[0]])
    return ctx


def test_no_guard_zone_is_touched(guarded):
    import torch
    frs = guarded
    ctxs = []
    for key in ((1, dict(n=128)), (3, dict(ny=32, nx=1024)), (3, dict(ny=2048, nx=32)), (3, dict(ny=64, nx=256)),
                (5, dict(n=64, nchan=3)), (1, dict(n=512))):
        ctxs.append(_exercise(frs, wl.make_config(key[0], **key[1]), eq9=key[1].get("n", 0) != 512 or True))
    # the learned spectrum with point sources, an embedded image, a major-cycle residual
    w = wl.make_config(1, n=128, seed=5)
    c = frs.Context(128, 128, 1)
    c.set_psf_weights(dev(w.w_half)); c.set_dirty(dev(w.dirty))
    c.set_amplitude_model((float(np.log(np.median(w.sky_true))), 1.0, 0.1, 1.0, 0.3, -3.0, 0.2, 0.5, 0.2, 0.2, 0.1))
    c.set_point_sources([[64, 64], [0, 127]], 0.5, 1e-3)
    rng = np.random.default_rng(1)
    xi, th = dev(0.3 * rng.normal(size=(1, 128, 128))), dev(0.3 * rng.normal(size=c.ntheta_joint))
    gx, gt = torch.empty_like(xi), torch.empty_like(th)
    c.energy_grad_joint(xi, th, gx, gt)
    c.metric_apply_joint(gx, gt, torch.empty_like(xi), torch.empty_like(th))
    ctxs.append(c)
    wi = wl.make_config(3, ny=48, nx=40, npts=5000)
    e = frs.Context(64, 64, 1)
    e.set_psf_embedded(dev(o.psf_from_weights(wi.w_half[0])[None]), 48, 40)
    e.set_dirty(dev(o.embed(wi.dirty[0], 64, 64)[None]))
    e.set_amplitude(dev(wl.make_config(1, n=64).amp), [0.0])
    ge = e.new_latent()
    e.energy_grad(dev(0.1 * rng.normal(size=(1, 64, 64))), ge)
    ctxs.append(e)
    total = 0
    for ctx in ctxs:
        bad, n = ctx.check_guards()
        assert bad == 0 and n >= 10, (bad, n)
        total += n
    assert total > 150


def test_a_write_past_an_array_is_caught(guarded):
    from paper_2406_09144_b200.binding import _device_view
    frs = guarded
    w = wl.make_config(1, n=64)
    ctx = _exercise(frs, w, eq9=False)
    assert ctx.check_guards()[0] == 0
    q = ctx.cg_step_begin()                                      # view of a ctx-owned latent array
    past = _device_view(q.data_ptr() + 2 * ctx.npix * 4, (1,), ctx.device)   # the array holds 2 npix floats
    past.fill_(1.0)
    assert ctx.check_guards()[0] == 1
    before = _device_view(q.data_ptr() - 4, (1,), ctx.device)
    before.fill_(1.0)
    assert ctx.check_guards()[0] == 1                            # same array, both zones


def test_results_repeat_bit_for_bit():
    """A race in a shared-memory exchange or between a TMA landing and its readers shows up as run-to-run differences:
    every deterministic call, repeated on the same inputs at several launch shapes, must return identical bits (all
    reductions are fixed-order; only the bin sums of the learned spectrum use fp64 atomics and are excluded)."""
    import torch
    import paper_2406_09144_b200 as frs
    frs.load_library()
    for key in ((1, dict(n=512)), (3, dict(ny=2048, nx=256)), (5, dict(n=256, nchan=3)), (1, dict(n=2048))):
        w = wl.make_config(key[0], **key[1])
        ctx = frs.Context(w.ny, w.nx, w.nchan)
        ctx.set_psf_weights(dev(w.w_half)); ctx.set_dirty(dev(w.dirty)); ctx.set_amplitude(dev(w.amp), w.mu); ctx.set_channel_lognu(w.lognu)
        rng = np.random.default_rng(0)
        xi = dev(0.3 * rng.normal(size=(w.nfield, w.ny, w.nx)))
        x = dev(rng.normal(size=(w.nchan, w.ny, w.nx)))
        ref = None
        for rep in range(4):
            y, g, out = ctx.new_image(), ctx.new_latent(), ctx.new_latent()
            ctx.sky_forward(xi)
            ctx.sky_metric_apply(x, y)
            e = ctx.energy_grad(xi, g, with_prior=True)
            ctx.metric_apply(g, out, with_prior=True)
            sol = torch.zeros_like(g)
            it, rn = ctx.cg_solve((-g).contiguous(), sol, 6)
            cur = (y, g, out, sol, e, rn)
            if ref is None:
                ref = cur
            else:
                assert all(torch.equal(a, b) for a, b in zip(cur[:4], ref[:4])) and cur[4] == ref[4] and cur[5] == ref[5], (key, rep)
