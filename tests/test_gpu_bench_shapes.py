"""Parity at every launch shape bench.py times beyond the headline operator: the Eq. 9 likelihood at
configs 4 and 5, the joint (xi, theta) model at 2048^2 and 4096^2, MGVI samples and the KL calls at 1024^2, the embedded
3600^2-in-4096^2 energy / gradient / metric, and the major cycle on the uv lists of configs 1 and 2.  Each against the fp64
oracle on the same seeded inputs (sampled outputs where the oracle's direct sums are too slow), guard zones on."""
import time

import numpy as np
import pytest

from gen import workloads as wl
from oracle import frs_oracle as o
from oracle import prior_oracle as po

pytestmark = pytest.mark.gpu
TOL = 1e-5


def rel(a, b):
    a, b = np.asarray(a), np.asarray(b)
    dt = np.complex128 if np.iscomplexobj(a) or np.iscomplexobj(b) else np.float64
    a, b = a.astype(dt), b.astype(dt)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.fixture(scope="module")
def frs():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2406_09144_b200 as m
    m.load_library()
    return m


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def setup(frs, w, eps_rel=1e-2):
    ctx = frs.Context(w.ny, w.nx, w.nchan)
    ctx.set_psf_weights(dev(w.w_half))
    ctx.set_dirty(dev(w.dirty))
    ctx.set_amplitude(dev(w.amp), w.mu)
    ctx.set_channel_lognu(w.lognu)
    eps = eps_rel * float(np.sum(o.full_spectrum(w.w_half[0])))
    ctx.set_noise_kernel(eps)
    return ctx, eps


@pytest.mark.parametrize("cfg", [4, 5])
def test_eq9_full_size_configs_4_and_5(frs, cfg, monkeypatch):
    """Mode 1 at the shapes bench.py times it on: config 4 (4096^2, one field: rows_inv<4096, plain> -> hart_cols<4096, mul> x 2 ->
    second convolution) and config 5 (16 x 1024^2, two fields: the jvp_combine / vjp_combine path of the Eq. 9 metric).  The fit
    of K, energy, gradient, metric apply and one teacher-forced CG step against the oracle on the GPU's own K; guard zones on."""
    import torch
    monkeypatch.setenv("FRS_GUARD", "1")
    w = wl.make_config(cfg)
    ctx, eps = setup(frs, w)
    ctx.set_likelihood(1)
    k_gpu = ctx.get_noise_kernel().cpu().numpy()
    for c in (0, w.nchan - 1):
        k_ref = o.noise_kernel_from_psf(w.w_half[c], eps)
        assert np.max(np.abs(k_gpu[c] - k_ref)) <= TOL * np.max(k_ref)
    xi = (0.3 * np.random.default_rng(36).normal(size=(w.nfield, w.ny, w.nx))).astype(np.float32)
    g = ctx.new_latent()
    e = ctx.energy_grad(dev(xi), g, with_prior=True)
    e_ref, g_ref = o.energy_grad_eq9(w.w_half, k_gpu, w.dirty, w.amp, w.mu, w.lognu, xi, True)
    assert abs(e - e_ref) <= TOL * abs(e_ref)
    assert rel(g.cpu().numpy(), g_ref) <= TOL
    s64 = o.sky(xi, w.amp, w.mu, w.lognu)
    ap = lambda u: o.metric_apply_eq9(w.w_half, k_gpu, w.amp, w.mu, w.lognu, xi, u, True, s=s64)  # noqa: E731
    v = np.random.default_rng(37).normal(size=xi.shape).astype(np.float32)
    out = ctx.new_latent()
    ctx.metric_apply(dev(v), out, with_prior=True)
    assert rel(out.cpu().numpy(), ap(v)) <= TOL
    b = dev(np.random.default_rng(38).normal(size=xi.shape).astype(np.float32))
    x = torch.zeros_like(b)
    ctx.cg_solve(b, x, 0)                                                      # r = p = b, rr = <b, b>
    r, p, q, sc = ctx.cg_read_state()
    x0, r0, p0 = (t.cpu().numpy().astype(np.float64) for t in (x, r, p))
    ctx.cg_step(x, True)
    r, p, q, sc1 = ctx.cg_read_state()
    st = o.cg_step(ap, x0, r0, p0, float(sc[0]))
    assert rel(q.cpu().numpy(), st["q"]) <= TOL
    assert abs(sc1[3] - st["alpha"]) <= TOL * abs(st["alpha"])
    assert rel(x.cpu().numpy(), st["x"]) <= TOL
    bad, n = ctx.check_guards()
    assert bad == 0 and n >= 10, (bad, n)
    del ctx
    torch.cuda.empty_cache()


# ---------------------------------------------------------------------------------- joint (xi, theta) model (reading R17)
@pytest.mark.parametrize("cfg", [3, 4])
def test_joint_model_full_size(frs, cfg, monkeypatch):
    """Image-sized results of the joint model at 2048^2 and 4096^2 (bench.py times joint_* at 4096^2: amp_gather, the bin
    reduction of 16.7 M modes onto 2 897 bins, joint_prologue): energy, both gradients and the metric, hyper-parameters as in
    bench.py."""
    import torch
    monkeypatch.setenv("FRS_GUARD", "1")
    w = wl.make_config(cfg)
    rng = np.random.default_rng(40 + cfg)
    hyper = (float(w.mu[0]), 1.0, 0.1, 1.0, 0.3, -3.0, 0.2, 0.5, 0.2, 0.2, 0.1)
    _, _, t = po.bins(w.ny, w.nx)
    xi = (0.3 * rng.normal(size=(w.ny, w.nx))).astype(np.float32)
    th = (0.3 * rng.normal(size=po.ntheta(len(t)))).astype(np.float32)
    ctx = frs.Context(w.ny, w.nx, 1)
    ctx.set_psf_weights(dev(w.w_half))
    ctx.set_dirty(dev(w.dirty))
    ctx.set_amplitude_model(hyper)
    assert ctx.ntheta == th.size
    gx, gt = torch.empty(1, w.ny, w.nx, device="cuda"), torch.empty(th.size, device="cuda")
    e = ctx.energy_grad_joint(dev(xi[None]), dev(th), gx, gt, True)
    e_ref, gx_ref, gt_ref = po.energy_grad_joint(w.w_half[0], w.dirty[0], hyper, xi, th, True)
    assert abs(e - e_ref) <= TOL * abs(e_ref)
    assert rel(gx.cpu().numpy()[0], gx_ref) <= TOL
    assert rel(gt.cpu().numpy(), gt_ref) <= TOL
    dxi = rng.normal(size=xi.shape).astype(np.float32)
    dth = rng.normal(size=th.shape).astype(np.float32)
    ox, ot = torch.empty_like(gx), torch.empty_like(gt)
    ctx.metric_apply_joint(dev(dxi[None]), dev(dth), ox, ot, True)
    ox_ref, ot_ref = po.metric_apply_joint(w.w_half[0], hyper, xi, th, dxi, dth, True)
    assert rel(ox.cpu().numpy()[0], ox_ref) <= TOL
    assert rel(ot.cpu().numpy(), ot_ref) <= TOL
    bad, n = ctx.check_guards()
    assert bad == 0 and n >= 10, (bad, n)
    del ctx
    torch.cuda.empty_cache()


# ---------------------------------------------------------------------------------- MGVI at 1024^2 (reading R15)
def test_mgvi_sample_and_kl_at_1024(frs, monkeypatch):
    """frs_draw_sample (graph-replayed CG in mode 1) and the KL calls on two mirrored samples at 1024^2."""
    monkeypatch.setenv("FRS_GUARD", "1")
    w = wl.make_config(3, n=1024)
    ctx, eps = setup(frs, w)
    ctx.set_likelihood(1)
    k_gpu = ctx.get_noise_kernel().cpu().numpy()
    rng = np.random.default_rng(51)
    xi = (0.2 * rng.normal(size=(1, w.ny, w.nx))).astype(np.float32)
    eta_xi = rng.normal(size=xi.shape).astype(np.float32)
    eta_d = rng.normal(size=(1, w.ny, w.nx)).astype(np.float32)
    ctx.sky_forward(dev(xi))
    sample = ctx.new_latent()
    assert ctx.draw_sample(dev(eta_xi), dev(eta_d), sample, 4) == 4
    sg_ref, m_ref = o.draw_sample_eq9(w.w_half, k_gpu, w.amp, w.mu, w.lognu, xi, eta_xi, eta_d, cg_iters=4)
    r, p, q, sc = ctx.cg_read_state()
    s64 = o.sky(xi, w.amp, w.mu, w.lognu)
    resid = m_ref - o.metric_apply_eq9(w.w_half, k_gpu, w.amp, w.mu, w.lognu, xi, sample.cpu().numpy(), True, s=s64)
    assert np.linalg.norm(r.cpu().numpy() - resid) <= 1e-4 * np.linalg.norm(m_ref)
    assert rel(sample.cpu().numpy(), sg_ref) <= 1e-4
    samples = (0.1 * rng.normal(size=(2,) + xi.shape)).astype(np.float32)
    g = ctx.new_latent()
    kl = ctx.kl_energy_grad(dev(xi), dev(samples), g, mirrored=True)
    kl_ref, g_ref = o.kl_energy_grad_eq9(w.w_half, k_gpu, w.dirty, w.amp, w.mu, w.lognu, xi, list(samples), True)
    assert abs(kl - kl_ref) <= TOL * abs(kl_ref)
    assert rel(g.cpu().numpy(), g_ref) <= TOL
    v = rng.normal(size=xi.shape).astype(np.float32)
    out = ctx.new_latent()
    ctx.kl_metric_apply(dev(xi), dev(samples), dev(v), out, mirrored=True)
    assert rel(out.cpu().numpy(), o.kl_metric_apply_eq9(w.w_half, k_gpu, w.amp, w.mu, w.lognu, xi, list(samples), v, True)) <= TOL
    bad, n = ctx.check_guards()
    assert bad == 0 and n >= 10, (bad, n)


# ---------------------------------------------------------------------------------- 3600^2 embedded in 4096^2 (reading R19)
def test_embedded_3600_energy_gradient_and_metric(frs, monkeypatch):
    """the paper's 3600^2 image in a 4096^2 context -- energy, gradient and metric, not only the convolution."""
    import torch
    monkeypatch.setenv("FRS_GUARD", "1")
    nyi = nxi = 3600
    ny = nx = 4096
    w = wl.make_config(3, ny=nyi, nx=nxi, npts=200000)
    amp = wl.amplitude_spectrum(ny, nx, "pow3.5", 1.0).astype(np.float32)          # a prior spectrum on the embedding grid
    psf = o.psf_from_weights(w.w_half[0]).astype(np.float32)
    w_img = o.psf_spectrum_from_psf(psf.astype(np.float64))[0]
    mu = float(np.log(np.median(w.sky_true)))
    ctx = frs.Context(ny, nx, 1)
    ctx.set_psf_embedded(dev(psf[None]), nyi, nxi)
    ctx.set_dirty(dev(o.embed(w.dirty[0], ny, nx)[None]))
    ctx.set_amplitude(dev(amp[None]), [mu])
    rng = np.random.default_rng(3)
    xi = (0.3 * rng.normal(size=(ny, nx))).astype(np.float32)
    g = ctx.new_latent()
    e = ctx.energy_grad(dev(xi[None]), g, with_prior=True)
    e_ref, g_ref = o.energy_grad_embedded(w_img, w.dirty[0], amp, mu, xi)
    assert abs(e - e_ref) <= TOL * abs(e_ref) and rel(g.cpu().numpy()[0], g_ref) <= TOL
    v = rng.normal(size=(ny, nx)).astype(np.float32)
    out = ctx.new_latent()
    ctx.metric_apply(dev(v[None]), out, with_prior=True)
    assert rel(out.cpu().numpy()[0], o.metric_apply_embedded(w_img, nyi, nxi, amp, mu, xi, v)) <= TOL
    bad, n = ctx.check_guards()
    assert bad == 0 and n >= 10, (bad, n)
    del ctx
    torch.cuda.empty_cache()


# ---------------------------------------------------------------------------------- major cycle on the uv lists of configs 1 and 2
def _uv_list(cfg):
    """The uv list gen/workloads.py draws first for BASELINE.json config `cfg` (seed 0), kept where the direct sums are
    defined (|u| < nx - 1/2, |v| < ny - 1/2)."""
    rng = np.random.default_rng(0)
    if cfg == 1:
        n, (u, v) = 128, wl.uv_gaussian(rng, 20_000, 256, 256, 0.25)
    else:
        n, (u, v) = 512, wl.uv_vla_like(rng, 200_000, 1024, 1024)
    keep = (np.abs(u) < n - 0.5) & (np.abs(v) < n - 0.5)
    return n, np.stack([u[keep], v[keep]], axis=1).astype(np.float32)


def _gpu_ms(fn):
    import torch
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    a.record()
    fn()
    b.record()
    torch.cuda.synchronize()
    return a.elapsed_time(b)


def test_major_cycle_on_the_uv_list_of_config_1(frs):
    """2 x 10^4 visibilities at 128^2: response, adjoint and the residual of Eq. 20-22 against the oracle's full direct sums."""
    import torch
    n, uv = _uv_list(1)
    nvis = uv.shape[0]
    assert nvis > 18_000                                                          # the rest falls outside |u|, |v| < n - 1/2
    rng = np.random.default_rng(72)
    wgt = rng.uniform(0.5, 2.0, nvis).astype(np.float32)
    sky = np.exp(rng.normal(size=(n, n))).astype(np.float32)
    ctx = frs.Context(n, n, 1)
    vis = torch.empty((nvis, 2), device="cuda")
    ctx.exact_response(dev(uv), dev(sky), vis)
    v_ref = o.exact_response(uv, sky, 2 * n, 2 * n)
    vh = vis.cpu().numpy()
    assert rel(vh[:, 0] + 1j * vh[:, 1], v_ref) <= TOL
    dirty = (o.exact_adjoint(uv, wgt, v_ref, n, n, 2 * n, 2 * n) * 1.01).astype(np.float32)
    d = torch.empty((n, n), device="cuda")
    ctx.major_cycle_residual(dev(uv), dev(wgt), dev(dirty), dev(sky), d)       # warm-up, then timed
    ms = _gpu_ms(lambda: ctx.major_cycle_residual(dev(uv), dev(wgt), dev(dirty), dev(sky), d))
    print(f"major cycle residual, config 1 uv list ({nvis} vis, {n}^2): {ms:.3f} ms")
    d_ref = o.major_cycle_residual(uv, wgt, dirty, sky, 2 * n, 2 * n)
    assert np.linalg.norm(d.cpu().numpy() - d_ref) <= TOL * np.linalg.norm(dirty)


def test_major_cycle_on_the_uv_list_of_config_2(frs):
    """2 x 10^5 visibilities at 512^2.  The oracle's direct sums are O(nvis npix) = 5 x 10^10 terms, so it computes SAMPLED
    outputs one by one: 400 visibilities of R sky (each V_k is independent of the others), and two blocks of pixels of the
    adjoint -- the corner block directly (the same call with a smaller image and the full padded size), one block elsewhere
    through the shift theorem (pixel offset (y0, x0) = visibilities times exp(+2 pi i (u x0 / Mx + v y0 / My)))."""
    import torch
    n, uv = _uv_list(2)
    nvis = uv.shape[0]
    assert nvis > 190_000
    m = 2 * n
    rng = np.random.default_rng(73)
    wgt = rng.uniform(0.5, 2.0, nvis).astype(np.float32)
    sky = np.exp(rng.normal(size=(n, n))).astype(np.float32)
    ctx = frs.Context(n, n, 1)
    vis = torch.empty((nvis, 2), device="cuda")
    ctx.exact_response(dev(uv), dev(sky), vis)
    vh = vis.cpu().numpy().astype(np.float64)
    vg = vh[:, 0] + 1j * vh[:, 1]
    pick = rng.choice(nvis, 400, replace=False)
    assert rel(vg[pick], o.exact_response(uv[pick], sky, m, m)) <= TOL
    blocks = [(0, 0), (300, 411), (n - 24, n - 24)]
    uv64 = uv.astype(np.float64)

    def adjoint_block(v, y0, x0, nb=24):
        shift = np.exp(2j * np.pi * (uv64[:, 0] * x0 / m + uv64[:, 1] * y0 / m))
        return o.exact_adjoint(uv, wgt, v * shift, nb, nb, m, m)

    vin = (rng.normal(size=nvis) + 1j * rng.normal(size=nvis)).astype(np.complex64)
    y = torch.empty((n, n), device="cuda")
    ctx.exact_adjoint(dev(uv), dev(wgt), dev(np.stack([vin.real, vin.imag], 1)), y)
    yh = y.cpu().numpy()
    scale = np.linalg.norm(yh) / n                                               # rms pixel of the adjoint image
    for y0, x0 in blocks:
        ref = adjoint_block(vin.astype(np.complex128), y0, x0)
        assert np.linalg.norm(yh[y0:y0 + 24, x0:x0 + 24] - ref) <= TOL * max(np.linalg.norm(ref), 24 * scale)
    # the residual of Eq. 20-22, teacher-forced on the GPU's own visibilities (checked on the sample above)
    dirty = np.exp(rng.normal(size=(n, n))).astype(np.float32) * float(np.sum(wgt))
    d = torch.empty((n, n), device="cuda")
    ctx.major_cycle_residual(dev(uv), dev(wgt), dev(dirty), dev(sky), d)
    ms = _gpu_ms(lambda: ctx.major_cycle_residual(dev(uv), dev(wgt), dev(dirty), dev(sky), d))
    print(f"major cycle residual, config 2 uv list ({nvis} vis, {n}^2): {ms:.3f} ms")
    dh = d.cpu().numpy()
    for y0, x0 in blocks:
        back = adjoint_block(vg, y0, x0)
        ref = dirty[y0:y0 + 24, x0:x0 + 24].astype(np.float64) - back
        assert np.linalg.norm(dh[y0:y0 + 24, x0:x0 + 24] - ref) <= TOL * (np.linalg.norm(dirty[y0:y0 + 24, x0:x0 + 24]) + np.linalg.norm(back))
