"""GPU parity of the learned amplitude spectrum and the joint (xi, theta) model (NEXT-3, reading R17)
against oracle/prior_oracle.py, through the C ABI.  Tolerances: the spectrum is evaluated in fp64 on the device and
rounded once (<= 2e-7 relative per value); image-sized results rel-L2 <= 1e-5 as everywhere (north_star)."""
import numpy as np
import pytest

from gen import workloads as wl
from oracle import prior_oracle as po

pytestmark = pytest.mark.gpu

HYPER = (18.0, 1.0, 0.1, 5.0, 1.0, -2.0, 0.2, 1.2, 0.4, 0.2, 0.2)        # Table A.1, S band


def rel(a, b):
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
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


def theta_of(nb, seed, scale=0.5):
    return (scale * np.random.default_rng(seed).normal(size=po.ntheta(nb))).astype(np.float32)


@pytest.mark.parametrize("shape", [(32, 32), (64, 128), (512, 512), (256, 1024), (4096, 4096)])
def test_amplitude_forward_jvp_vjp(frs, shape):
    import torch
    ny, nx = shape
    ctx = frs.Context(ny, nx, 1)
    ctx.set_amplitude_model(HYPER)
    b, mult, t = po.bins(ny, nx)
    assert ctx.nb == len(t) and ctx.ntheta == po.ntheta(len(t))
    th = theta_of(len(t), 1)
    amp = torch.empty(1, ny, nx, device="cuda")
    ctx.amplitude_forward(dev(th), amp)
    ref = po.amplitude(th.astype(np.float64), HYPER, ny, nx)
    got = amp.cpu().numpy()[0].astype(np.float64)
    assert np.max(np.abs(got - ref) / ref) <= 2e-7                 # every mode, relative: one fp32 rounding
    dth = theta_of(len(t), 2, 1.0)
    da = torch.empty(1, ny, nx, device="cuda")
    ctx.amplitude_jvp(dev(dth), da)
    ref_j = po.amplitude_jvp(th.astype(np.float64), dth.astype(np.float64), HYPER, ny, nx)
    assert np.max(np.abs(da.cpu().numpy()[0] - ref_j)) <= 3e-7 * np.max(np.abs(ref_j))
    g = np.random.default_rng(3).normal(size=(ny, nx)).astype(np.float32)
    gt = torch.empty(ctx.ntheta, device="cuda")
    ctx.amplitude_vjp(dev(g[None]), gt)
    ref_v = po.amplitude_vjp(th.astype(np.float64), g.astype(np.float64), HYPER, ny, nx)
    assert np.max(np.abs(gt.cpu().numpy() - ref_v)) <= 3e-7 * np.max(np.abs(ref_v))
    # adjointness of what the GPU computes, in fp64 on the host
    lhs = float((da.double() * dev(g[None]).double()).sum())
    rhs = float((dev(dth).double() * gt.double()).sum())
    assert abs(lhs - rhs) <= 1e-5 * abs(lhs)


def _problem(n, seed=5, ny=None, nx=None):
    w = wl.make_config(1, n=n, seed=seed) if ny is None else wl.make_config(3, ny=ny, nx=nx, seed=seed)
    rng = np.random.default_rng(seed)
    _, _, t = po.bins(w.ny, w.nx)
    hyper = (float(np.log(np.median(w.sky_true))), 1.0, 0.1, 1.0, 0.3, -3.0, 0.2, 0.5, 0.2, 0.2, 0.1)
    xi = (0.3 * rng.normal(size=(w.ny, w.nx))).astype(np.float32)
    th = (0.3 * rng.normal(size=po.ntheta(len(t)))).astype(np.float32)
    return w, hyper, xi, th, rng


@pytest.mark.parametrize("size", [(128, None, None), (0, 64, 256), (512, None, None)])
@pytest.mark.parametrize("with_prior", [True, False])
def test_joint_energy_gradient_and_metric(frs, size, with_prior):
    import torch
    w, hyper, xi, th, rng = _problem(size[0], ny=size[1], nx=size[2])
    ctx = frs.Context(w.ny, w.nx, 1)
    ctx.set_psf_weights(dev(w.w_half))
    ctx.set_dirty(dev(w.dirty))
    ctx.set_amplitude_model(hyper)
    gx = torch.empty(1, w.ny, w.nx, device="cuda")
    gt = torch.empty(ctx.ntheta, device="cuda")
    e = ctx.energy_grad_joint(dev(xi[None]), dev(th), gx, gt, with_prior)
    e_ref, gx_ref, gt_ref = po.energy_grad_joint(w.w_half[0], w.dirty[0], hyper, xi, th, with_prior)
    assert abs(e - e_ref) <= 1e-5 * abs(e_ref)
    assert rel(gx.cpu().numpy()[0], gx_ref) <= 1e-5
    assert rel(gt.cpu().numpy(), gt_ref) <= 1e-5
    # the sky of the joint position
    s = ctx.new_image()
    ctx.sky_forward(dev(xi[None]), s)
    assert rel(s.cpu().numpy()[0], po.sky_joint(None, hyper, xi, th)[0]) <= 1e-5
    dxi = rng.normal(size=xi.shape).astype(np.float32)
    dth = rng.normal(size=th.shape).astype(np.float32)
    ox = torch.empty(1, w.ny, w.nx, device="cuda")
    ot = torch.empty(ctx.ntheta, device="cuda")
    ctx.energy_grad_joint(dev(xi[None]), dev(th), gx, gt, with_prior)      # position (sky_forward kept it; explicit here)
    ctx.metric_apply_joint(dev(dxi[None]), dev(dth), ox, ot, with_prior)
    ox_ref, ot_ref = po.metric_apply_joint(w.w_half[0], hyper, xi, th, dxi, dth, with_prior)
    assert rel(ox.cpu().numpy()[0], ox_ref) <= 1e-5
    assert rel(ot.cpu().numpy(), ot_ref) <= 1e-5


def test_joint_model_with_the_eq9_likelihood(frs):
    """Mode 1 (Eq. 9 with the fitted noise kernel, R14) under the joint model: the oracle runs on the GPU's K."""
    import torch
    from oracle import frs_oracle as fo
    w, hyper, xi, th, rng = _problem(128)
    ctx = frs.Context(w.ny, w.nx, 1)
    ctx.set_psf_weights(dev(w.w_half))
    ctx.set_dirty(dev(w.dirty))
    ctx.set_amplitude_model(hyper)
    ctx.set_noise_kernel(1e-2 * float(fo.psf_from_weights(w.w_half[0])[0, 0]))
    ctx.set_likelihood(1)
    kern = ctx.get_noise_kernel().cpu().numpy()[0].astype(np.float64)
    gx, gt = torch.empty(1, w.ny, w.nx, device="cuda"), torch.empty(ctx.ntheta, device="cuda")
    e = ctx.energy_grad_joint(dev(xi[None]), dev(th), gx, gt, True)
    e_ref, gx_ref, gt_ref = po.energy_grad_joint(w.w_half[0], w.dirty[0], hyper, xi, th, True, kern)
    assert abs(e - e_ref) <= 1e-5 * abs(e_ref) and rel(gx.cpu().numpy()[0], gx_ref) <= 1e-5 and rel(gt.cpu().numpy(), gt_ref) <= 1e-5
    dxi, dth = rng.normal(size=xi.shape).astype(np.float32), rng.normal(size=th.shape).astype(np.float32)
    ox, ot = torch.empty_like(gx), torch.empty_like(gt)
    ctx.metric_apply_joint(dev(dxi[None]), dev(dth), ox, ot, True)
    ox_ref, ot_ref = po.metric_apply_joint(w.w_half[0], hyper, xi, th, dxi, dth, True, kern)
    assert rel(ox.cpu().numpy()[0], ox_ref) <= 1e-5 and rel(ot.cpu().numpy(), ot_ref) <= 1e-5


def test_joint_model_state_errors_and_switch_back(frs):
    import torch
    w, hyper, xi, th, rng = _problem(64)
    ctx = frs.Context(w.ny, w.nx, 1)
    ctx.set_psf_weights(dev(w.w_half))
    ctx.set_dirty(dev(w.dirty))
    gx, gt = torch.empty(1, w.ny, w.nx, device="cuda"), torch.empty(po.ntheta(len(po.bins(64, 64)[2])), device="cuda")
    ctx.ntheta = gt.numel()
    with pytest.raises(frs.FrsError):
        ctx.energy_grad_joint(dev(xi[None]), dev(th), gx, gt)               # no model set
    ctx.set_amplitude_model(hyper)
    with pytest.raises(frs.FrsError):
        ctx.metric_apply_joint(dev(xi[None]), dev(th), gx, gt)              # no joint position yet
    with pytest.raises(frs.FrsError):
        ctx.set_amplitude_model((1.0, -1.0) + tuple(hyper[2:]))             # log-normal mean <= 0
    e = ctx.energy_grad_joint(dev(xi[None]), dev(th), gx, gt)
    # a fixed amplitude array switches the learned spectrum off again; the fixed-amplitude path at A(theta) agrees
    amp = torch.empty(1, w.ny, w.nx, device="cuda")
    ctx.amplitude_forward(dev(th), amp)
    ctx.set_amplitude(amp, [hyper[0]])
    g2 = ctx.new_latent()
    e2 = ctx.energy_grad(dev(xi[None]), g2, with_prior=True)
    assert abs(e2 + 0.5 * float(np.sum(th.astype(np.float64) ** 2)) - e) <= 1e-6 * abs(e)
    assert rel(g2.cpu().numpy(), gx.cpu().numpy()) <= 1e-6
    with pytest.raises(frs.FrsError):
        ctx.energy_grad_joint(dev(xi[None]), dev(th), gx, gt)
    multi = frs.Context(64, 64, 2)
    with pytest.raises(frs.FrsError):
        multi.set_amplitude_model(hyper)


# ---------------------------------------------------------------------------------- point sources (reading R18)
@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("size", [(128, None, None), (0, 64, 256)])
def test_full_model_with_point_sources(frs, size, mode):
    import torch
    from oracle import frs_oracle as fo
    w, hyper, xi, th, rng = _problem(size[0], ny=size[1], nx=size[2])
    ny, nx = w.ny, w.nx
    yx = np.array([[ny // 2, nx // 2], [ny // 2 + 1, nx // 2 - 2], [0, nx - 1], [ny - 1, 0]])
    alpha, q = 0.5, 0.05 * float(np.median(w.sky_true))
    pts = (yx, alpha, q)
    xp = np.array([0.8, -0.4, 2.5, -3.0], np.float32)
    ctx = frs.Context(ny, nx, 1)
    ctx.set_psf_weights(dev(w.w_half))
    ctx.set_dirty(dev(w.dirty))
    ctx.set_amplitude_model(hyper)
    ctx.set_point_sources(yx, alpha, q)
    kern = None
    if mode == 1:
        ctx.set_noise_kernel(1e-2 * float(fo.psf_from_weights(w.w_half[0])[0, 0]))
        ctx.set_likelihood(1)
        kern = ctx.get_noise_kernel().cpu().numpy()[0].astype(np.float64)
    theta = np.concatenate([th, xp]).astype(np.float32)
    assert ctx.ntheta_joint == theta.size
    gx, gt = torch.empty(1, ny, nx, device="cuda"), torch.empty(theta.size, device="cuda")
    e = ctx.energy_grad_joint(dev(xi[None]), dev(theta), gx, gt, True)
    e_ref, gx_ref, gt_ref, gp_ref = po.energy_grad_full(w.w_half[0], w.dirty[0], hyper, xi, th, pts, xp, True, kern)
    assert abs(e - e_ref) <= 1e-5 * abs(e_ref)
    assert rel(gx.cpu().numpy()[0], gx_ref) <= 1e-5
    got = gt.cpu().numpy()
    assert rel(got[:th.size], gt_ref) <= 1e-5
    # each point gradient is dflux x (C s - j)[pixel]: a difference of two image values, held to 1e-5 of its operands
    s_ref = po.sky_full(hyper, xi, th, pts, xp)[0]
    cs = fo.psf_apply(w.w_half[0], s_ref)
    scale = po.point_flux_prime(xp, alpha, q) * np.array([abs(cs[y, x]) + abs(w.dirty[0][y, x]) for y, x in yx]) + np.abs(xp)
    if mode == 0:
        assert np.all(np.abs(got[th.size:] - gp_ref) <= 1e-5 * scale)
    else:
        assert rel(got[th.size:], gp_ref) <= 1e-4
    # the cached sky carries the fluxes, in the natural orientation too
    s = ctx.new_image()
    ctx.sky_forward(dev(xi[None]), s)
    assert rel(s.cpu().numpy()[0], s_ref) <= 1e-5
    for (y, x), f in zip(yx, po.point_flux(xp, alpha, q)):
        assert abs(float(s[0, y, x]) - s_ref[y, x]) <= 2e-6 * s_ref[y, x]
    dxi = rng.normal(size=xi.shape).astype(np.float32)
    dth = rng.normal(size=theta.shape).astype(np.float32)
    ox, ot = torch.empty_like(gx), torch.empty_like(gt)
    ctx.energy_grad_joint(dev(xi[None]), dev(theta), gx, gt, True)
    ctx.metric_apply_joint(dev(dxi[None]), dev(dth), ox, ot, True)
    ox_ref, ot_ref, op_ref = po.metric_apply_full(w.w_half[0], hyper, xi, th, pts, xp, dxi, dth[:th.size], dth[th.size:], True, kern)
    assert rel(ox.cpu().numpy()[0], ox_ref) <= 1e-5
    assert rel(ot.cpu().numpy()[:th.size], ot_ref) <= 1e-5
    assert rel(ot.cpu().numpy()[th.size:], op_ref) <= 1e-5
    # the xi-block operators of the fixed-amplitude API see the same Jacobian (diffuse sky at the point pixels)
    out = ctx.new_latent()
    ctx.metric_apply(dev(dxi[None]), out, with_prior=True)
    ref0 = po.metric_apply_full(w.w_half[0], hyper, xi, th, pts, xp, dxi, np.zeros_like(th), np.zeros(4), True, kern)[0]
    assert rel(out.cpu().numpy()[0], ref0) <= 1e-5


def test_point_source_argument_errors(frs):
    ctx = frs.Context(64, 64, 1)
    for bad in ([[64, 0]], [[0, -1]], [[3, 4], [3, 4]]):
        with pytest.raises(frs.FrsError):
            ctx.set_point_sources(bad, 0.5, 1.0)
    with pytest.raises(frs.FrsError):
        ctx.set_point_sources([[1, 1]], 0.0, 1.0)
    ctx.set_point_sources([], 0.5, 1.0)
    # the field of view, not the grid, bounds the pixels -- in either order of the two calls
    ctx.set_field_of_view(48, 40)
    with pytest.raises(frs.FrsError, match="field of view"):
        ctx.set_point_sources([[10, 40]], 0.5, 1.0)
    with pytest.raises(frs.FrsError, match="field of view"):
        ctx.set_point_sources([[48, 3]], 0.5, 1.0)
    ctx.set_point_sources([[47, 39]], 0.5, 1.0)
    with pytest.raises(frs.FrsError, match="field of view"):
        ctx.set_field_of_view(47, 40)
    ctx.set_field_of_view(64, 64)
    ctx.set_point_sources([[63, 63]], 0.5, 1.0)
    with pytest.raises(frs.FrsError, match="field of view"):
        ctx.set_field_of_view(48, 40)
    with pytest.raises(frs.FrsError, match="field of view"):
        ctx.set_psf_embedded(torch_zeros_psf(24, 20), 24, 20)


def torch_zeros_psf(ny_img, nx_img):
    import torch
    return torch.zeros(1, 2 * ny_img, 2 * nx_img, device="cuda")


def test_cg_graph_is_rebuilt_when_the_model_changes(frs):
    """The captured CG iteration freezes the launch sequence; adding point sources changes it (two patch kernels per
    apply): the same solve into the same x must match plain launches bit for bit after the change."""
    import torch
    w, hyper, xi, th, rng = _problem(128)
    ctx = frs.Context(w.ny, w.nx, 1)
    ctx.set_psf_weights(dev(w.w_half))
    ctx.set_dirty(dev(w.dirty))
    ctx.set_amplitude_model(hyper)
    gx, gt = torch.empty(1, w.ny, w.nx, device="cuda"), torch.empty(ctx.ntheta, device="cuda")
    ctx.energy_grad_joint(dev(xi[None]), dev(th), gx, gt)
    b = (-gx).contiguous()
    x = torch.zeros_like(b)
    ctx.cg_solve(b, x, 8)
    x1 = x.clone()
    ctx.set_point_sources([[64, 64], [10, 100]], 0.5, 0.05 * float(np.median(w.sky_true)))
    theta = torch.cat([dev(th), dev(np.array([1.5, 2.0], np.float32))])
    gt2 = torch.empty(theta.numel(), device="cuda")
    ctx.energy_grad_joint(dev(xi[None]), theta, gx, gt2)
    x.zero_()
    ctx.cg_solve(b, x, 8)                      # same x pointer, same arguments: only the model changed
    x2 = x.clone()
    ctx.set_cuda_graphs(False)
    x.zero_()
    ctx.cg_solve(b, x, 8)
    assert torch.equal(x, x2) and not torch.equal(x1, x2)


def test_cg_graph_is_rebuilt_when_point_fluxes_enter_the_cached_sky(frs):
    """Whether the cached sky carries point fluxes decides the launch sequence of an iteration (two patch kernels, no fused
    inverse pass), and frs_set_sky / frs_sky_forward flip that without any setter being called: set_sky -> solve (graph
    without the patch kernels) -> sky_forward -> solve into the same x must match plain launches bit for bit."""
    import torch
    w, hyper, xi, th, rng = _problem(128)
    ctx = frs.Context(w.ny, w.nx, 1)
    ctx.set_psf_weights(dev(w.w_half))
    ctx.set_dirty(dev(w.dirty))
    ctx.set_amplitude_model(hyper)
    ctx.set_point_sources([[64, 64], [10, 100]], 0.5, 0.05 * float(np.median(w.sky_true)))
    theta = torch.cat([dev(th), dev(np.array([1.5, 2.0], np.float32))])
    gx, gt = torch.empty(1, w.ny, w.nx, device="cuda"), torch.empty(theta.numel(), device="cuda")
    ctx.energy_grad_joint(dev(xi[None]), theta, gx, gt)
    b = (-gx).contiguous()
    s = ctx.new_image()
    ctx.sky_forward(dev(xi[None]), s)
    ctx.set_sky(s)                             # a caller's sky: no point bookkeeping, fused launch sequence
    x = torch.zeros_like(b)
    ctx.cg_solve(b, x, 8)
    x_plain_sky = x.clone()
    ctx.sky_forward(dev(xi[None]))             # fluxes back in the cached sky; no setter ran in between
    x.zero_()
    ctx.cg_solve(b, x, 8)                      # same x pointer, same arguments
    x_graph = x.clone()
    ctx.set_cuda_graphs(False)
    x.zero_()
    ctx.cg_solve(b, x, 8)
    assert torch.equal(x, x_graph) and not torch.equal(x_plain_sky, x_graph)


def test_mgvi_sample_with_point_sources_uses_the_diffuse_jacobian(frs):
    """frs_draw_sample with point fluxes in the cached sky: the source m = eta_xi + J^T C N'^-1/2 eta_d is formed with the
    Jacobian of the DIFFUSE sky at the point pixels, the one the metric of the CG that follows uses (Cov m = M)."""
    from oracle import frs_oracle as fo
    w, hyper, xi, th, rng = _problem(128)
    ny, nx = w.ny, w.nx
    yx = np.array([[ny // 2, nx // 2], [ny // 2 + 1, nx // 2 - 2], [0, nx - 1]])
    alpha, q = 0.5, 0.05 * float(np.median(w.sky_true))
    pts, xp = (yx, alpha, q), np.array([0.8, 2.5, -1.0], np.float32)
    ctx = frs.Context(ny, nx, 1)
    ctx.set_psf_weights(dev(w.w_half))
    ctx.set_dirty(dev(w.dirty))
    ctx.set_amplitude_model(hyper)
    ctx.set_point_sources(yx, alpha, q)
    ctx.set_noise_kernel(1e-2 * float(fo.psf_from_weights(w.w_half[0])[0, 0]))
    ctx.set_likelihood(1)
    kern = ctx.get_noise_kernel().cpu().numpy().astype(np.float64)
    theta = np.concatenate([th, xp]).astype(np.float32)
    import torch
    gx, gt = torch.empty(1, ny, nx, device="cuda"), torch.empty(theta.size, device="cuda")
    ctx.energy_grad_joint(dev(xi[None]), dev(theta), gx, gt, True)          # joint position: fluxes in the cached sky
    eta_xi = rng.normal(size=(1, ny, nx)).astype(np.float32)
    eta_d = rng.normal(size=(1, ny, nx)).astype(np.float32)
    sample = ctx.new_latent()
    assert ctx.draw_sample(dev(eta_xi), dev(eta_d), sample, 4) == 4
    amp = po.amplitude(th.astype(np.float64), hyper, ny, nx)
    s_diff = po.sky_joint(None, hyper, xi, th)[0][None]
    s_tot = po.sky_full(hyper, xi, th, pts, xp)[0][None]
    lognu = np.zeros(1)
    m_ref = fo.sample_source_eq9(w.w_half, kern, amp[None], lognu, s_diff, eta_xi, eta_d)
    m_wrong = fo.sample_source_eq9(w.w_half, kern, amp[None], lognu, s_tot, eta_xi, eta_d)
    assert rel(m_wrong, m_ref) > 1e-3                                        # the two Jacobians are told apart here
    zt, zp = np.zeros_like(th), np.zeros(len(xp))
    apply = lambda v: po.metric_apply_full(w.w_half[0], hyper, xi, th, pts, xp, v[0], zt, zp, True, kern[0])[0][None]  # noqa: E731
    sol = fo.cg(apply, m_ref, max_iter=4)
    r, p, qq, sc = ctx.cg_read_state()
    resid = m_ref - apply(sample.cpu().numpy().astype(np.float64))          # r_4 = m - M sigma_4 pins the GPU's m
    assert np.linalg.norm(r.cpu().numpy() - resid) <= 1e-4 * np.linalg.norm(m_ref)
    assert rel(sample.cpu().numpy(), sol["x"]) <= 1e-4
