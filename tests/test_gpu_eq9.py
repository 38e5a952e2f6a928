"""GPU parity of the paper's literal likelihood -- Eq. 9 with the fitted noise kernel (Eq. 15-18; R14)
-- against oracle.noise_kernel_from_psf / ninv_apply / energy_grad_eq9 / metric_apply_eq9.  The fit of K is compared on its
own; every operator built on K is then compared with the oracle running on the GPU's own K (teacher-forced), so that the
rounding of the fit is not counted twice."""
import numpy as np
import pytest

from gen import workloads as wl
from oracle import frs_oracle as o

pytestmark = pytest.mark.gpu
TOL = 1e-5


def rel(a, b):
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


@pytest.fixture(scope="module")
def frs():
    import torch
    assert torch.cuda.is_available()
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


WORKLOADS = {"c1": lambda: wl.make_config(1), "rect": lambda: wl.make_config(3, ny=64, nx=128),
             "sq512": lambda: wl.make_config(2, n=512), "multi": lambda: wl.make_config(5, n=64, nchan=3)}


@pytest.mark.parametrize("key", ["c1", "rect", "sq512", "multi"])
def test_noise_kernel_fit_and_ninv_apply(frs, key):
    w = WORKLOADS[key]()
    ctx, eps = setup(frs, w)
    k_gpu = ctx.get_noise_kernel().cpu().numpy()
    k_ref = np.stack([o.noise_kernel_from_psf(w.w_half[c], eps) for c in range(w.nchan)])
    assert np.max(np.abs(k_gpu - k_ref)) <= TOL * np.max(k_ref)              # Eq. 17 closed form
    assert np.all(k_gpu >= np.float32(eps))
    x = np.random.default_rng(31).normal(size=(w.nchan, w.ny, w.nx)).astype(np.float32)
    y = ctx.new_image()
    ctx.ninv_apply(dev(x), y)
    ref = np.stack([o.ninv_apply(k_gpu[c], x[c]) for c in range(w.nchan)])   # Eq. 18 on the GPU's own K
    assert rel(y.cpu().numpy(), ref) <= TOL


def test_ninv_apply_flat_kernel_and_errors(frs):
    import torch
    w = wl.make_config(1)
    ctx = frs.Context(w.ny, w.nx, 1)
    with pytest.raises(frs.FrsError) as ei:                                   # no PSF yet
        ctx.set_noise_kernel(1.0)
    assert ei.value.code == frs.binding.FRS_ESTATE
    ctx.set_psf_weights(dev(w.w_half))
    for bad in (0.0, -1.0):
        with pytest.raises(frs.FrsError) as ei:
            ctx.set_noise_kernel(bad)
        assert ei.value.code == frs.binding.FRS_EINVAL
    with pytest.raises(frs.FrsError) as ei:                                   # Eq. 9 mode needs a kernel
        ctx.set_likelihood(1)
    assert ei.value.code == frs.binding.FRS_ESTATE
    x = torch.randn(1, w.ny, w.nx, device="cuda")
    y = torch.empty_like(x)
    ctx.set_noise_kernel(kern=torch.full((1, w.ny, w.nx), 2.5, device="cuda"))
    ctx.ninv_apply(x, y)                                                      # K == c: N'^-1 = 1/c
    assert rel(y.cpu().numpy(), x.cpu().numpy() / 2.5) <= 1e-6
    k = torch.rand(1, w.ny, w.nx, device="cuda") + 0.5                        # not even
    with pytest.raises(frs.FrsError) as ei:
        ctx.set_noise_kernel(kern=k)
    assert ei.value.code == frs.binding.FRS_ENOTPSD
    k = torch.ones(1, w.ny, w.nx, device="cuda")
    k[0, 3, 5] = k[0, w.ny - 3, w.nx - 5] = -1.0                              # even but not positive
    with pytest.raises(frs.FrsError):
        ctx.set_noise_kernel(kern=k)
    ctx.set_noise_kernel(1.0)
    ctx.set_likelihood(1)
    ctx.set_psf_weights(dev(w.w_half))                                        # a new PSF discards the kernel
    with pytest.raises(frs.FrsError):
        ctx.get_noise_kernel()


@pytest.mark.parametrize("key", ["c1", "rect", "sq512", "multi"])
@pytest.mark.parametrize("with_prior", [True, False])
def test_eq9_energy_grad_and_metric_apply(frs, key, with_prior):
    w = WORKLOADS[key]()
    ctx, eps = setup(frs, w)
    ctx.set_likelihood(1)
    k_gpu = ctx.get_noise_kernel().cpu().numpy()
    xi = (0.3 * np.random.default_rng(32).normal(size=(w.nfield, w.ny, w.nx))).astype(np.float32)
    g = ctx.new_latent()
    e = ctx.energy_grad(dev(xi), g, with_prior=with_prior)
    e_ref, g_ref = o.energy_grad_eq9(w.w_half, k_gpu, w.dirty, w.amp, w.mu, w.lognu, xi, with_prior)
    assert abs(e - e_ref) <= TOL * abs(e_ref)
    assert rel(g.cpu().numpy(), g_ref) <= TOL
    v = np.random.default_rng(33).normal(size=xi.shape).astype(np.float32)
    out = ctx.new_latent()
    ctx.metric_apply(dev(v), out, with_prior=with_prior)
    assert rel(out.cpu().numpy(), o.metric_apply_eq9(w.w_half, k_gpu, w.amp, w.mu, w.lognu, xi, v, with_prior)) <= TOL
    # back to the N' = R' limit: the same context gives the plain metric again
    ctx.set_likelihood(0)
    ctx.metric_apply(dev(v), out, with_prior=with_prior)
    assert rel(out.cpu().numpy(), o.metric_apply(w.w_half, w.amp, w.mu, w.lognu, xi, v, with_prior)) <= TOL


def test_eq9_cg_teacher_forced(frs):
    import torch
    w = WORKLOADS["c1"]()
    ctx, eps = setup(frs, w)
    ctx.set_likelihood(1)
    k_gpu = ctx.get_noise_kernel().cpu().numpy()
    xi = np.zeros((1, w.ny, w.nx), np.float32)
    g = ctx.new_latent()
    ctx.energy_grad(dev(xi), g, with_prior=True)
    s64 = o.sky(xi, w.amp, w.mu, w.lognu)
    ap = lambda u: o.metric_apply_eq9(w.w_half, k_gpu, w.amp, w.mu, w.lognu, xi, u, True, s=s64)  # noqa: E731
    b = (-g).contiguous()
    x = torch.zeros_like(b)
    ctx.cg_solve(b, x, 0)
    r, p, q, sc = ctx.cg_read_state()
    for k in range(5):
        x0, r0, p0 = (t.cpu().numpy().astype(np.float64) for t in (x, r, p))
        rr0 = float(sc[0])
        ctx.cg_step(x, True)
        r, p, q, sc = ctx.cg_read_state()
        st = o.cg_step(ap, x0, r0, p0, rr0)
        assert rel(q.cpu().numpy(), st["q"]) <= TOL
        assert abs(sc[3] - st["alpha"]) <= TOL * abs(st["alpha"])
        assert rel(x.cpu().numpy(), st["x"]) <= TOL


def test_eq9_full_size_config3(frs):
    """2048^2 (BASELINE.json configs[2]) in the launch configuration of that size."""
    w = wl.make_config(3)
    ctx, eps = setup(frs, w)
    ctx.set_likelihood(1)
    k_gpu = ctx.get_noise_kernel().cpu().numpy()
    k_ref = o.noise_kernel_from_psf(w.w_half[0], eps)
    assert np.max(np.abs(k_gpu[0] - k_ref)) <= TOL * np.max(k_ref)
    xi = (0.5 * np.random.default_rng(34).normal(size=(1, w.ny, w.nx))).astype(np.float32)
    g = ctx.new_latent()
    e = ctx.energy_grad(dev(xi), g, with_prior=True)
    e_ref, g_ref = o.energy_grad_eq9(w.w_half, k_gpu, w.dirty, w.amp, w.mu, w.lognu, xi, True)
    assert abs(e - e_ref) <= TOL * abs(e_ref)
    assert rel(g.cpu().numpy(), g_ref) <= TOL
    v = np.random.default_rng(35).normal(size=xi.shape).astype(np.float32)
    out = ctx.new_latent()
    ctx.metric_apply(dev(v), out, with_prior=True)
    assert rel(out.cpu().numpy(), o.metric_apply_eq9(w.w_half, k_gpu, w.amp, w.mu, w.lognu, xi, v, True)) <= TOL


# ------------------------------------------------------------------ MGVI samples and the sample-averaged KL (R15)
@pytest.mark.parametrize("key", ["c1", "multi"])
def test_mgvi_sample_and_kl_average(frs, key):
    import torch
    w = WORKLOADS[key]()
    ctx, eps = setup(frs, w)
    k_gpu = ctx.get_noise_kernel().cpu().numpy()
    rng = np.random.default_rng(50)
    xi = (0.2 * rng.normal(size=(w.nfield, w.ny, w.nx))).astype(np.float32)
    eta_xi = rng.normal(size=xi.shape).astype(np.float32)
    eta_d = rng.normal(size=(w.nchan, w.ny, w.nx)).astype(np.float32)
    sample = ctx.new_latent()
    ctx.sky_forward(dev(xi))
    with pytest.raises(frs.FrsError) as ei:                                   # sampling needs the Eq. 9 likelihood
        ctx.draw_sample(dev(eta_xi), dev(eta_d), sample, 3)
    assert ei.value.code == frs.binding.FRS_ESTATE
    ctx.set_likelihood(1)
    # the sample source m (0 CG iterations leave sigma = 0; read m back through one metric-free identity: max_iter = 0, then
    # compare sigma after a few iterations with the oracle's CG on the oracle's m -- both from the same white noise)
    iters = ctx.draw_sample(dev(eta_xi), dev(eta_d), sample, 4)
    assert iters == 4
    sg_ref, m_ref = o.draw_sample_eq9(w.w_half, k_gpu, w.amp, w.mu, w.lognu, xi, eta_xi, eta_d, cg_iters=4)
    r, p, q, sc = ctx.cg_read_state()
    # b = m is the right-hand side of that solve: r_0 = m; check it through the residual identity r_4 = m - M sigma_4
    s64 = o.sky(xi, w.amp, w.mu, w.lognu)
    resid = m_ref - o.metric_apply_eq9(w.w_half, k_gpu, w.amp, w.mu, w.lognu, xi, sample.cpu().numpy(), True, s=s64)
    assert np.linalg.norm(r.cpu().numpy() - resid) <= 1e-4 * np.linalg.norm(m_ref)
    assert rel(sample.cpu().numpy(), sg_ref) <= 1e-4
    # sample-averaged KL, gradient and metric on two mirrored samples
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
    # the position is back at the mean: a plain metric apply is the one at xi
    ctx.metric_apply(dev(v), out, with_prior=True)
    assert rel(out.cpu().numpy(), o.metric_apply_eq9(w.w_half, k_gpu, w.amp, w.mu, w.lognu, xi, v, True, s=s64)) <= TOL
    # not mirrored, one sample at sigma = 0: the plain energy and gradient
    z = torch.zeros((1,) + xi.shape, device="cuda")
    e0 = ctx.kl_energy_grad(dev(xi), z, g, mirrored=False)
    g0 = ctx.new_latent()
    e1 = ctx.energy_grad(dev(xi), g0, with_prior=True)
    assert e0 == e1 and torch.equal(g, g0)


def test_a_new_psf_discards_the_fitted_noise_kernel(frs):
    """frs.h (frs_set_noise_kernel): a later frs_set_psf* discards the kernel and returns to mode 0 -- for the image-space
    setter too, not only for frs_set_psf_weights: K was fitted to the old PSF."""
    w = WORKLOADS["c1"]()
    for setter in ("weights", "image"):
        ctx, eps = setup(frs, w)
        ctx.set_likelihood(1)
        if setter == "weights":
            ctx.set_psf_weights(dev(2.0 * w.w_half))
        else:
            psf = np.stack([o.psf_from_weights(2.0 * w.w_half[c]) for c in range(w.nchan)])
            ctx.set_psf(dev(psf))
        with pytest.raises(frs.FrsError) as ei:
            ctx.set_likelihood(1)                                            # no kernel any more
        assert ei.value.code == frs.binding.FRS_ESTATE
        with pytest.raises(frs.FrsError):
            ctx.get_noise_kernel()
        # mode 0 is in force again: the energy is that of the N' = R' limit with the new PSF
        xi = np.zeros((1, w.ny, w.nx), np.float32)
        g = ctx.new_latent()
        e = ctx.energy_grad(dev(xi), g, with_prior=True)
        e_ref, g_ref = o.energy_grad(2.0 * w.w_half, w.dirty, w.amp, w.mu, w.lognu, xi, True)
        assert abs(e - e_ref) <= TOL * abs(e_ref) and rel(g.cpu().numpy(), g_ref) <= TOL


def test_draws_into_fresh_buffers_agree_with_plain_launches(frs):
    """frs_draw_sample solves in a buffer of the context's own and copies the result out, so a caller that hands in a new
    `sample` buffer per draw (SampleShard.draw) replays one captured CG iteration instead of re-capturing it per draw; the
    samples are the same bits as with plain launches."""
    import torch
    w = WORKLOADS["c1"]()
    ctx, eps = setup(frs, w)
    ctx.set_likelihood(1)
    rng = np.random.default_rng(77)
    xi = (0.2 * rng.normal(size=(w.nfield, w.ny, w.nx))).astype(np.float32)
    ctx.sky_forward(dev(xi))
    etas = [(dev(rng.normal(size=xi.shape)), dev(rng.normal(size=(w.nchan, w.ny, w.nx)))) for _ in range(3)]
    graph = []
    for ex, ed in etas:
        out = torch.full_like(ex, float("nan"))                                  # a fresh buffer per draw
        assert ctx.draw_sample(ex, ed, out, 6) == 6
        graph.append(out)
    ctx.set_cuda_graphs(False)
    for (ex, ed), g in zip(etas, graph):
        out = torch.empty_like(ex)
        ctx.draw_sample(ex, ed, out, 6)
        assert torch.equal(out, g)
    assert not torch.equal(graph[0], graph[1])

