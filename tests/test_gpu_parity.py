"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element, on the
same seeded fp32-rounded inputs.  Tolerances (BASELINE.json north_star): relative L2 <= 1e-5 for sky,
convolution and gradient, <= 1e-4 after 20 CG iterations; exact for index/padding layouts."""
import numpy as np
import pytest

from gen import workloads as wl
from oracle import frs_oracle as o

pytestmark = pytest.mark.gpu

TOL = 1e-5


def rel(a, b):
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
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


def make_ctx(frs, w, with_model=True):
    ctx = frs.Context(w.ny, w.nx, w.nchan)
    ctx.set_psf_weights(dev(w.w_half))
    ctx.set_dirty(dev(w.dirty))
    if with_model:
        ctx.set_amplitude(dev(w.amp), w.mu)
        ctx.set_channel_lognu(w.lognu)
    return ctx


_CACHE = {}


def workload(key):
    if key not in _CACHE:
        kind = key[0]
        if kind == "c1":
            _CACHE[key] = wl.make_config(1)
        elif kind == "c1b":
            _CACHE[key] = wl.make_config(1, sigma_rel=0.1)
        elif kind == "rect":
            _CACHE[key] = wl.make_config(3, ny=key[1], nx=key[2])
        elif kind == "sq":
            _CACHE[key] = wl.make_config(key[1], n=key[2])
        elif kind == "multi":
            _CACHE[key] = wl.make_config(5, n=key[1], nchan=key[2])
    return _CACHE[key]


SHAPES = [("rect", 32, 32), ("rect", 64, 128), ("rect", 256, 64), ("sq", 2, 512), ("rect", 32, 1024), ("rect", 2048, 32)]


# ---------------------------------------------------------------------------------- convolution (Eq. 14)
@pytest.mark.parametrize("key", SHAPES)
def test_psf_apply_matches_oracle(frs, key):
    w = workload(key)
    ctx = make_ctx(frs, w, with_model=False)
    rng = np.random.default_rng(1)
    x = rng.normal(size=(1, w.ny, w.nx)).astype(np.float32)
    y = ctx.new_image()
    ctx.psf_apply(dev(x), y)
    ref = o.psf_apply(w.w_half[0], x[0])
    assert rel(y.cpu().numpy()[0], ref) <= TOL
    # truth-like positive input with point sources
    ctx.psf_apply(dev(w.sky_true), y)
    assert rel(y.cpu().numpy()[0], o.psf_apply(w.w_half[0], w.sky_true[0])) <= TOL


def test_index_and_padding_layout_exact(frs):
    """Index / padding layout: delta images must put the PSF peak exactly where the delta was (corner
    deltas exercise the wrapped half of the PSF and the crop), and with W == 1 (C = My Mx identity)
    an integer-valued image must come back exactly after rounding."""
    ny, nx = 64, 128
    w = wl.make_config(1, ny=ny, nx=nx, npts=300)
    counts = w.w_counts.astype(np.float32)                        # small integers
    assert counts.max() <= 8
    ctx = frs.Context(ny, nx, 1)
    ctx.set_psf_weights(dev(counts))
    psf = o.psf_from_weights(counts[0].astype(np.float64))
    y = ctx.new_image()
    for (y0, x0) in [(0, 0), (0, nx - 1), (ny - 1, 0), (ny - 1, nx - 1), (17, 93)]:
        d = np.zeros((1, ny, nx), np.float32)
        d[0, y0, x0] = 1.0
        ctx.psf_apply(dev(d), y)
        got = y.cpu().numpy()[0].astype(np.float64)
        exp = np.array([[psf[(a - y0) % (2 * ny), (b - x0) % (2 * nx)] for b in range(nx)] for a in range(ny)])
        assert np.unravel_index(np.argmax(got), got.shape) == (y0, x0)
        assert np.rint(got[y0, x0]) == psf[0, 0]                     # the peak = sum of weights (an integer)
        assert np.max(np.abs(got - exp)) <= 2e-6 * psf[0, 0]
    ones = np.ones((1, 2 * ny, nx + 1), np.float32)
    ctx.set_psf_weights(dev(ones))
    img = np.random.default_rng(0).integers(-50, 50, size=(1, ny, nx)).astype(np.float32)
    ctx.psf_apply(dev(img), y)
    assert np.array_equal(np.rint(y.cpu().numpy() / (4.0 * ny * nx)), img)


def test_psf_apply_linearity_zero_and_symmetry(frs):
    w = workload(("rect", 64, 128))
    ctx = make_ctx(frs, w, with_model=False)
    import torch
    z = torch.zeros((1, w.ny, w.nx), device="cuda")
    y = ctx.new_image()
    ctx.psf_apply(z, y)
    assert float(y.abs().max()) == 0.0
    rng = np.random.default_rng(2)
    a, b = rng.normal(size=(2, 1, w.ny, w.nx)).astype(np.float32)
    ya, yb = ctx.new_image(), ctx.new_image()
    ctx.psf_apply(dev(a), ya)
    ctx.psf_apply(dev(b), yb)
    lhs = float((ya.double() * dev(b).double()).sum())
    rhs = float((dev(a).double() * yb.double()).sum())
    assert abs(lhs - rhs) <= 1e-5 * max(abs(lhs), abs(rhs), float(ya.double().norm() * np.linalg.norm(b)) * 1e-1)


def test_set_psf_from_image_space_psf(frs):
    w = workload(("rect", 64, 128))
    psf = o.psf_from_weights(w.w_half[0].astype(np.float64)).astype(np.float32)
    ctx = frs.Context(w.ny, w.nx, 1)
    ctx.set_psf(dev(psf[None]))
    x = np.random.default_rng(3).normal(size=(1, w.ny, w.nx)).astype(np.float32)
    y = ctx.new_image()
    ctx.psf_apply(dev(x), y)
    ref = o.psf_apply(o.psf_spectrum_from_psf(psf.astype(np.float64))[0], x[0])
    assert rel(y.cpu().numpy()[0], ref) <= 3e-5      # W itself went through an fp32 transform here
    bad = psf.copy()
    bad[1, 2] += 0.3 * psf[0, 0]
    with pytest.raises(frs.FrsError) as e:
        ctx.set_psf(dev(bad[None]))
    assert e.value.code == frs.FRS_ENOTPSD


def test_error_behaviour(frs):
    import torch
    with pytest.raises(frs.FrsError):
        frs.Context(48, 64)
    ctx = frs.Context(64, 64, 1)
    x = torch.zeros((1, 64, 64), device="cuda")
    with pytest.raises(frs.FrsError) as e:
        ctx.psf_apply(x, ctx.new_image())                         # PSF not set
    assert e.value.code == frs.FRS_ESTATE
    neg = torch.full((1, 128, 65), -1.0, device="cuda")
    with pytest.raises(frs.FrsError) as e:
        ctx.set_psf_weights(neg)
    assert e.value.code == frs.FRS_ENOTPSD
    ctx.set_psf_weights(neg.abs())
    with pytest.raises(frs.FrsError) as e:
        ctx.sky_metric_apply(x, ctx.new_image())                  # no position
    assert e.value.code == frs.FRS_ESTATE
    with pytest.raises(ValueError):
        ctx.psf_apply(torch.zeros((1, 64, 32), device="cuda"), ctx.new_image())


# ---------------------------------------------------------------------------------- sky, L1 apply
@pytest.mark.parametrize("key", [("c1",), ("rect", 64, 128), ("sq", 2, 512), ("multi", 64, 3)])
def test_sky_forward_and_sky_metric_apply(frs, key):
    w = workload(key)
    ctx = make_ctx(frs, w)
    rng = np.random.default_rng(4)
    xi = (0.5 * rng.normal(size=(w.nfield, w.ny, w.nx))).astype(np.float32)
    s = ctx.new_image()
    ctx.sky_forward(dev(xi), s)
    s_ref = o.sky(xi, w.amp, w.mu, w.lognu)
    assert rel(s.cpu().numpy(), s_ref) <= TOL
    x = rng.normal(size=(w.nchan, w.ny, w.nx)).astype(np.float32)
    y = ctx.new_image()
    ctx.sky_metric_apply(dev(x), y)
    s32 = s.cpu().numpy()                      # teacher-forced on the GPU's own fp32 sky
    ref = o.sky_metric_apply(w.w_half, s32, x)
    for c in range(w.nchan):
        assert rel(y.cpu().numpy()[c], ref[c]) <= TOL
    # host-buffer entry point gives the same numbers
    import torch
    xh = torch.from_numpy(x).pin_memory()
    yh = torch.empty_like(xh).pin_memory()
    ctx.sky_metric_apply_host(xh, yh)
    assert np.array_equal(yh.numpy(), y.cpu().numpy())


# ---------------------------------------------------------------------------------- energy, gradient, metric
@pytest.mark.parametrize("key", [("c1",), ("rect", 64, 128), ("sq", 2, 512), ("multi", 64, 3)])
@pytest.mark.parametrize("with_prior", [True, False])
def test_energy_grad_and_metric_apply(frs, key, with_prior):
    w = workload(key)
    ctx = make_ctx(frs, w)
    rng = np.random.default_rng(5)
    xi = (0.3 * rng.normal(size=(w.nfield, w.ny, w.nx))).astype(np.float32)
    g = ctx.new_latent()
    e = ctx.energy_grad(dev(xi), g, with_prior=with_prior)
    e_ref, g_ref = o.energy_grad(w.w_half, w.dirty, w.amp, w.mu, w.lognu, xi, with_prior)
    assert abs(e - e_ref) <= 1e-5 * abs(e_ref) + 1e-6 * np.abs(g_ref).sum() * 0
    assert rel(g.cpu().numpy(), g_ref) <= TOL
    v = rng.normal(size=(w.nfield, w.ny, w.nx)).astype(np.float32)
    out = ctx.new_latent()
    ctx.metric_apply(dev(v), out, with_prior=with_prior)
    ref = o.metric_apply(w.w_half, w.amp, w.mu, w.lognu, xi, v, with_prior)
    assert rel(out.cpu().numpy(), ref) <= TOL


def test_energy_device_scalar_and_xi_zero(frs):
    import torch
    w = workload(("c1",))
    ctx = make_ctx(frs, w)
    xi = torch.zeros((1, w.ny, w.nx), device="cuda")
    g = ctx.new_latent()
    d_e = torch.zeros(1, dtype=torch.float64, device="cuda")
    e = ctx.energy_grad(xi, g, with_prior=True, d_energy=d_e)
    assert float(d_e.cpu()[0]) == e
    e_ref, g_ref = o.energy_grad(w.w_half, w.dirty, w.amp, w.mu, w.lognu, np.zeros((1, w.ny, w.nx)), True)
    assert abs(e - e_ref) <= 1e-5 * abs(e_ref)
    assert rel(g.cpu().numpy(), g_ref) <= TOL


def test_non_hermitian_weights_are_rejected(frs):
    """W[-k] = W[k] (R4) is implied by the half grid except on the self-conjugate columns kx = 0 and kx = nx, where both
    members of a pair are stored: a mismatch there would make the two orientations of the operator differ silently."""
    w = workload(("c1",))
    for kx in (0, w.nx):
        bad = w.w_half.copy()
        bad[0, 3, kx] += 1.0                                      # its partner (2 ny - 3, kx) is left alone
        ctx = frs.Context(w.ny, w.nx, 1)
        with pytest.raises(frs.FrsError) as ei:
            ctx.set_psf_weights(dev(bad))
        assert ei.value.code == frs.binding.FRS_ENOTPSD
        ok = w.w_half.copy()
        ok[0, 3, kx] += 1.0
        ok[0, 2 * w.ny - 3, kx] += 1.0
        ctx.set_psf_weights(dev(ok))


def test_cg_rtol_stops_on_the_device_at_the_right_iterate(frs):
    """The stopping test runs on the device; the host only looks every 8 iterations, and the iterations enqueued past
    the stopping point must leave x untouched: x equals the iterate of a run with max_iter = the reported count."""
    import torch
    w, ctx, b, ap = _cg_problem(frs, ("c1b",))
    x = torch.zeros_like(b)
    it, rn = ctx.cg_solve(b, x, 200, rtol=1e-2)
    assert 0 < it < 200 and it % 8 != 0 or it < 200
    assert rn <= 1e-2 * float(b.double().norm())
    x2 = torch.zeros_like(b)
    it2, rn2 = ctx.cg_solve(b, x2, it)
    assert it2 == it and torch.equal(x, x2) and rn2 == rn
    x3 = torch.zeros_like(b)
    it3, rn3 = ctx.cg_solve(b, x3, it - 1)
    assert rn3 > 1e-2 * float(b.double().norm())                   # one iteration earlier the criterion was not met


def test_cg_graph_replay_equals_plain_launches(frs):
    """frs_cg_solve replays iterations 1.. as one captured CUDA graph (the iteration index lives on the device): same
    kernels on the same data, so x, the residual history and the iteration count must be bit-identical to plain
    launches -- without and with the stopping test, single- and multi-channel, and in the Eq. 9 mode."""
    import torch
    for key, mode in ((("c1b",), 0), (("multi", 64, 3), 0), (("c1b",), 1)):
        w, ctx, b, ap = _cg_problem(frs, key)
        if mode == 1:
            ctx.set_noise_kernel(1e-2 * float(np.sum(w.w_half[0][:, 0]) + 2 * np.sum(w.w_half[0][:, 1:-1]) + np.sum(w.w_half[0][:, -1])))
            ctx.set_likelihood(1)
        out = {}
        for on in (1, 0, 1):
            ctx.set_cuda_graphs(on)
            l0 = ctx.launch_count()
            x = torch.zeros_like(b)
            hist = torch.zeros(21, dtype=torch.float64, device="cuda")
            it, rn = ctx.cg_solve(b, x, 20, res_history=hist)
            xr = torch.zeros_like(b)
            itr, rnr = ctx.cg_solve(b, xr, 200, rtol=1e-2)
            res = (x.clone(), hist.clone(), it, rn, xr.clone(), itr, rnr, ctx.launch_count() - l0)
            if on in out and on == 1:
                prev = out[1]                                      # the cached graph of the first round is reused
                assert torch.equal(prev[0], res[0]) and torch.equal(prev[4], res[4])
            out[on] = res
        g, e = out[1], out[0]
        assert torch.equal(g[0], e[0]) and torch.equal(g[1], e[1]) and g[2] == e[2] == 20 and g[3] == e[3]
        assert torch.equal(g[4], e[4]) and g[5] == e[5] and g[6] == e[6]
        assert g[7] == e[7] > 0                                    # the launch count is kept honest under replay


# ---------------------------------------------------------------------------------- CG (protocol of DESIGN.md R9)
def _cg_problem(frs, key):
    import torch
    w = workload(key)
    ctx = make_ctx(frs, w)
    xi = np.zeros((w.nfield, w.ny, w.nx), np.float32)
    g = ctx.new_latent()
    ctx.energy_grad(dev(xi), g, with_prior=True)
    b = (-g).contiguous()
    s32 = ctx.new_image()
    ctx.sky_forward(dev(xi), s32)
    s = s32.cpu().numpy().astype(np.float64)
    ap = lambda v: o.metric_apply(w.w_half, w.amp, w.mu, w.lognu, xi, v, True, s=s)
    return w, ctx, b, ap


def test_cg_teacher_forced_every_iteration(frs):
    """At every k <= 20 the oracle takes the GPU's own (x_k, r_k, p_k) and recomputes one step."""
    import torch
    w, ctx, b, ap = _cg_problem(frs, ("c1",))
    x = torch.zeros_like(b)
    ctx.cg_solve(b, x, 0)                                          # initialises r = p = b, rr
    r, p, q, sc = ctx.cg_read_state()
    assert rel(r.cpu().numpy(), b.cpu().numpy()) == 0.0
    for k in range(20):
        x0, r0, p0, rr0 = x.cpu().numpy().astype(np.float64), r.cpu().numpy().astype(np.float64), \
            p.cpu().numpy().astype(np.float64), float(sc[0])
        assert abs(rr0 - np.sum(r0 * r0)) <= 1e-10 * rr0
        ctx.cg_step(x, True)
        r, p, q, sc = ctx.cg_read_state()
        st = o.cg_step(ap, x0, r0, p0, rr0)
        assert rel(q.cpu().numpy(), st["q"]) <= TOL
        assert abs(sc[3] - st["alpha"]) <= TOL * abs(st["alpha"])
        assert abs(sc[4] - st["beta"]) <= 1e-4 * abs(st["beta"])
        assert rel(x.cpu().numpy(), st["x"]) <= TOL
        # r and p: the update's own rounding is measured against the size of the operands
        assert np.linalg.norm(r.cpu().numpy() - st["r"]) <= TOL * np.linalg.norm(r0)
        assert np.linalg.norm(p.cpu().numpy() - st["p"]) <= TOL * np.linalg.norm(p0)
        assert st["pq"] > 0


def test_cg_free_running_within_horizon_and_literal(frs):
    import torch
    w, ctx, b, ap = _cg_problem(frs, ("c1",))
    bh = b.cpu().numpy().astype(np.float64)
    sol = o.cg(ap, bh, max_iter=20, keep=True)
    # the envelope is a random quantity (one seeded noise draw per apply): take the upper envelope of
    # four draws, so that the horizon does not hinge on one lucky realisation (R9)
    env = np.max([o.cg_fp32_envelope(ap, bh, max_iter=20, seed=sd) for sd in (1234, 1235, 1236, 1237)], axis=0)
    horizon = max([k + 1 for k in range(20) if env[k] <= 2e-5] or [0])
    assert horizon >= 5
    hist = torch.zeros(21, dtype=torch.float64, device="cuda")
    errs = []
    for k in range(1, 21):
        x = torch.zeros_like(b)
        it, rn = ctx.cg_solve(b, x, k, res_history=hist)
        assert it == k
        errs.append(rel(x.cpu().numpy(), sol["xs"][k - 1]))
    for k in range(1, horizon + 1):
        assert errs[k - 1] <= 1e-4, (k, errs[k - 1])
    assert errs[19] <= max(1e-4, 3 * env[19]), (errs[19], env[19])   # literal x_20, reported vs envelope
    h = hist.cpu().numpy()
    assert h[20] < h[0] and abs(h[0] - np.linalg.norm(bh)) <= 1e-6 * h[0]


def test_cg_split_step_equals_fused_step(frs):
    """frs_cg_step_begin / frs_cg_step_end (the channel-sharded iteration, world size 1: nothing to
    sum) reproduces frs_cg_step up to the rounding of the separately added prior term."""
    import torch
    w, ctx, b, ap = _cg_problem(frs, ("c1",))
    xa, xb = torch.zeros_like(b), torch.zeros_like(b)
    ctx.cg_solve(b, xa, 0)
    for _ in range(4):
        ctx.cg_step(xa, True)
    ctx.cg_solve(b, xb, 0)
    for _ in range(4):
        q = ctx.cg_step_begin()
        assert q.shape == b.shape and q.data_ptr() % 16 == 0
        ctx.cg_step_end(xb, True)
    assert rel(xb.cpu().numpy(), xa.cpu().numpy()) <= TOL


def test_cg_literal_on_well_conditioned_companion(frs):
    """config 1b (sigma = 0.1 peak): rel L2(x_20) <= 1e-4 literally."""
    import torch
    w, ctx, b, ap = _cg_problem(frs, ("c1b",))
    sol = o.cg(ap, b.cpu().numpy().astype(np.float64), max_iter=20)
    x = torch.zeros_like(b)
    it, rn = ctx.cg_solve(b, x, 20)
    assert it == 20
    assert rel(x.cpu().numpy(), sol["x"]) <= 1e-4
    # both have converged to the fp32 floor of the recurrence: compare against ||b||, not each other
    bn = float(b.double().norm())
    assert rn <= 1e-5 * bn and sol["res"][-1] <= 1e-5 * bn
    # rtol stop
    x2 = torch.zeros_like(b)
    it2, rn2 = ctx.cg_solve(b, x2, 200, rtol=1e-3)
    assert it2 < 200 and rn2 <= 1e-3 * float(b.double().norm()) * 1.001


def test_cg_multichannel_teacher_forced(frs):
    import torch
    w, ctx, b, ap = _cg_problem(frs, ("multi", 64, 3))
    x = torch.zeros_like(b)
    ctx.cg_solve(b, x, 0)
    r, p, q, sc = ctx.cg_read_state()
    for k in range(3):
        x0, r0, p0, rr0 = (t.cpu().numpy().astype(np.float64) for t in (x, r, p)), None, None, float(sc[0])
        x0, r0, p0 = list(x0)
        ctx.cg_step(x, True)
        r, p, q, sc = ctx.cg_read_state()
        st = o.cg_step(ap, x0, r0, p0, rr0)
        assert rel(q.cpu().numpy(), st["q"]) <= TOL
        assert rel(x.cpu().numpy(), st["x"]) <= TOL


def test_outer_newton_steps_teacher_forced(frs):
    """config-2 recipe (reduced): outer KL steps x CG; at each visited xi (the GPU's) the oracle
    recomputes s, E, grad (reading R10)."""
    import torch
    w = workload(("sq", 2, 128))
    ctx = make_ctx(frs, w)
    xi = torch.zeros((1, w.ny, w.nx), device="cuda")
    g = ctx.new_latent()
    e_prev = None
    for step in range(3):
        e = ctx.energy_grad(xi, g, with_prior=True)
        xih = xi.cpu().numpy()
        e_ref, g_ref = o.energy_grad(w.w_half, w.dirty, w.amp, w.mu, w.lognu, xih, True)
        assert abs(e - e_ref) <= 1e-5 * abs(e_ref)
        assert rel(g.cpu().numpy(), g_ref) <= TOL
        if e_prev is not None:
            assert e < e_prev
        e_prev = e
        b = (-g).contiguous()
        d = torch.zeros_like(b)
        ctx.cg_solve(b, d, 10)
        scale = 1.0
        gt = ctx.new_latent()
        for _ in range(5):
            e1 = ctx.energy_grad((xi + scale * d).contiguous(), gt, with_prior=True)
            if e1 < e:
                break
            scale *= 0.5
        xi = (xi + scale * d).contiguous()


def _check_l2_apply_and_one_cg_step(frs, ctx, w, xi, s32):
    """Latent metric apply (with and without the prior term) and ONE teacher-forced CG step at the position xi,
    in the launch configuration of this size: the oracle repeats the step from the GPU's own (x, r, p, rr)."""
    import torch
    s64 = s32.astype(np.float64)
    ap = lambda v, pr=True: o.metric_apply(w.w_half, w.amp, w.mu, w.lognu, xi, v, pr, s=s64)  # noqa: E731
    v = np.random.default_rng(11).normal(size=xi.shape).astype(np.float32)
    out = ctx.new_latent()
    ctx.metric_apply(dev(v), out, with_prior=True)
    mv = ap(v)
    assert rel(out.cpu().numpy(), mv) <= TOL
    ctx.metric_apply(dev(v), out, with_prior=False)
    assert rel(out.cpu().numpy(), mv - v.astype(np.float64)) <= TOL
    b = dev(np.random.default_rng(12).normal(size=xi.shape).astype(np.float32))
    x = torch.zeros_like(b)
    ctx.cg_solve(b, x, 0)                                          # r = p = b, rr = <b, b>
    r, p, q, sc = ctx.cg_read_state()
    x0, r0, p0, rr0 = (t.cpu().numpy().astype(np.float64) for t in (x, r, p)), None, None, float(sc[0])
    x0, r0, p0 = list(x0)
    assert abs(rr0 - np.sum(r0 * r0)) <= 1e-10 * rr0
    ctx.cg_step(x, True)
    r, p, q, sc = ctx.cg_read_state()
    st = o.cg_step(ap, x0, r0, p0, rr0)
    assert rel(q.cpu().numpy(), st["q"]) <= TOL
    assert abs(sc[3] - st["alpha"]) <= TOL * abs(st["alpha"])
    assert rel(x.cpu().numpy(), st["x"]) <= TOL
    # r+ = r - alpha q: its rounding is measured against the size of the two operands
    assert np.linalg.norm(r.cpu().numpy() - st["r"]) <= TOL * (np.linalg.norm(r0) + abs(st["alpha"]) * np.linalg.norm(st["q"]))
    assert abs(sc[4] - st["beta"]) <= 1e-4 * abs(st["beta"])


# ---------------------------------------------------------------------------------- full-size configs
@pytest.mark.parametrize("cfg", [3, 4])
def test_full_size_config_parity(frs, cfg, monkeypatch):
    """BASELINE.json configs 3 and 4 at full size, in the launch configuration bench.py times:
    sky, C s (through the L1 apply) and gradient against the full fp64 oracle.  The context runs with guard zones around
    every array it owns (FRS_GUARD, the stand-in for memcheck): none may be touched at these launch shapes."""
    import torch
    monkeypatch.setenv("FRS_GUARD", "1")
    w = wl.make_config(cfg)
    ctx = make_ctx(frs, w)
    xi = (0.5 * np.random.default_rng(6).normal(size=(1, w.ny, w.nx))).astype(np.float32)
    s = ctx.new_image()
    ctx.sky_forward(dev(xi), s)
    s32 = s.cpu().numpy()
    assert rel(s32, o.sky(xi, w.amp, w.mu, w.lognu)) <= TOL
    x = np.random.default_rng(7).normal(size=(1, w.ny, w.nx)).astype(np.float32)
    y = ctx.new_image()
    ctx.sky_metric_apply(dev(x), y)
    assert rel(y.cpu().numpy()[0], o.sky_metric_apply(w.w_half, s32, x)[0]) <= TOL
    ctx.psf_apply(dev(w.sky_true), y)
    assert rel(y.cpu().numpy()[0], o.psf_apply(w.w_half[0], w.sky_true[0])) <= TOL
    g = ctx.new_latent()
    e = ctx.energy_grad(dev(xi), g, with_prior=True)
    e_ref, g_ref = o.energy_grad(w.w_half, w.dirty, w.amp, w.mu, w.lognu, xi, True)
    assert abs(e - e_ref) <= 1e-5 * abs(e_ref)
    assert rel(g.cpu().numpy(), g_ref) <= TOL
    _check_l2_apply_and_one_cg_step(frs, ctx, w, xi, s32)
    bad, n = ctx.check_guards()
    assert bad == 0 and n >= 10, (bad, n)
    del ctx
    torch.cuda.empty_cache()


def test_config5_multichannel_parity(frs, monkeypatch):
    """config 5 (16 x 1024^2, two latent fields): per-channel L1 apply and the gradient (guard zones on, as above)."""
    monkeypatch.setenv("FRS_GUARD", "1")
    w = wl.make_config(5)
    ctx = make_ctx(frs, w)
    xi = (0.5 * np.random.default_rng(8).normal(size=(2, w.ny, w.nx))).astype(np.float32)
    s = ctx.new_image()
    ctx.sky_forward(dev(xi), s)
    s32 = s.cpu().numpy()
    assert rel(s32, o.sky(xi, w.amp, w.mu, w.lognu)) <= TOL
    x = np.random.default_rng(9).normal(size=(w.nchan, w.ny, w.nx)).astype(np.float32)
    y = ctx.new_image()
    ctx.sky_metric_apply(dev(x), y)
    ref = o.sky_metric_apply(w.w_half, s32, x)
    yh = y.cpu().numpy()
    for c in range(w.nchan):
        assert rel(yh[c], ref[c]) <= TOL
    g = ctx.new_latent()
    e = ctx.energy_grad(dev(xi), g, with_prior=True)
    e_ref, g_ref = o.energy_grad(w.w_half, w.dirty, w.amp, w.mu, w.lognu, xi, True)
    assert abs(e - e_ref) <= 1e-5 * abs(e_ref)
    assert rel(g.cpu().numpy(), g_ref) <= TOL
    _check_l2_apply_and_one_cg_step(frs, ctx, w, xi, s32)
    bad, n = ctx.check_guards()
    assert bad == 0 and n >= 10, (bad, n)


def test_config2_as_stated_outer_steps_teacher_forced(frs):
    """BASELINE.json configs[1] as stated: 512^2, 5 outer KL steps x 50 CG iterations (reading R10: zero-sample
    Newton-CG with step halving).  Teacher-forced: at every xi the GPU visits, the oracle recomputes s, E and the
    gradient; the energy must go down from step to step and every solve must run its 50 iterations."""
    import torch
    w = wl.make_config(2)
    assert (w.ny, w.nx) == (512, 512)
    ctx = make_ctx(frs, w)
    xi = torch.zeros((1, w.ny, w.nx), device="cuda")
    g, gt, s = ctx.new_latent(), ctx.new_latent(), ctx.new_image()
    e_prev = None
    for step in range(5):
        e = ctx.energy_grad(xi, g, with_prior=True)
        xih = xi.cpu().numpy()
        ctx.sky_forward(xi, s)
        assert rel(s.cpu().numpy(), o.sky(xih, w.amp, w.mu, w.lognu)) <= TOL
        e_ref, g_ref = o.energy_grad(w.w_half, w.dirty, w.amp, w.mu, w.lognu, xih, True)
        assert abs(e - e_ref) <= 1e-5 * abs(e_ref)
        # Near the optimum the gradient J^T (C s - j) + xi is a cancellation (80-fold at the fifth step: |g| = 1e5 out of
        # operands of 8e6), so there the error is held to 1e-6 of the operands J^T C s and J^T j; elsewhere to 1e-5 of g.
        s64 = o.sky(xih, w.amp, w.mu, w.lognu)
        ops = np.linalg.norm(o.vjp(w.amp, w.lognu, s64, np.stack([o.psf_apply(w.w_half[0], s64[0])]))) \
            + np.linalg.norm(o.vjp(w.amp, w.lognu, s64, w.dirty.astype(np.float64)))
        err = np.linalg.norm(g.cpu().numpy().astype(np.float64) - g_ref)
        assert err <= max(TOL * np.linalg.norm(g_ref), 1e-6 * ops), (step, err, np.linalg.norm(g_ref), ops)
        if step == 0:
            assert err <= TOL * np.linalg.norm(g_ref)
        if e_prev is not None:
            assert e < e_prev
        e_prev = e
        b = (-g).contiguous()
        d = torch.zeros_like(b)
        it, rn = ctx.cg_solve(b, d, 50)
        assert it == 50 and np.isfinite(rn)
        scale = 1.0
        for _ in range(5):
            e1 = ctx.energy_grad((xi + scale * d).contiguous(), gt, with_prior=True)
            if e1 < e:
                break
            scale *= 0.5
        assert e1 < e
        xi = (xi + scale * d).contiguous()


def test_tensor_core_stage_measurement_runs(frs):
    """The measurement behind the decision not to run DFT stages on the tensor cores: tcgen05.mma
    kind::tf32 at the shape of a radix-16 stage.  24 instructions (3-term split, both output parities) per column pair
    against the 640 SM-cycles of the packed-FP32 butterflies: recorded in profiles/r2_tensor_core_stage.md."""
    clk = frs.selftest_tcgen05_stage(64, 24, 500)
    assert 8.0 < clk < 1000.0
    print(f"tcgen05.mma kind::tf32 M=128 K=8 N=64: {clk:.1f} clk per instruction -> {24 * clk:.0f} clk per stage and column pair")


def test_host_batch_apply_equals_single_calls(frs):
    """frs_sky_metric_apply_host_batch overlaps copies and kernels of neighbouring items on its own streams: every result
    must be bit-identical to the one-apply-per-call entry point, also when buffers are reused two items later."""
    import torch
    w = workload(("sq", 2, 512))
    ctx = make_ctx(frs, w)
    xi = (0.3 * np.random.default_rng(0).normal(size=(1, w.ny, w.nx))).astype(np.float32)
    ctx.sky_forward(dev(xi))
    rng = np.random.default_rng(1)
    xs = [torch.from_numpy(rng.normal(size=(1, w.ny, w.nx)).astype(np.float32)).pin_memory() for _ in range(5)]
    ref = []
    for x in xs:
        y = torch.empty_like(x).pin_memory()
        ctx.sky_metric_apply_host(x, y)
        ref.append(y.clone())
    ys = [torch.empty_like(xs[0]).pin_memory() for _ in range(5)]
    ctx.sky_metric_apply_host_batch(xs, ys)
    assert all(torch.equal(a, b) for a, b in zip(ys, ref))
    # two input and two output buffers rotated: the last two results survive
    ctx.sky_metric_apply_host_batch([xs[0], xs[1], xs[2], xs[3]], [ys[0], ys[1], ys[0], ys[1]])
    assert torch.equal(ys[0], ref[2]) and torch.equal(ys[1], ref[3])
    ctx.sky_metric_apply_host_batch([], [])
    y_dev = ctx.new_image()
    ctx.sky_metric_apply(xs[4].cuda(), y_dev)
    assert torch.equal(y_dev.cpu(), ref[4])


@pytest.mark.parametrize("key", [("sq", 2, 1024), ("rect", 2048, 1024), ("rect", 1024, 4096)])
def test_fused_inverse_and_hartley_row_pass_equals_separate_passes(frs, key):
    """The fused kernel (rows_inv + the row pass of the following Hartley transform) against the two separate passes:
    same arithmetic on the same data, so gradient and metric agree to rounding (1e-6), the energy to fp64 summation order;
    both likelihood modes.  (Against the oracle the fused path is the default of every other test.)"""
    w = workload(key)
    ctx = make_ctx(frs, w)
    rng = np.random.default_rng(3)
    xi = dev(0.3 * rng.normal(size=(1, w.ny, w.nx)))
    v = dev(rng.normal(size=(1, w.ny, w.nx)))
    for mode in (0, 1):
        if mode == 1:
            ctx.set_noise_kernel(1e-2 * float(o.psf_from_weights(w.w_half[0])[0, 0]))
            ctx.set_likelihood(1)
        res = {}
        for fused in (1, 0):
            ctx.set_fused_passes(fused)
            g, out = ctx.new_latent(), ctx.new_latent()
            e = ctx.energy_grad(xi, g, with_prior=True)
            ctx.metric_apply(v, out, with_prior=True)
            res[fused] = (e, g.cpu().numpy(), out.cpu().numpy())
        assert abs(res[1][0] - res[0][0]) <= 1e-10 * abs(res[0][0])
        assert rel(res[1][1], res[0][1]) <= 1e-6 and rel(res[1][2], res[0][2]) <= 1e-6
        assert not np.array_equal(res[1][1], np.zeros_like(res[1][1]))
