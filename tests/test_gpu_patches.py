"""Several Gaussian processes on patches (reading R20): PatchModel (C-ABI calls strung together) against
oracle/prior_oracle.py, plus the building blocks on their own."""
import numpy as np
import pytest

from gen import workloads as wl
from oracle import frs_oracle as fo
from oracle import prior_oracle as po

pytestmark = pytest.mark.gpu


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


def _setup(frs, n=128):
    w = wl.make_config(1, n=n, seed=4)
    mu = float(np.log(np.median(w.sky_true)))
    rng = np.random.default_rng(9)
    shapes = [((n, n), 0, 0, mu - 1.0), ((n // 2, n // 2), 10, 40, mu), ((n // 4, n // 2), 90, 5, mu + 0.5)]
    comps, ctxs = [], []
    for (ny, nx), y0, x0, m in shapes:
        amp = (wl.make_config(1, n=ny, seed=4) if ny == nx else wl.make_config(3, ny=ny, nx=nx, npts=2000)).amp[0].astype(np.float32)
        comps.append((amp.astype(np.float64), m, y0, x0))
        c = frs.Context(ny, nx, 1)
        c.set_amplitude(dev(amp[None]), [m])
        ctxs.append((c, y0, x0))
    field = frs.Context(n, n, 1)
    field.set_psf_weights(dev(w.w_half))
    field.set_dirty(dev(w.dirty))
    xis = [(0.3 * rng.normal(size=c[0].shape)).astype(np.float32) for c in comps]
    return w, comps, ctxs, field, xis, rng


@pytest.mark.parametrize("mode", [0, 1])
def test_patch_model_against_oracle(frs, mode):
    import torch
    from paper_2406_09144_b200.patches import PatchModel
    w, comps, ctxs, field, xis, rng = _setup(frs)
    kern = None
    model = PatchModel(field, ctxs)
    if mode == 1:
        field.set_noise_kernel(1e-2 * float(fo.psf_from_weights(w.w_half[0])[0, 0]))
        model.set_likelihood(1)
        kern = field.get_noise_kernel().cpu().numpy()[0].astype(np.float64)
    dxis = [dev(x[None]) for x in xis]
    grads = [torch.empty_like(x) for x in dxis]
    e = model.energy_grad(dxis, grads, True)
    e_ref, g_ref = po.energy_grad_patches(w.w_half[0], w.dirty[0], comps, xis, True, kern)
    assert abs(e - e_ref) <= 1e-5 * abs(e_ref)
    for g, r in zip(grads, g_ref):
        assert rel(g.cpu().numpy()[0], r) <= 1e-5
    assert rel(model.sky.cpu().numpy()[0], po.sky_patches(comps, xis, w.ny, w.nx)[0]) <= 1e-5
    vs = [rng.normal(size=x.shape).astype(np.float32) for x in xis]
    outs = [torch.empty_like(x) for x in dxis]
    model.metric_apply([dev(v[None]) for v in vs], outs, True)
    m_ref = po.metric_apply_patches(w.w_half[0], w.ny, w.nx, comps, xis, vs, True, kern)
    for o_, r in zip(outs, m_ref):
        assert rel(o_.cpu().numpy()[0], r) <= 1e-5


def test_building_blocks(frs):
    import torch
    w, comps, ctxs, field, xis, rng = _setup(frs, 128)
    s = np.exp(0.3 * rng.normal(size=(128, 128))).astype(np.float32)
    g = torch.empty(1, 128, 128, device="cuda")
    e = field.sky_energy_grad(dev(s[None]), g)
    cs = fo.psf_apply(w.w_half[0], s)
    assert abs(e - (0.5 * np.sum(s * cs) - np.sum(w.dirty[0] * s))) <= 1e-5 * abs(e)
    # C s - j is a difference: held to 1e-5 of its operands
    assert np.linalg.norm(g.cpu().numpy()[0] - (cs - w.dirty[0])) <= 1e-5 * (np.linalg.norm(cs) + np.linalg.norm(w.dirty[0]))
    c, y0, x0 = ctxs[1]                                                      # the 64 x 64 component
    amp, mu = comps[1][0], comps[1][1]
    xi = xis[1]
    part = torch.empty(1, 64, 64, device="cuda")
    c.sky_forward(dev(xi[None]), part)
    sk = np.exp(mu + fo.hartley2(amp * xi))
    v = rng.normal(size=(64, 64)).astype(np.float32)
    out = torch.empty_like(part)
    c.latent_jvp(dev(v[None]), out)
    assert rel(out.cpu().numpy()[0], sk * fo.hartley2(amp * v)) <= 1e-5
    c.latent_vjp(dev(v[None]), out, add=dev(xi[None]))
    assert rel(out.cpu().numpy()[0], amp * fo.hartley2(sk * v) + xi) <= 1e-5
    # insert / crop are exact; a patch sticking out is refused
    f = torch.zeros(1, 128, 128, device="cuda")
    field.patch_insert_add(part, y0, x0, f)
    field.patch_insert_add(part, y0, x0, f)
    back = torch.empty_like(part)
    field.patch_crop(f, y0, x0, back)
    assert torch.equal(back, part + part) and float(f.sum()) == float((part + part).sum())
    with pytest.raises(frs.FrsError):
        field.patch_insert_add(part, 70, 70, f)
    assert abs(c.dot(part, part) - float((part.double() ** 2).sum())) <= 1e-12 * float((part.double() ** 2).sum())
