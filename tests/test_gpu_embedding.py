"""Images that are not a power of two (3600^2), embedded in the next power of two (DESIGN.md reading
R19): GPU through the C ABI against the oracle on the IMAGE-sized problem."""
import numpy as np
import pytest

from gen import workloads as wl
from oracle import frs_oracle as o

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


@pytest.mark.parametrize("shape", [(48, 40, 64, 64), (360, 300, 512, 512), (100, 500, 128, 512), (3600, 3600, 4096, 4096)])
def test_embedded_convolution(frs, shape):
    nyi, nxi, ny, nx = shape
    w = wl.make_config(3, ny=nyi, nx=nxi, npts=200000 if nyi > 1000 else 20000)
    psf = o.psf_from_weights(w.w_half[0]).astype(np.float32)                 # [2 nyi, 2 nxi], the image-sized PSF
    ctx = frs.Context(ny, nx, 1)
    ctx.set_psf_embedded(dev(psf[None]), nyi, nxi)
    rng = np.random.default_rng(1)
    x = rng.normal(size=(nyi, nxi)).astype(np.float32)
    y = ctx.new_image()
    ctx.psf_apply(dev(o.embed(x, ny, nx)[None]), y)
    ref = o.psf_apply(o.psf_spectrum_from_psf(psf.astype(np.float64))[0], x)  # the oracle on the fp32-rounded PSF
    assert rel(y.cpu().numpy()[0, :nyi, :nxi], ref) <= 1e-5


@pytest.mark.parametrize("shape", [(48, 40, 64, 64), (360, 300, 512, 512)])
def test_embedded_energy_gradient_metric_and_cg_step(frs, shape):
    import torch
    nyi, nxi, ny, nx = shape
    w = wl.make_config(3, ny=nyi, nx=nxi, npts=20000)
    wf = wl.make_config(3, ny=ny, nx=nx, npts=2000)                          # only for an amplitude spectrum on the grid
    psf = o.psf_from_weights(w.w_half[0]).astype(np.float32)
    w_img = o.psf_spectrum_from_psf(psf.astype(np.float64))[0]
    mu = float(np.log(np.median(w.sky_true)))
    ctx = frs.Context(ny, nx, 1)
    ctx.set_psf_embedded(dev(psf[None]), nyi, nxi)
    ctx.set_dirty(dev(o.embed(w.dirty[0], ny, nx)[None]))
    ctx.set_amplitude(dev(wf.amp), [mu])
    rng = np.random.default_rng(2)
    xi = (0.3 * rng.normal(size=(ny, nx))).astype(np.float32)
    g = ctx.new_latent()
    e = ctx.energy_grad(dev(xi[None]), g, with_prior=True)
    e_ref, g_ref = o.energy_grad_embedded(w_img, w.dirty[0], wf.amp[0], mu, xi)
    assert abs(e - e_ref) <= 1e-5 * abs(e_ref) and rel(g.cpu().numpy()[0], g_ref) <= 1e-5
    s = ctx.new_image()
    ctx.sky_forward(dev(xi[None]), s)
    sn = s.cpu().numpy()[0]
    assert np.all(sn[nyi:, :] == 0) and np.all(sn[:, nxi:] == 0) and np.all(sn[:nyi, :nxi] > 0)
    v = rng.normal(size=(ny, nx)).astype(np.float32)
    out = ctx.new_latent()
    ctx.metric_apply(dev(v[None]), out, with_prior=True)
    assert rel(out.cpu().numpy()[0], o.metric_apply_embedded(w_img, nyi, nxi, wf.amp[0], mu, xi, v)) <= 1e-5
    # one teacher-forced CG step on the embedded metric
    b = (-g).contiguous()
    x = torch.zeros_like(b)
    ctx.cg_solve(b, x, 1)
    ap = lambda u: o.metric_apply_embedded(w_img, nyi, nxi, wf.amp[0], mu, xi, u)     # noqa: E731
    ref = o.cg(lambda u: ap(u[0])[None], b.cpu().numpy().astype(np.float64), max_iter=1)
    assert rel(x.cpu().numpy(), ref["x"]) <= 1e-5


def test_field_of_view_arguments(frs):
    ctx = frs.Context(64, 64, 1)
    for bad in ((0, 10), (65, 10), (10, 65)):
        with pytest.raises(frs.FrsError):
            ctx.set_field_of_view(*bad)
    ctx.set_field_of_view(64, 64)
