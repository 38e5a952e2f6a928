"""GPU parity of the exact (ungridded) response on uv points and of the major-cycle residual (Alg. 1, Eq. 20-22;
DESIGN.md R16) against oracle.exact_response / exact_adjoint / major_cycle_residual (direct sums in fp64)."""
import numpy as np
import pytest

from gen import workloads as wl
from oracle import frs_oracle as o

pytestmark = pytest.mark.gpu
TOL = 1e-5


def rel(a, b):
    a, b = np.asarray(a, np.complex128), np.asarray(b, np.complex128)
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


def draw_uv(ny, nx, npts, seed):
    rng = np.random.default_rng(seed)
    u, v = wl.uv_gaussian(rng, npts, 2 * ny, 2 * nx, 0.2)
    keep = (np.abs(u) < nx - 0.5) & (np.abs(v) < ny - 0.5)
    return np.stack([u[keep], v[keep]], axis=1).astype(np.float32), rng


@pytest.mark.parametrize("shape", [(128, 128), (64, 256), (32, 32)])
def test_exact_response_adjoint_and_residual(frs, shape):
    import torch
    ny, nx = shape
    uv, rng = draw_uv(ny, nx, 3000, 70)
    nvis = uv.shape[0]
    wgt = rng.uniform(0.5, 2.0, nvis).astype(np.float32)
    x = np.exp(rng.normal(size=(ny, nx))).astype(np.float32)
    ctx = frs.Context(ny, nx, 1)
    vis = torch.empty((nvis, 2), device="cuda")
    ctx.exact_response(dev(uv), dev(x), vis)
    v_ref = o.exact_response(uv, x, 2 * ny, 2 * nx)
    vh = vis.cpu().numpy()
    assert rel(vh[:, 0] + 1j * vh[:, 1], v_ref) <= TOL
    y = torch.empty((ny, nx), device="cuda")
    vin = (rng.normal(size=nvis) + 1j * rng.normal(size=nvis)).astype(np.complex64)
    ctx.exact_adjoint(dev(uv), dev(wgt), dev(np.stack([vin.real, vin.imag], 1)), y)
    assert rel(y.cpu().numpy(), o.exact_adjoint(uv, wgt, vin, ny, nx, 2 * ny, 2 * nx)) <= TOL
    dirty = o.exact_adjoint(uv, wgt, v_ref, ny, nx, 2 * ny, 2 * nx).astype(np.float32) * 1.01      # some I^D
    sky = (x * rng.uniform(0.9, 1.1, size=x.shape)).astype(np.float32)                            # some I_i
    d = torch.empty((ny, nx), device="cuda")
    ctx.major_cycle_residual(dev(uv), dev(wgt), dev(dirty), dev(sky), d)
    d_ref = o.major_cycle_residual(uv, wgt, dirty, sky, 2 * ny, 2 * nx)
    assert np.linalg.norm(d.cpu().numpy() - d_ref) <= TOL * np.linalg.norm(dirty)                 # a difference of two images of that size


def test_major_cycle_closes_on_the_truth_and_matches_the_psf_on_the_grid(frs):
    """Alg. 1 in miniature: I^D = R^+ N^-1 R s* (noise-free); with I_0 = s* the major cycle returns d_1 = 0.  And for uv points
    ON grid cells the exact R^+ N^-1 R is the PSF convolution with the gridded weights (R5) -- the minor cycle's operator."""
    import torch
    ny = nx = 128
    uv, rng = draw_uv(ny, nx, 4000, 71)
    nvis = uv.shape[0]
    wgt = np.full(nvis, 0.7, np.float32)
    s_true = np.exp(rng.normal(size=(ny, nx))).astype(np.float32)
    ctx = frs.Context(ny, nx, 1)
    vis = torch.empty((nvis, 2), device="cuda")
    dirty = torch.empty((ny, nx), device="cuda")
    ctx.exact_response(dev(uv), dev(s_true), vis)
    ctx.exact_adjoint(dev(uv), dev(wgt), vis, dirty)                       # I^D = R^+ N^-1 V
    d1 = torch.empty_like(dirty)
    ctx.major_cycle_residual(dev(uv), dev(wgt), dirty, dev(s_true), d1)
    assert float(d1.double().norm()) <= 2e-6 * float(dirty.double().norm())
    # on-grid: the same operator through the FFT path of the minor cycle
    uvg = np.rint(uv)
    wgrid = np.zeros((2 * ny, 2 * nx))
    for (u, v), wk in zip(uvg, wgt):
        wgrid[int(v) % (2 * ny), int(u) % (2 * nx)] += wk
        wgrid[int(-v) % (2 * ny), int(-u) % (2 * nx)] += wk
    ctx.set_psf_weights(dev(wgrid[None, :, : nx + 1]))
    y_fft = ctx.new_image()
    ctx.psf_apply(dev(s_true[None]), y_fft)
    ctx.exact_response(dev(uvg), dev(s_true), vis)
    y_dir = torch.empty((ny, nx), device="cuda")
    ctx.exact_adjoint(dev(uvg), dev(wgt), vis, y_dir)
    assert rel(y_dir.cpu().numpy(), y_fft.cpu().numpy()[0]) <= TOL


def test_exact_response_argument_errors(frs):
    import torch
    ctx = frs.Context(2048, 64, 1)
    uv = torch.zeros((4, 2), device="cuda")
    with pytest.raises(frs.FrsError) as ei:                                # direct sums stop at 1024
        ctx.exact_response(uv, torch.zeros((2048, 64), device="cuda"), torch.zeros((4, 2), device="cuda"))
    assert ei.value.code == frs.binding.FRS_EINVAL
