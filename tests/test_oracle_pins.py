"""Pins of oracle/frs_oracle.py against what the paper and the mathematics fix (CPU only).

Each test names the passage / reading it pins (P:<n> = PAPER.md line n; R<k> = DESIGN.md reading k).
"""
import os

import numpy as np
import pytest

from gen import workloads as wl
from oracle import frs_oracle as o


def rel(a, b):
    return np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(b)


@pytest.fixture(scope="module")
def small():
    """config-1 recipe at 16x16 (brute-force size)."""
    return wl.make_config(1, n=16, npts=4000)


@pytest.fixture(scope="module")
def rect():
    """config-3 recipe on a 16x32 rectangle (ny != nx catches transposed operands)."""
    return wl.make_config(3, ny=16, nx=32, npts=6000)


@pytest.fixture(scope="module")
def multi():
    """config-5 recipe, 3 channels of 16x16, two latent fields."""
    return wl.make_config(5, n=16, nchan=3, npts=5000)


# ------------------------------------------------------------------ library FFT vs the definition
@pytest.mark.parametrize("n", [1, 2, 3, 8, 16, 64])
def test_fft_is_the_dft_definition(n):
    rng = np.random.default_rng(n)
    x = rng.normal(size=n) + 1j * rng.normal(size=n)
    assert rel(np.fft.fft(x), o.dft_naive(x)) < 1e-12 if n > 1 else True
    assert np.allclose(np.fft.ifft(x) * n, o.dft_naive(x, +1), atol=1e-12)
    assert np.allclose(o.dft_naive(o.dft_naive(x), +1), n * x, atol=1e-10)          # inverse o forward = n id
    assert np.isclose(np.sum(np.abs(o.dft_naive(x)) ** 2), n * np.sum(np.abs(x) ** 2))  # Parseval


def test_fft2_and_rfft2_are_the_2d_definition():
    rng = np.random.default_rng(0)
    x = rng.normal(size=(8, 16))
    f = o.dft2_naive(x)
    assert rel(np.fft.fft2(x), f) < 1e-12
    assert rel(np.fft.rfft2(x), f[:, :9]) < 1e-12
    assert rel(np.fft.irfft2(f[:, :9], s=x.shape) * x.size, np.real(o.dft2_naive(f, +1))) < 1e-12


# ------------------------------------------------------------------ Eq. 14, R2, R3
def test_golden_hand_worked_2x2(golden_dir):
    rows = [l for l in open(os.path.join(golden_dir, "hand_conv_2x2.txt")) if not l.startswith("#")]
    img = np.array([rows[0].split(), rows[1].split()], float)
    exp = np.array([rows[2].split(), rows[3].split()], float)
    w_half = np.zeros((4, 3))
    w_half[0, 1] = 1.0                       # W[0][1] (and, by Hermitian symmetry, W[0][3])
    assert np.allclose(o.psf_from_weights(w_half)[0], [2, 0, -2, 0], atol=1e-14)
    assert np.allclose(o.psf_apply(w_half, img), exp, atol=1e-13)
    assert np.isclose(np.sum(img * o.psf_apply(w_half, img)), float(rows[4]))
    assert np.isclose(o.quadratic_form_spectral(w_half, img), float(rows[4]))


def test_convolution_theorem_vs_direct_sum_16(small, rect):
    """padded FFT convolution == O(N^4) linear convolution with the 2N PSF."""
    for w in (small, rect):
        rng = np.random.default_rng(1)
        x = rng.normal(size=(w.ny, w.nx))
        wh = w.w_half[0].astype(np.float64)
        psf = o.psf_from_weights(wh)
        ref = o.conv_direct(psf, x)
        assert rel(o.psf_apply(wh, x), ref) < 1e-12
        assert rel(o.psf_apply_full(wh, x), ref) < 1e-12


def test_psf_peak_is_sum_of_weights(small, rect):
    for w in (small, rect):
        wh = w.w_half[0].astype(np.float64)
        psf = o.psf_from_weights(wh)
        tot = np.sum(o.full_spectrum(wh))
        assert np.isclose(psf[0, 0], tot, rtol=1e-13)
        assert np.all(np.abs(psf) <= psf[0, 0] * (1 + 1e-12))
        assert np.isclose(psf[0, 0], np.max(psf))


def test_special_kernels_closed_forms():
    ny, nx = 8, 16
    my, mx = 2 * ny, 2 * nx
    rng = np.random.default_rng(2)
    x = rng.normal(size=(ny, nx))
    # W == c  =>  C = c My Mx identity
    assert rel(o.psf_apply(np.full((my, nx + 1), 0.25), x), 0.25 * my * mx * x) < 1e-13
    # one +-k0 pair  =>  psf = 2 w cos(2 pi k0.x/M)
    wh = np.zeros((my, nx + 1))
    wh[3, 5] = 0.7
    wh[my - 3, 5] = 0.0                       # (-k0 lives at [my-3][mx-5], outside the half grid)
    yy, xx = np.mgrid[0:my, 0:mx]
    assert np.allclose(o.psf_from_weights(wh), 2 * 0.7 * np.cos(2 * np.pi * (3 * yy / my + 5 * xx / mx)), atol=1e-12)
    # s = delta_{x0}  =>  C s = psf[x - x0] cropped; corners exercise the wrapped half
    w = wl.make_config(2, ny=ny, nx=nx, npts=3000)
    wh = w.w_half[0].astype(np.float64)
    psf = o.psf_from_weights(wh)
    for (y0, x0) in [(0, 0), (0, nx - 1), (ny - 1, 0), (ny - 1, nx - 1), (3, 7)]:
        d = np.zeros((ny, nx))
        d[y0, x0] = 1.0
        exp = np.array([[psf[(y - y0) % my, (xq - x0) % mx] for xq in range(nx)] for y in range(ny)])
        got = o.psf_apply(wh, d)
        assert np.allclose(got, exp, atol=1e-9 * psf[0, 0])
        assert np.unravel_index(np.argmax(got), got.shape) == (y0, x0)      # index/padding layout, exact


def test_quadratic_form_independent_route(small, rect):
    for w in (small, rect):
        x = np.random.default_rng(3).normal(size=(w.ny, w.nx))
        wh = w.w_half[0].astype(np.float64)
        q = float(np.sum(x * o.psf_apply(wh, x)))
        assert q >= 0
        assert np.isclose(q, o.quadratic_form_spectral(wh, x), rtol=1e-12)


def test_pruned_even_odd_identity():
    """Zero-padded N->2N transform: even bins = FFT_N(x), odd bins = FFT_N(x w_2N^n); the cropped
    inverse is y[n] = (IFFT_N(Y_even) + w_2N^-n IFFT_N(Y_odd))/2 -- lets the GPU prune while the
    oracle stays plain."""
    n = 32
    rng = np.random.default_rng(4)
    x = rng.normal(size=n) + 1j * rng.normal(size=n)
    full = np.fft.fft(np.concatenate([x, np.zeros(n)]))
    tw = np.exp(-2j * np.pi * np.arange(n) / (2 * n))
    assert rel(full[0::2], np.fft.fft(x)) < 1e-14
    assert rel(full[1::2], np.fft.fft(x * tw)) < 1e-14
    y = rng.normal(size=2 * n) + 1j * rng.normal(size=2 * n)
    exp = np.fft.ifft(y)[:n]
    got = 0.5 * (np.fft.ifft(y[0::2]) + np.conj(tw) * np.fft.ifft(y[1::2]))
    assert rel(got, exp) < 1e-14


# ------------------------------------------------------------------ symmetry / adjointness to 1e-12
def test_adjointness(small, rect, multi):
    rng = np.random.default_rng(5)
    for w in (small, rect):
        wh = w.w_half[0].astype(np.float64)
        x, y = rng.normal(size=(2, w.ny, w.nx))
        a, b = np.sum(o.psf_apply(wh, x) * y), np.sum(x * o.psf_apply(wh, y))
        assert abs(a - b) <= 1e-12 * max(abs(a), abs(b))
        a, b = np.sum(o.hartley2(x) * y), np.sum(x * o.hartley2(y))
        assert abs(a - b) <= 1e-12 * np.linalg.norm(o.hartley2(x)) * np.linalg.norm(y)
        big = rng.normal(size=(2 * w.ny, 2 * w.nx))
        assert np.isclose(np.sum(o.pad(x) * big), np.sum(x * o.crop(big)), rtol=1e-13)
    for w in (small, multi):
        xi = rng.normal(size=(w.nfield, w.ny, w.nx))
        v = rng.normal(size=(w.nfield, w.ny, w.nx))
        u = rng.normal(size=(w.nchan, w.ny, w.nx))
        s = o.sky(xi, w.amp, w.mu, w.lognu)
        a = np.sum(o.jvp(w.amp, w.mu, w.lognu, xi, v) * u)
        b = np.sum(v * o.vjp(w.amp.astype(np.float64), w.lognu, s, u))
        assert abs(a - b) <= 1e-12 * max(abs(a), abs(b), 1.0) * 10


def test_generated_weights_are_hermitian_and_integer(small, rect, multi):
    for w in (small, rect, multi):
        for c in range(w.nchan):
            full = o.full_spectrum(w.w_counts[c])
            my, mx = full.shape
            ky, kx = (-np.arange(my)) % my, (-np.arange(mx)) % mx
            assert np.array_equal(full, full[np.ix_(ky, kx)])           # W[-k] = W[k], bit-exact
            assert np.array_equal(full, np.rint(full)) and full.min() >= 0
            assert np.array_equal(full[:, : w.nx + 1], w.w_counts[c])   # half-grid round trip
            # the self-conjugate columns kx = 0 and kx = nx are even in ky
            for col in (0, w.nx):
                assert np.array_equal(w.w_counts[c][:, col], w.w_counts[c][ky, col])


def test_set_psf_semantics(small):
    wh = small.w_half[0].astype(np.float64)
    psf = o.psf_from_weights(wh)
    back, ok = o.psf_spectrum_from_psf(psf)
    assert ok and rel(back, wh) < 1e-12
    bad = psf.copy()
    bad[1, 2] += 0.3 * psf[0, 0]              # breaks evenness -> imaginary spectrum
    assert not o.psf_spectrum_from_psf(bad)[1]


# ------------------------------------------------------------------ correlated field (R6)
def test_hartley_closed_forms():
    ny, nx = 8, 16
    rng = np.random.default_rng(6)
    z = rng.normal(size=(ny, nx))
    assert rel(o.hartley2(o.hartley2(z)), ny * nx * z) < 1e-13
    yy, xx = np.mgrid[0:ny, 0:nx]
    for (ky, kx) in [(0, 0), (1, 0), (3, 5), (7, 15), (4, 8)]:
        d = np.zeros((ny, nx))
        d[ky, kx] = 1.0
        th = 2 * np.pi * (ky * yy / ny + kx * xx / nx)
        assert np.allclose(o.hartley2(d), np.cos(th) + np.sin(th), atol=1e-12)
    # definition written out as the O(N^4) sum
    kyy, kxx = np.mgrid[0:ny, 0:nx]
    brute = np.array([[np.sum(z * (np.cos(2 * np.pi * (kyy * y / ny + kxx * x / nx))
                                   + np.sin(2 * np.pi * (kyy * y / ny + kxx * x / nx))))
                       for x in range(nx)] for y in range(ny)])
    assert rel(o.hartley2(z), brute) < 1e-12


def test_golden_hand_worked_two_field_sky(golden_dir):
    """Pins sky / log_sky / channel_coeff (R6, c-6): which field carries ln nu_c, where mu enters, and the
    orientation of the Hartley modes -- against exponents derived by hand in tests/golden/."""
    rows = [l.split() for l in open(os.path.join(golden_dir, "hand_sky_two_fields.txt")) if not l.startswith("#")]
    log_s = np.array(rows, float).reshape(3, 2, 4)
    ny, nx = 2, 4
    xi = np.zeros((2, ny, nx)); amp = np.zeros((2, ny, nx))
    xi[0, 0, 1], amp[0, 0, 1] = 1.0, 0.5
    xi[1, 1, 0], amp[1, 1, 0] = 2.0, 0.25
    mu, lognu = [0.3, -0.7], [-0.5, 0.0, 0.25]
    assert np.allclose(o.sky(xi, amp, mu, lognu), np.exp(log_s), rtol=1e-13)
    assert np.allclose(o.log_sky(xi, amp, mu)[0], log_s[1], atol=1e-13)              # lognu = 0: tau_0 alone
    assert np.allclose(o.log_sky(xi, amp, mu)[1], np.array([[-0.2] * 4, [-1.2] * 4]), atol=1e-13)
    # a single field ignores lognu altogether: s = exp(tau)
    assert np.allclose(o.sky(xi[:1], amp[:1], mu[:1], [0.4]), np.exp(log_s[1])[None], rtol=1e-13)
    co = o.channel_coeff(2, lognu)
    assert np.array_equal(co, np.array([[1, -0.5], [1, 0.0], [1, 0.25]]))
    assert np.array_equal(o.channel_coeff(1, lognu), np.ones((3, 1)))


def test_sky_closed_form_single_modes_and_offset():
    """xi = delta_k  =>  s[x] = exp(mu + A[k] cas(2 pi k.x/N)) on a rectangle, incl. k = 0 and Nyquist modes;
    mu enters exactly once: field 0 scales every channel by e^c, field 1 channel c by e^(c lognu_c)."""
    ny, nx = 4, 8
    yy, xx = np.mgrid[0:ny, 0:nx]
    rng = np.random.default_rng(61)
    a = rng.uniform(0.2, 1.0, size=(1, ny, nx))
    for (ky, kx) in [(0, 0), (2, 0), (0, 4), (2, 4), (1, 3), (3, 7)]:
        xi = np.zeros((1, ny, nx))
        xi[0, ky, kx] = -1.5
        th = 2 * np.pi * (ky * yy / ny + kx * xx / nx)
        want = np.exp(0.37 - 1.5 * a[0, ky, kx] * (np.cos(th) + np.sin(th)))
        assert np.allclose(o.sky(xi, a, [0.37], [0.0])[0], want, rtol=1e-12)
    xi2, a2 = rng.normal(size=(2, ny, nx)), rng.uniform(0.1, 0.5, size=(2, ny, nx))
    lognu = np.array([-0.3, 0.2, 0.6])
    s0 = o.sky(xi2, a2, [0.1, -0.7], lognu)
    c = 0.25
    assert np.allclose(o.sky(xi2, a2, [0.1 + c, -0.7], lognu), np.exp(c) * s0, rtol=1e-12)
    assert np.allclose(o.sky(xi2, a2, [0.1, -0.7 + c], lognu), np.exp(c * lognu)[:, None, None] * s0, rtol=1e-12)
    # two channels with the same lognu see the same sky; distinct lognu do not
    s_same = o.sky(xi2, a2, [0.1, -0.7], [0.2, 0.2])
    assert np.array_equal(s_same[0], s_same[1]) and not np.allclose(s0[0], s0[1])


def test_cg_fp32_envelope_on_a_scaled_identity():
    """M = c 1: CG converges in one step to b/c, and the seeded relative perturbation of the operator output
    (|u| <= 2^-24) moves x_1 by a weighted mean of u -- so the envelope is > 0 and <= 2^-24 there."""
    b = np.random.default_rng(5).normal(size=(4, 8))
    env = o.cg_fp32_envelope(lambda v: 3.0 * v, b, max_iter=1)
    assert env.shape == (1,) and 0.0 < env[0] <= 2.0 ** -24


def test_field_variance_is_sum_of_A_squared():
    """Var(lin[x]) = sum_k A[k]^2 at every pixel, exact for even A (R6)."""
    ny, nx = 8, 16
    a = wl.amplitude_spectrum(ny, nx, "lorentz4", 1.0)
    kyi, kxi = (-np.arange(ny)) % ny, (-np.arange(nx)) % nx
    assert np.array_equal(a, a[np.ix_(kyi, kxi)])                       # A[-k] = A[k]
    assert np.isclose(np.sum(a ** 2) - a[0, 0] ** 2, 1.0)
    # exact: Var = sum_k A_k^2 cas^2 = sum A^2 (1 + sin 2 theta), and the sine term cancels k <-> -k
    yy, xx = 3, 11
    kyy, kxx = np.mgrid[0:ny, 0:nx]
    th = 2 * np.pi * (kyy * yy / ny + kxx * xx / nx)
    assert np.isclose(np.sum(a ** 2 * (np.cos(th) + np.sin(th)) ** 2), np.sum(a ** 2), rtol=1e-12)
    rng = np.random.default_rng(7)
    draws = np.stack([o.hartley2(a * rng.normal(size=(ny, nx))) for _ in range(4000)])
    assert abs(draws.var() / np.sum(a ** 2) - 1.0) < 0.02


# ------------------------------------------------------------------ gradient / JVP vs central differences (1e-6)
@pytest.mark.parametrize("which", ["small", "multi"])
def test_gradient_and_jvp_vs_finite_differences(which, small, multi):
    w = small if which == "small" else multi
    rng = np.random.default_rng(8)
    xi = 0.3 * rng.normal(size=(w.nfield, w.ny, w.nx))
    args = (w.w_half, w.dirty, w.amp, w.mu, w.lognu)
    e, g = o.energy_grad(*args, xi, True)
    assert np.isclose(e, o.energy(*args, xi, True), rtol=1e-13)
    h = 1e-5 * np.linalg.norm(xi)
    for _ in range(10):
        d = rng.normal(size=xi.shape)
        d /= np.linalg.norm(d)
        fd = (o.energy(*args, xi + h * d, True) - o.energy(*args, xi - h * d, True)) / (2 * h)
        an = np.sum(g * d)
        assert abs(fd - an) <= 1e-6 * max(abs(an), np.linalg.norm(g) * 1e-2)
    v = rng.normal(size=xi.shape)
    hh = 1e-6
    fd = (o.sky(xi + hh * v, w.amp, w.mu, w.lognu) - o.sky(xi - hh * v, w.amp, w.mu, w.lognu)) / (2 * hh)
    assert rel(fd, o.jvp(w.amp, w.mu, w.lognu, xi, v)) < 1e-6


# ------------------------------------------------------------------ metric (Eq. 10)
@pytest.mark.parametrize("which", ["small", "multi"])
def test_metric_invariants(which, small, multi):
    w = small if which == "small" else multi
    rng = np.random.default_rng(9)
    xi = 0.3 * rng.normal(size=(w.nfield, w.ny, w.nx))
    u, v = rng.normal(size=(2, w.nfield, w.ny, w.nx))
    mv = o.metric_apply(w.w_half, w.amp, w.mu, w.lognu, xi, v, True)
    mu_ = o.metric_apply(w.w_half, w.amp, w.mu, w.lognu, xi, u, True)
    a, b = np.sum(u * mv), np.sum(mu_ * v)
    assert abs(a - b) <= 1e-12 * max(abs(a), abs(b)) * 10              # symmetric
    assert np.sum(v * mv) >= np.sum(v * v)                              # M >= identity
    # composition J^T (C (J v)) + v written out step by step
    s = o.sky(xi, w.amp, w.mu, w.lognu)
    jv = o.jvp(w.amp, w.mu, w.lognu, xi, v)
    cj = np.stack([o.psf_apply(w.w_half[c], jv[c]) for c in range(w.nchan)])
    assert rel(mv, o.vjp(w.amp.astype(np.float64), w.lognu, s, cj) + v) < 1e-13
    # the sky-space ('L1') apply is the same thing without the Hartley maps
    x = rng.normal(size=(w.nchan, w.ny, w.nx))
    l1 = o.sky_metric_apply(w.w_half, s, x)
    assert rel(l1[0], s[0] * o.psf_apply(w.w_half[0], s[0] * x[0])) < 1e-14


def test_fisher_identity_monte_carlo():
    """E_n[(J^T n)(J^T n)^T v] -> M_lh v for n ~ N(0, C): data noise (generator), energy and metric
    are mutually consistent (Eq. 10)."""
    n = 8
    w = wl.make_config(1, n=n, npts=3000, sigma_rel=0.1)
    wh = w.w_half[0].astype(np.float64)
    rng = np.random.default_rng(10)
    xi = 0.2 * rng.normal(size=(1, n, n))
    v = rng.normal(size=(1, n, n))
    s = o.sky(xi, w.amp, w.mu, w.lognu)
    m_lh = o.metric_apply(w.w_half, w.amp, w.mu, w.lognu, xi, v, False)
    wfull = o.full_spectrum(wh)
    acc = np.zeros_like(v)
    ndraw = 6000
    for _ in range(ndraw):
        eta = rng.normal(size=(2 * n, 2 * n))
        noise = o.crop(np.real(np.fft.ifft2(np.sqrt(wfull) * np.fft.fft2(eta))) * (2 * n))   # Cov = C
        jn = o.vjp(w.amp.astype(np.float64), w.lognu, s, noise[None])
        acc += jn * np.sum(jn * v)
    assert rel(acc / ndraw, m_lh) < 0.12                                   # ~ a few / sqrt(ndraw)


def test_noise_scale_of_generator():
    """std(n')/max(C s*) = sigma_rel and Var(n'[x]) = sum W (R7): check sum W against w0."""
    w = wl.make_config(1, n=32, npts=8000, sigma_rel=1e-3)
    wh = w.w_half[0].astype(np.float64)
    sig = o.psf_apply(wh, w.sky_true[0])
    var = np.sum(o.full_spectrum(wh))
    assert np.isclose(np.sqrt(var) / sig.max(), 1e-3, rtol=2e-3)
    resid = w.dirty[0] - sig
    assert 0.5 < resid.std() / np.sqrt(var) < 1.5


# ------------------------------------------------------------------ CG (R9)
def test_cg_reaches_dense_solve_and_phi_decreases():
    n = 8
    w = wl.make_config(1, n=n, npts=3000, sigma_rel=0.05)
    rng = np.random.default_rng(11)
    xi = 0.2 * rng.normal(size=(1, n, n))
    s = o.sky(xi, w.amp, w.mu, w.lognu)
    ap = lambda v: o.metric_apply(w.w_half, w.amp, w.mu, w.lognu, xi, v, True, s=s)
    dense = np.stack([ap(e.reshape(1, n, n)).ravel() for e in np.eye(n * n)], axis=1)
    assert np.allclose(dense, dense.T, rtol=1e-11, atol=1e-11 * np.abs(dense).max())
    assert np.linalg.eigvalsh(0.5 * (dense + dense.T)).min() >= 1 - 1e-9
    b = rng.normal(size=(1, n, n))
    exact = np.linalg.solve(dense, b.ravel()).reshape(1, n, n)
    sol = o.cg(ap, b, max_iter=4 * n * n, rtol=1e-13, keep=True)
    assert rel(sol["x"], exact) < 1e-10
    phi = [0.5 * np.sum(x * ap(x)) - np.sum(b * x) for x in sol["xs"]]
    assert all(p1 < p0 + 1e-9 * abs(p0) for p0, p1 in zip([0.0] + phi[:-1], phi))    # phi strictly decreases
    assert sol["res"][-1] < sol["res"][0]
    # teacher-forced step == the loop's own step
    st = o.cg_step(ap, np.zeros_like(b), b.copy(), b.copy(), float(np.sum(b * b)))
    assert rel(st["x"], sol["xs"][0]) < 1e-14


def test_cg_on_config1_recipe_residual_decreases_and_envelope_grows():
    w = wl.make_config(1, n=32, npts=6000)
    xi = np.zeros((1, 32, 32))
    e, g = o.energy_grad(w.w_half, w.dirty, w.amp, w.mu, w.lognu, xi, True)
    s = o.sky(xi, w.amp, w.mu, w.lognu)
    ap = lambda v: o.metric_apply(w.w_half, w.amp, w.mu, w.lognu, xi, v, True, s=s)
    sol = o.cg(ap, -g, max_iter=20)
    assert sol["iters"] == 20 and sol["res"][-1] < sol["res"][0]
    env = o.cg_fp32_envelope(ap, -g, max_iter=20)
    assert env[0] < 1e-6 and env[-1] >= env[0]


def test_newton_cg_step_decreases_energy():
    w = wl.make_config(2, n=16, npts=3000, sigma_rel=0.05)
    xi = np.zeros((1, 16, 16))
    xi1, e0, e1 = o.newton_cg_step(w.w_half, w.dirty, w.amp, w.mu, w.lognu, xi, cg_iters=30)
    assert e1 < e0


# ------------------------------------------------------------------ Eq. 9 with the fitted noise kernel (Eq. 15-18, R14)
def test_noise_kernel_is_the_minimiser_of_eq17(small):
    """Eq. 17 by brute force on a tiny grid: a generic minimiser over xi (K = exp xi + eps) lands on the closed form
    wherever the unconstrained optimum is above the floor, and no perturbation of K lowers the residual."""
    from scipy.optimize import minimize
    w = wl.make_config(1, n=4, npts=300)
    ny = nx = 4
    eps = 1e-2 * float(np.sum(o.full_spectrum(w.w_half[0])))
    kern = o.noise_kernel_from_psf(w.w_half[0], eps)
    assert kern.shape == (ny, nx) and np.all(kern >= eps)
    delta = np.zeros((ny, nx)); delta[ny // 2, nx // 2] = 1.0
    target = o.psf_apply(w.w_half[0], delta) + eps * delta           # N'(I_delta)

    def resid(k):
        return float(np.sum(np.abs(target - np.fft.ifft2(k.reshape(ny, nx) * np.fft.fft2(delta))) ** 2))

    r0 = resid(kern)
    rng = np.random.default_rng(1)
    for _ in range(50):                                              # K is a minimum among admissible kernels
        trial = np.maximum(kern * (1 + 1e-3 * rng.normal(size=kern.shape)), eps)
        assert resid(trial) >= r0 * (1 - 1e-12)
    sol = minimize(lambda xi: resid(np.exp(xi) + eps), np.log(np.maximum(kern.ravel() - eps, 1e-3 * eps) + 1e-30),
                   method="L-BFGS-B", options={"maxiter": 500, "ftol": 1e-15, "gtol": 1e-12})
    free = kern.ravel() > 1.001 * eps
    assert np.allclose((np.exp(sol.x) + eps)[free], kern.ravel()[free], rtol=1e-4)
    assert sol.fun >= r0 * (1 - 1e-9)


def test_noise_kernel_closed_forms():
    ny, nx = 8, 16
    # W == c: the PSF is a delta of weight c (2ny)(2nx), so N' = (c M + eps) 1 and K is flat
    c, eps = 0.37, 0.05
    wc = np.full((2 * ny, nx + 1), c)
    assert np.allclose(o.noise_kernel_from_psf(wc, eps), c * 4 * ny * nx + eps, rtol=1e-12)
    # K is real, even (K[-k] = K[k]) and >= eps for a generated PSF; its mean is the PSF peak + eps (sum_k K = N^2 n_delta[0])
    w = wl.make_config(3, ny=ny, nx=nx, npts=3000)
    eps = 1e-3 * float(np.sum(o.full_spectrum(w.w_half[0])))
    k = o.noise_kernel_from_psf(w.w_half[0], eps)
    kyi, kxi = (-np.arange(ny)) % ny, (-np.arange(nx)) % nx
    assert np.allclose(k, k[np.ix_(kyi, kxi)], rtol=1e-12) and np.all(k >= eps)
    unfloored = np.real(np.fft.fft2(np.roll(o.psf_from_weights(w.w_half[0]), (ny // 2, nx // 2), (0, 1))[:ny, :nx]
                                    ) * np.conj(np.fft.fft2(np.eye(1, ny * nx, (ny // 2) * nx + nx // 2).reshape(ny, nx)))) + eps
    assert np.allclose(k, np.maximum(unfloored, eps), rtol=1e-10, atol=1e-10 * k.max())      # the PSF stamp route


def test_ninv_apply_closed_forms_and_symmetry():
    ny, nx = 8, 16
    rng = np.random.default_rng(21)
    k = np.exp(rng.normal(size=(ny, nx)))
    kyi, kxi = (-np.arange(ny)) % ny, (-np.arange(nx)) % nx
    k = 0.5 * (k + k[np.ix_(kyi, kxi)])                              # a real even positive kernel
    x, y = rng.normal(size=(ny, nx)), rng.normal(size=(ny, nx))
    d = np.zeros((ny, nx)); d[0, 0] = 1.0
    assert np.allclose(o.ninv_apply(k, d), np.real(np.fft.ifft2(1.0 / k)), atol=1e-14)      # N'^-1 delta = IFFT(1/K)
    assert np.allclose(o.ninv_apply(np.full((ny, nx), 2.5), x), x / 2.5, atol=1e-14)        # K == c: N'^-1 = 1/c
    assert abs(np.sum(o.ninv_apply(k, x) * y) - np.sum(x * o.ninv_apply(k, y))) <= 1e-12 * np.linalg.norm(x) * np.linalg.norm(y) / k.min()
    assert np.sum(x * o.ninv_apply(k, x)) > 0
    # inverse of the forward convolution of Eq. 15, and periodic: a shift commutes with it
    assert np.allclose(o.ninv_apply(k, np.real(np.fft.ifft2(k * np.fft.fft2(x)))), x, atol=1e-12)
    assert np.allclose(o.ninv_apply(k, np.roll(x, (3, 5), (0, 1))), np.roll(o.ninv_apply(k, x), (3, 5), (0, 1)), atol=1e-13)
    # the Hartley form the kernels use: N'^-1 x = H[ K^-1 . H[x] ] / (ny nx) for an even kernel
    assert np.allclose(o.hartley2(o.hartley2(x) / k) / (ny * nx), o.ninv_apply(k, x), atol=1e-13)


@pytest.mark.parametrize("which", ["small", "multi"])
def test_eq9_gradient_metric_and_limits(which, small, multi):
    w = small if which == "small" else multi
    rng = np.random.default_rng(22)
    eps = 1e-2 * float(np.sum(o.full_spectrum(w.w_half[0])))
    kern = np.stack([o.noise_kernel_from_psf(w.w_half[c], eps) for c in range(w.nchan)])
    xi = 0.3 * rng.normal(size=(w.nfield, w.ny, w.nx))
    e0, g = o.energy_grad_eq9(w.w_half, kern, w.dirty, w.amp, w.mu, w.lognu, xi, True)
    # written out: E = 1/2 sum_c r_c^T N'^-1 r_c + 1/2 xi^2, r = j - C s
    s = o.sky(xi, w.amp, w.mu, w.lognu)
    e_def = 0.5 * np.sum(xi ** 2)
    for c in range(w.nchan):
        r = w.dirty[c] - o.psf_apply(w.w_half[c], s[c])
        e_def += 0.5 * np.sum(r * np.real(np.fft.ifft2(np.fft.fft2(r) / kern[c])))
    assert abs(e0 - e_def) <= 1e-12 * abs(e_def)
    for _ in range(5):                                               # central differences, 1e-6
        d = rng.normal(size=xi.shape)
        h = 1e-5 * np.linalg.norm(xi) / np.linalg.norm(d)
        ep = o.energy_grad_eq9(w.w_half, kern, w.dirty, w.amp, w.mu, w.lognu, xi + h * d, True)[0]
        em = o.energy_grad_eq9(w.w_half, kern, w.dirty, w.amp, w.mu, w.lognu, xi - h * d, True)[0]
        fd = (ep - em) / (2 * h)
        assert abs(fd - np.sum(g * d)) <= 1e-6 * max(abs(fd), np.linalg.norm(g) * np.linalg.norm(d) * 1e-3)
    # metric: composition, symmetry, M >= 1
    u, v = rng.normal(size=xi.shape), rng.normal(size=xi.shape)
    mv = o.metric_apply_eq9(w.w_half, kern, w.amp, w.mu, w.lognu, xi, v, True)
    jv = o.jvp(w.amp, w.mu, w.lognu, xi, v)
    comp = o.vjp(w.amp, w.lognu, s, np.stack([o.psf_apply(w.w_half[c], o.ninv_apply(kern[c], o.psf_apply(w.w_half[c], jv[c])))
                                              for c in range(w.nchan)])) + v
    assert rel(mv, comp) < 1e-13
    mu_ = o.metric_apply_eq9(w.w_half, kern, w.amp, w.mu, w.lognu, xi, u, True)
    assert abs(np.sum(u * mv) - np.sum(mu_ * v)) <= 1e-10 * abs(np.sum(u * mv))
    assert np.sum(v * mv) >= np.sum(v * v)
    # eps -> infinity: N'^-1 -> 1/eps, so eps E_lh -> 1/2 |j - C s|^2 and eps M_lh -> J^T C C J
    big = 1e12 * float(np.max(kern))
    kbig = np.stack([o.noise_kernel_from_psf(w.w_half[c], big) for c in range(w.nchan)])
    e_big = o.energy_grad_eq9(w.w_half, kbig, w.dirty, w.amp, w.mu, w.lognu, xi, False)[0]
    r2 = sum(np.sum((w.dirty[c] - o.psf_apply(w.w_half[c], s[c])) ** 2) for c in range(w.nchan))
    assert abs(big * e_big - 0.5 * r2) <= 1e-9 * r2


# ------------------------------------------------------------------ MGVI samples and the sample-averaged KL (R15)
def test_mgvi_sample_source_has_the_metric_as_covariance():
    """Cov(eta_xi + J^T C N'^-1/2 eta_d) = 1 + J^T C N'^-1 C J = M: checked against the dense metric of a 4x4 problem,
    entry by entry, both by the exact linear map (m is linear in eta) and by Monte Carlo."""
    w = wl.make_config(1, n=4, npts=300)
    n = w.ny * w.nx
    eps = 1e-2 * float(np.sum(o.full_spectrum(w.w_half[0])))
    kern = np.stack([o.noise_kernel_from_psf(w.w_half[0], eps)])
    rng = np.random.default_rng(40)
    xi = 0.3 * rng.normal(size=(1, w.ny, w.nx))
    s = o.sky(xi, w.amp, w.mu, w.lognu)
    dense = np.stack([o.metric_apply_eq9(w.w_half, kern, w.amp, w.mu, w.lognu, xi, e.reshape(1, w.ny, w.nx), True).ravel()
                      for e in np.eye(n)], axis=1)
    # m = eta_xi + A eta_d with A = J^T C N'^-1/2: assemble A column by column, Cov m = 1 + A A^T exactly
    z = np.zeros((1, w.ny, w.nx))
    a_mat = np.stack([o.sample_source_eq9(w.w_half, kern, w.amp, w.lognu, s, z, e.reshape(1, w.ny, w.nx)).ravel() for e in np.eye(n)], axis=1)
    assert np.allclose(np.eye(n) + a_mat @ a_mat.T, dense, rtol=1e-10, atol=1e-10 * np.abs(dense).max())
    assert np.allclose(o.sample_source_eq9(w.w_half, kern, w.amp, w.lognu, s, xi, 0 * z), xi)       # eta_xi enters with weight 1
    draws = np.stack([o.sample_source_eq9(w.w_half, kern, w.amp, w.lognu, s, rng.normal(size=z.shape), rng.normal(size=z.shape)).ravel()
                      for _ in range(4000)])
    emp = draws.T @ draws / len(draws)
    assert np.linalg.norm(emp - dense) / np.linalg.norm(dense) < 0.08
    # N'^-1/2 is the symmetric square root of N'^-1
    x = rng.normal(size=(w.ny, w.nx))
    assert np.allclose(o.ninv_sqrt_apply(kern[0], o.ninv_sqrt_apply(kern[0], x)), o.ninv_apply(kern[0], x), atol=1e-12)
    # a sample solves M sigma = m: against the dense solve
    eta_xi, eta_d = rng.normal(size=z.shape), rng.normal(size=z.shape)
    sg, m = o.draw_sample_eq9(w.w_half, kern, w.amp, w.mu, w.lognu, xi, eta_xi, eta_d, cg_iters=3 * n)
    assert np.allclose(sg.ravel(), np.linalg.solve(dense, m.ravel()), rtol=1e-8, atol=1e-10)


def test_kl_average_gradient_and_metric(multi):
    w = multi
    rng = np.random.default_rng(41)
    eps = 1e-2 * float(np.sum(o.full_spectrum(w.w_half[0])))
    kern = np.stack([o.noise_kernel_from_psf(w.w_half[c], eps) for c in range(w.nchan)])
    xi = 0.2 * rng.normal(size=(w.nfield, w.ny, w.nx))
    samples = [0.1 * rng.normal(size=xi.shape) for _ in range(2)]
    kl, g = o.kl_energy_grad_eq9(w.w_half, kern, w.dirty, w.amp, w.mu, w.lognu, xi, samples, True)
    # written out: the mean over the four positions xi +- sigma_i
    es = [o.energy_grad_eq9(w.w_half, kern, w.dirty, w.amp, w.mu, w.lognu, xi + sg * sgn, True)[0] for sg in samples for sgn in (1, -1)]
    assert abs(kl - np.mean(es)) <= 1e-12 * abs(kl)
    # mirrored: invariant under sigma -> -sigma; one sample at sigma = 0 is the plain energy
    kl2, g2 = o.kl_energy_grad_eq9(w.w_half, kern, w.dirty, w.amp, w.mu, w.lognu, xi, [-sg for sg in samples], True)
    assert abs(kl - kl2) <= 1e-12 * abs(kl) and rel(g2, g) < 1e-12
    e0, g0 = o.energy_grad_eq9(w.w_half, kern, w.dirty, w.amp, w.mu, w.lognu, xi, True)
    kl0, gk0 = o.kl_energy_grad_eq9(w.w_half, kern, w.dirty, w.amp, w.mu, w.lognu, xi, [0 * xi], False)
    assert kl0 == e0 and np.array_equal(gk0, g0)
    for _ in range(3):                                               # gradient of the KL by central differences
        d = rng.normal(size=xi.shape)
        h = 1e-5 * np.linalg.norm(xi) / np.linalg.norm(d)
        kp = o.kl_energy_grad_eq9(w.w_half, kern, w.dirty, w.amp, w.mu, w.lognu, xi + h * d, samples, True)[0]
        km = o.kl_energy_grad_eq9(w.w_half, kern, w.dirty, w.amp, w.mu, w.lognu, xi - h * d, samples, True)[0]
        fd = (kp - km) / (2 * h)
        assert abs(fd - np.sum(g * d)) <= 1e-6 * max(abs(fd), np.linalg.norm(g) * np.linalg.norm(d) * 1e-3)
    v, u = rng.normal(size=xi.shape), rng.normal(size=xi.shape)
    mv = o.kl_metric_apply_eq9(w.w_half, kern, w.amp, w.mu, w.lognu, xi, samples, v, True)
    mu_ = o.kl_metric_apply_eq9(w.w_half, kern, w.amp, w.mu, w.lognu, xi, samples, u, True)
    assert abs(np.sum(u * mv) - np.sum(mu_ * v)) <= 1e-10 * abs(np.sum(u * mv)) and np.sum(v * mv) >= np.sum(v * v)
    one = np.mean([o.metric_apply_eq9(w.w_half, kern, w.amp, w.mu, w.lognu, xi + sg * sgn, v, True) for sg in samples for sgn in (1, -1)], axis=0)
    assert rel(mv, one) < 1e-13


# ------------------------------------------------------------------ exact response and the major cycle (Eq. 1, Eq. 20-22; R16)
def test_exact_response_closed_forms_and_grid_limit():
    ny, nx = 8, 16
    my, mx = 2 * ny, 2 * nx
    rng = np.random.default_rng(60)
    # one visibility, one pixel: the plane wave of Eq. 1
    uv = np.array([[2.3, -1.7]])
    d = np.zeros((ny, nx)); d[3, 5] = 2.0
    assert np.allclose(o.exact_response(uv, d, my, mx), 2.0 * np.exp(-2j * np.pi * (2.3 * 5 / mx - 1.7 * 3 / my)), atol=1e-14)
    # R^dagger N^-1 R delta = 2 w cos(2 pi (u dx / Mx + v dy / My)): the PSF of one visibility and its conjugate
    img = o.exact_adjoint(uv, [0.5], o.exact_response(uv, d, my, mx), ny, nx, my, mx)
    yy, xx = np.mgrid[0:ny, 0:nx]
    assert np.allclose(img, 2.0 * 2 * 0.5 * np.cos(2 * np.pi * (2.3 * (xx - 5) / mx - 1.7 * (yy - 3) / my)), atol=1e-13)
    # adjointness <R x, N^-1 V> summed with the conjugates = <x, R^dagger N^-1 V>
    uvs = np.stack(wl.uv_gaussian(rng, 40, my, mx, 0.2), axis=1)
    w = rng.uniform(0.5, 1.5, 40)
    x = rng.normal(size=(ny, nx))
    v = rng.normal(size=40) + 1j * rng.normal(size=40)
    lhs = 2.0 * np.real(np.sum(np.conj(o.exact_response(uvs, x, my, mx)) * w * v))
    assert abs(lhs - np.sum(x * o.exact_adjoint(uvs, w, v, ny, nx, my, mx))) <= 1e-12 * abs(lhs)
    # uv points ON grid cells: R^dagger N^-1 R is exactly the PSF convolution with the gridded weights (R5), so a major
    # cycle returns the residual of the minor cycle's own model, d = I^D - C I
    uvg = np.rint(uvs)
    wgrid = np.zeros((my, mx))
    for (u, vv), wk in zip(uvg, w):
        wgrid[int(vv) % my, int(u) % mx] += wk
        wgrid[int(-vv) % my, int(-u) % mx] += wk
    cx = o.psf_apply(wgrid[:, : nx + 1], x)
    assert np.allclose(o.exact_adjoint(uvg, w, o.exact_response(uvg, x, my, mx), ny, nx, my, mx), cx, rtol=1e-11, atol=1e-11 * np.abs(cx).max())
    dirty = rng.normal(size=(ny, nx))
    assert np.allclose(o.major_cycle_residual(uvg, w, dirty, x, my, mx), dirty - cx, atol=1e-10 * np.abs(cx).max())
    # off the grid the two differ (that difference is what the major cycle corrects)
    assert rel(o.exact_adjoint(uvs, w, o.exact_response(uvs, x, my, mx), ny, nx, my, mx), cx) > 1e-2


# ---------------------------------------------------------------------------------- embedding (reading R19)
def test_embedded_convolution_is_the_image_sized_convolution():
    """A 12 x 10 image in a 16 x 16 embedding: the linear convolution with the 24 x 20 PSF, computed on the 32 x 32 padded
    grid with the PSF copied to the offsets |d| < image size and zero elsewhere, equals the image-sized operator
    (checked against the O(N^4) direct sum) -- any padding of at least twice the image computes Eq. 14 exactly."""
    rng = np.random.default_rng(0)
    nyi, nxi, ny, nx = 12, 10, 16, 16
    w = wl.make_config(3, ny=nyi, nx=nxi, npts=400)
    psf = o.psf_from_weights(w.w_half[0])                      # [24, 20]
    x = rng.normal(size=(nyi, nxi))
    ref = o.conv_direct(psf, x)
    assert np.max(np.abs(o.psf_apply(w.w_half[0], x) - ref)) <= 1e-12 * np.max(np.abs(ref))
    big = np.zeros((2 * ny, 2 * nx))
    for dy in range(-nyi + 1, nyi):
        for dx in range(-nxi + 1, nxi):
            big[dy % (2 * ny), dx % (2 * nx)] = psf[dy % (2 * nyi), dx % (2 * nxi)]
    wbig = np.fft.rfft2(big) / (4 * ny * nx)
    assert np.max(np.abs(wbig.imag)) <= 1e-12 * np.max(np.abs(wbig.real))
    got = o.psf_apply(wbig.real, o.embed(x, ny, nx))[:nyi, :nxi]
    assert np.max(np.abs(got - ref)) <= 1e-12 * np.max(np.abs(ref))


def test_embedded_energy_gradient_and_metric():
    rng = np.random.default_rng(1)
    nyi, nxi, ny, nx = 12, 10, 16, 16
    w = wl.make_config(3, ny=nyi, nx=nxi, npts=400)
    wf = wl.make_config(1, n=16)
    amp, mu = wf.amp[0], float(np.log(np.median(w.sky_true)))
    xi = 0.3 * rng.normal(size=(ny, nx))
    e, g = o.energy_grad_embedded(w.w_half[0], w.dirty[0], amp, mu, xi)
    for _ in range(3):
        d = rng.normal(size=xi.shape)
        h = 1e-5
        fd = (o.energy_grad_embedded(w.w_half[0], w.dirty[0], amp, mu, xi + h * d)[0]
              - o.energy_grad_embedded(w.w_half[0], w.dirty[0], amp, mu, xi - h * d)[0]) / (2 * h)
        assert abs(fd - np.sum(g * d)) <= 1e-6 * max(abs(fd), np.linalg.norm(g))
    u, v = rng.normal(size=xi.shape), rng.normal(size=xi.shape)
    mu_, mv = (o.metric_apply_embedded(w.w_half[0], nyi, nxi, amp, mu, xi, t) for t in (u, v))
    assert abs(np.sum(v * mu_) - np.sum(u * mv)) <= 1e-12 * abs(np.sum(v * mu_)) and np.sum(u * mu_) >= np.sum(u * u)
    # image = embedding grid: the plain functions
    w16 = wl.make_config(1, n=16)
    e0, g0 = o.energy_grad(w16.w_half, w16.dirty, w16.amp, [mu], w16.lognu, xi[None])
    e1, g1 = o.energy_grad_embedded(w16.w_half[0], w16.dirty[0], w16.amp[0], mu, xi)
    assert abs(e0 - e1) <= 1e-12 * abs(e0) and np.max(np.abs(g0[0] - g1)) <= 1e-12 * np.max(np.abs(g1))
