"""Pins of oracle/prior_oracle.py (NEXT-3, readings R17): everything here is CPU-only and checks the oracle against
things other than itself -- a hand-worked fixture, closed forms, quadrature, finite differences, dense Jacobians."""
import os

import numpy as np

from gen import workloads as wl
from oracle import frs_oracle as fo
from oracle import prior_oracle as po

HYPER = (18.0, 1.0, 0.1, 5.0, 1.0, -2.0, 0.2, 1.2, 0.4, 0.2, 0.2)      # Table A.1, S band
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_bins_hand_worked_4x4():
    rows = [l.split() for l in open(os.path.join(GOLD, "hand_bins_4x4.txt")) if l.strip() and not l.startswith("#")]
    b_ref = np.array(rows[:4], dtype=np.int64)
    mult_ref = np.array(rows[4], dtype=np.float64)
    b, mult, t = po.bins(4, 4)
    assert np.array_equal(b, b_ref) and np.array_equal(mult, mult_ref)
    assert t[0] == 0.0 and np.allclose(t[1:], np.log([1.0, 2.0, 3.0]), rtol=0, atol=1e-15)


def test_bins_rectangle_uses_the_longer_side_and_is_even():
    b, mult, t = po.bins(8, 32)
    assert b[1, 0] == 4 and b[0, 1] == 1 and b[4, 16] == np.rint(np.hypot(16, 16))      # fy scaled by 32 / 8
    assert np.array_equal(b, b[(-np.arange(8)) % 8][:, (-np.arange(32)) % 32])           # b[-k] = b[k]: A is even (R6)
    assert mult.sum() == 8 * 32 and mult[0] == 1


def test_lognormal_has_the_stated_mean_and_std():
    x, w = np.polynomial.hermite_e.hermegauss(80)
    w = w / np.sqrt(2 * np.pi)
    for m, s in ((5.0, 1.0), (1.2, 0.4), (0.2, 0.2), (1.0, 0.1)):
        v = po.lognormal(x, m, s)
        mean = np.sum(w * v)
        assert abs(mean - m) <= 1e-10 * m and abs(np.sqrt(np.sum(w * v * v) - mean ** 2) - s) <= 1e-8 * s


def test_total_fluctuation_variance_and_zero_mode():
    rng = np.random.default_rng(0)
    ny, nx = 16, 32
    _, _, t = po.bins(ny, nx)
    th = rng.normal(size=po.ntheta(len(t)))
    a = po.amplitude(th, HYPER, ny, nx)
    fl, zm = po.lognormal(th[0], 5.0, 1.0), po.lognormal(th[4], 1.0, 0.1)
    assert abs(np.sum(a ** 2) - (fl ** 2 + zm ** 2)) <= 1e-12 * fl ** 2 and a[0, 0] == zm and np.all(a > 0)
    # Var(lin[x]) = sum A^2 (frs_oracle pin "Correlated field"): Monte Carlo over white xi at one pixel, ~1 %
    xi = rng.normal(size=(4000, ny, nx))
    lin0 = np.einsum("nyx,yx->n", xi, a)                    # H[A xi] at x = 0: cas = 1 for every mode
    assert abs(lin0.var() / (fl ** 2 + zm ** 2) - 1.0) < 0.08


def test_pure_power_law_without_walk():
    ny = nx = 32
    b, mult, t = po.bins(ny, nx)
    th = np.zeros(po.ntheta(len(t)))
    th[1] = 0.7
    slope = -2.0 + 0.2 * 0.7
    a = po.amplitude(th, HYPER, ny, nx)
    k = np.maximum(b, 1).astype(np.float64)
    ref = k ** (slope / 2)
    ref[0, 0] = 0.0
    ref *= po.lognormal(0.0, 5.0, 1.0) / np.sqrt(np.sum(ref ** 2))
    ref[0, 0] = po.lognormal(0.0, 1.0, 0.1)
    assert np.max(np.abs(a - ref)) <= 1e-13 * ref.max()


def test_walk_single_kick_closed_forms():
    """One zeta_j = 1: vel jumps by flex sqrt(D_j) at j+1, so dev_b = flex sqrt(D_j) (t_b - t_{j+1}) for b > j.
    One eta_j = 1: dev jumps by flex asp sqrt(D_j) and stays."""
    ny = nx = 32
    b, mult, t = po.bins(ny, nx)
    nb, n, j = len(t), len(t) - 2, 5
    flex, asp = po.lognormal(0.0, 1.2, 0.4), po.lognormal(0.0, 0.2, 0.2)
    d = t[j + 1] - t[j]
    for kind in (0, 1):
        th = np.zeros(po.ntheta(nb))
        th[po.NSCALAR + kind * n + (j - 1)] = 1.0
        ab = po.bin_amplitudes(th, HYPER, mult, t)
        dev = 2.0 * np.log(ab[1:] / ab[1]) - (-2.0) * t[1:]                 # ln P_b - slope t_b, relative to b = 1
        ref = np.zeros(nb - 1)
        bb = np.arange(1, nb)
        ref[bb > j] = flex * np.sqrt(d) * (t[bb[bb > j]] - t[j + 1]) if kind == 0 else flex * asp * np.sqrt(d)
        assert np.max(np.abs(dev - ref)) <= 1e-12


def test_jvp_vjp_against_finite_differences_dense_jacobian_and_each_other():
    rng = np.random.default_rng(3)
    ny, nx = 16, 16
    b, mult, t = po.bins(ny, nx)
    nb = len(t)
    th = 0.5 * rng.normal(size=po.ntheta(nb))
    d = rng.normal(size=po.ntheta(nb))
    g = rng.normal(size=(ny, nx))
    jv = po.amplitude_jvp(th, d, HYPER, ny, nx)
    h = 1e-6
    fd = (po.amplitude(th + h * d, HYPER, ny, nx) - po.amplitude(th - h * d, HYPER, ny, nx)) / (2 * h)
    assert np.linalg.norm(fd - jv) <= 1e-6 * np.linalg.norm(jv)
    jac = po.bin_jacobian(th, HYPER, mult, t)
    vj = po.amplitude_vjp(th, g, HYPER, ny, nx)
    ref = jac.T @ np.bincount(b.ravel(), weights=g.ravel(), minlength=nb)
    assert np.max(np.abs(vj - ref)) <= 1e-12 * np.max(np.abs(ref))
    assert abs(np.sum(jv * g) - np.sum(d * vj)) <= 1e-12 * abs(np.sum(jv * g))


def _problem(n=16, seed=5):
    from gen import workloads as wl
    w = wl.make_config(1, n=n, seed=seed)
    rng = np.random.default_rng(seed)
    _, _, t = po.bins(n, n)
    hyper = (float(np.log(np.median(w.sky_true))), 1.0, 0.1, 1.0, 0.3, -3.0, 0.2, 0.5, 0.2, 0.2, 0.1)
    xi = 0.3 * rng.normal(size=(n, n))
    th = 0.3 * rng.normal(size=po.ntheta(len(t)))
    return w, hyper, xi, th, rng


def test_joint_gradient_against_central_differences():
    w, hyper, xi, th, rng = _problem()
    e, gx, gt = po.energy_grad_joint(w.w_half[0], w.dirty[0], hyper, xi, th)
    for _ in range(4):
        dx, dt = rng.normal(size=xi.shape), rng.normal(size=th.shape)
        h = 1e-5
        ep = po.energy_grad_joint(w.w_half[0], w.dirty[0], hyper, xi + h * dx, th + h * dt)[0]
        em = po.energy_grad_joint(w.w_half[0], w.dirty[0], hyper, xi - h * dx, th - h * dt)[0]
        lin = np.sum(gx * dx) + np.sum(gt * dt)
        assert abs((ep - em) / (2 * h) - lin) <= 1e-6 * max(abs(lin), np.linalg.norm(gx) + np.linalg.norm(gt))
    # theta fixed: the joint model is the fixed-amplitude model of frs_oracle at A(theta)
    a = po.amplitude(th, hyper, *xi.shape)
    e0, g0 = fo.energy_grad(w.w_half, w.dirty, a[None], [hyper[0]], w.lognu, xi[None], True)
    assert abs(e0 + 0.5 * np.sum(th * th) - e) <= 1e-12 * abs(e) and np.max(np.abs(g0[0] - gx)) <= 1e-10 * np.max(np.abs(gx))


def test_joint_metric_symmetric_and_at_least_identity():
    w, hyper, xi, th, rng = _problem()
    u = (rng.normal(size=xi.shape), rng.normal(size=th.shape))
    v = (rng.normal(size=xi.shape), rng.normal(size=th.shape))
    mu = po.metric_apply_joint(w.w_half[0], hyper, xi, th, *u)
    mv = po.metric_apply_joint(w.w_half[0], hyper, xi, th, *v)
    a, b = np.sum(v[0] * mu[0]) + np.sum(v[1] * mu[1]), np.sum(u[0] * mv[0]) + np.sum(u[1] * mv[1])
    assert abs(a - b) <= 1e-11 * abs(a)
    assert np.sum(u[0] * mu[0]) + np.sum(u[1] * mu[1]) >= np.sum(u[0] ** 2) + np.sum(u[1] ** 2)
    # dtheta = 0 reduces to the fixed-amplitude metric of frs_oracle
    am = po.amplitude(th, hyper, *xi.shape)
    m0 = fo.metric_apply(w.w_half, am[None], [hyper[0]], w.lognu, xi[None], u[0][None], True)
    mj = po.metric_apply_joint(w.w_half[0], hyper, xi, th, u[0], np.zeros_like(th))
    assert np.max(np.abs(m0[0] - mj[0])) <= 1e-10 * np.max(np.abs(m0))


def test_joint_eq9_gradient_against_central_differences_and_metric_symmetry():
    w, hyper, xi, th, rng = _problem()
    kern = fo.noise_kernel_from_psf(w.w_half[0], 1e-2 * float(fo.psf_from_weights(w.w_half[0])[0, 0]))
    e, gx, gt = po.energy_grad_joint(w.w_half[0], w.dirty[0], hyper, xi, th, True, kern)
    dx, dt = rng.normal(size=xi.shape), rng.normal(size=th.shape)
    h = 1e-5
    ep = po.energy_grad_joint(w.w_half[0], w.dirty[0], hyper, xi + h * dx, th + h * dt, True, kern)[0]
    em = po.energy_grad_joint(w.w_half[0], w.dirty[0], hyper, xi - h * dx, th - h * dt, True, kern)[0]
    lin = np.sum(gx * dx) + np.sum(gt * dt)
    assert abs((ep - em) / (2 * h) - lin) <= 1e-6 * max(abs(lin), np.linalg.norm(gx) + np.linalg.norm(gt))
    u = (rng.normal(size=xi.shape), rng.normal(size=th.shape))
    mu = po.metric_apply_joint(w.w_half[0], hyper, xi, th, dx, dt, True, kern)
    mv = po.metric_apply_joint(w.w_half[0], hyper, xi, th, u[0], u[1], True, kern)
    a, b = np.sum(u[0] * mu[0]) + np.sum(u[1] * mu[1]), np.sum(dx * mv[0]) + np.sum(dt * mv[1])
    assert abs(a - b) <= 1e-11 * abs(a)


# ---------------------------------------------------------------------------------- point sources (reading R18)
def test_point_flux_closed_form_moments_and_derivative():
    from scipy import integrate, special
    xi = np.array([-8.0, -3.0, -1.0, 0.0, 0.5, 2.0, 5.0, 8.0])
    # alpha = 1: F(x) = exp(-q / x)  =>  flux = -q / ln Phi(xi), written for each tail without cancellation
    ref = -2.0 / np.where(xi < 0, np.log(special.ndtr(xi)), np.log1p(-special.ndtr(-xi)))
    assert np.max(np.abs(po.point_flux(xi, 1.0, 2.0) / ref - 1.0)) <= 1e-12
    # monotone, positive, median = q / Q^-1(alpha, 1/2)
    f = po.point_flux(np.linspace(-8, 8, 201), 0.5, 1e-4)
    assert np.all(f > 0) and np.all(np.diff(f) > 0)
    # alpha = 3, q = 2: mean q / (alpha - 1) = 1, variance q^2 / ((alpha-1)^2 (alpha-2)) = 1  (xi standard normal)
    phi = lambda t: np.exp(-0.5 * t * t) / np.sqrt(2 * np.pi)  # noqa: E731
    m1 = integrate.quad(lambda t: po.point_flux(t, 3.0, 2.0) * phi(t), -14, 14, limit=400)[0]
    m2 = integrate.quad(lambda t: po.point_flux(t, 3.0, 2.0) ** 2 * phi(t), -14, 14, limit=400)[0]
    assert abs(m1 - 1.0) <= 1e-7 and abs(m2 - m1 * m1 - 1.0) <= 1e-4
    h = 1e-6
    fd = (po.point_flux(xi + h, 0.5, 1e-4) - po.point_flux(xi - h, 0.5, 1e-4)) / (2 * h)
    assert np.max(np.abs(po.point_flux_prime(xi, 0.5, 1e-4) / fd - 1.0)) <= 1e-6


def _full_problem():
    w, hyper, xi, th, rng = _problem()
    n = xi.shape[0]
    pts = (np.array([[n // 2, n // 2], [n // 2 + 1, n // 2 - 2], [0, n - 1]]), 0.5, 0.05 * float(np.median(w.sky_true)))
    xp = np.array([0.8, -0.4, 1.5])
    return w, hyper, xi, th, pts, xp, rng


def test_full_model_gradient_against_central_differences():
    w, hyper, xi, th, pts, xp, rng = _full_problem()
    for kern in (None, fo.noise_kernel_from_psf(w.w_half[0], 1e-2 * float(fo.psf_from_weights(w.w_half[0])[0, 0]))):
        e, gx, gt, gp = po.energy_grad_full(w.w_half[0], w.dirty[0], hyper, xi, th, pts, xp, True, kern)
        for _ in range(3):
            dx, dt, dp = rng.normal(size=xi.shape), rng.normal(size=th.shape), rng.normal(size=xp.shape)
            h = 1e-5
            ep = po.energy_grad_full(w.w_half[0], w.dirty[0], hyper, xi + h * dx, th + h * dt, pts, xp + h * dp, True, kern)[0]
            em = po.energy_grad_full(w.w_half[0], w.dirty[0], hyper, xi - h * dx, th - h * dt, pts, xp - h * dp, True, kern)[0]
            lin = np.sum(gx * dx) + np.sum(gt * dt) + np.sum(gp * dp)
            assert abs((ep - em) / (2 * h) - lin) <= 1e-6 * max(abs(lin), np.linalg.norm(gx) + np.linalg.norm(gt) + np.linalg.norm(gp))
    # the sky has the fluxes added exactly at the listed pixels
    s, s_diff, _ = po.sky_full(hyper, xi, th, pts, xp)
    d = s - s_diff
    fl = po.point_flux(xp, pts[1], pts[2])
    assert np.count_nonzero(d) == 3 and all(abs(d[y, x] - f) <= 1e-12 * f for (y, x), f in zip(pts[0], fl))


def test_full_model_metric_symmetric_and_reduces_to_joint():
    w, hyper, xi, th, pts, xp, rng = _full_problem()
    u = (rng.normal(size=xi.shape), rng.normal(size=th.shape), rng.normal(size=xp.shape))
    v = (rng.normal(size=xi.shape), rng.normal(size=th.shape), rng.normal(size=xp.shape))
    mu = po.metric_apply_full(w.w_half[0], hyper, xi, th, pts, xp, *u)
    mv = po.metric_apply_full(w.w_half[0], hyper, xi, th, pts, xp, *v)
    a = sum(np.sum(p * q) for p, q in zip(v, mu))
    b = sum(np.sum(p * q) for p, q in zip(u, mv))
    assert abs(a - b) <= 1e-11 * abs(a)
    assert sum(np.sum(p * q) for p, q in zip(u, mu)) >= sum(np.sum(p * p) for p in u)
    none = (np.zeros((0, 2), np.int64), 0.5, 1.0)
    m0 = po.metric_apply_full(w.w_half[0], hyper, xi, th, none, np.zeros(0), u[0], u[1], np.zeros(0))
    mj = po.metric_apply_joint(w.w_half[0], hyper, xi, th, u[0], u[1])
    assert np.array_equal(m0[0], mj[0]) and np.array_equal(m0[1], mj[1])


# ---------------------------------------------------------------------------------- several GPs on patches (reading R20)
def _patch_problem():
    w = wl.make_config(1, n=32, seed=4)
    rng = np.random.default_rng(9)
    mu = float(np.log(np.median(w.sky_true)))
    amp32 = w.amp[0]
    amp16 = wl.make_config(1, n=16, seed=4).amp[0]
    amp8x16 = wl.make_config(3, ny=8, nx=16, npts=300).amp[0]
    comps = [(amp32, mu - 1.0, 0, 0), (amp16, mu, 4, 10), (amp8x16, mu + 0.5, 20, 2)]
    xis = [0.3 * rng.normal(size=c[0].shape) for c in comps]
    return w, comps, xis, rng


def test_patch_model_gradient_metric_and_reduction():
    w, comps, xis, rng = _patch_problem()
    for kern in (None, fo.noise_kernel_from_psf(w.w_half[0], 1e-2 * float(fo.psf_from_weights(w.w_half[0])[0, 0]))):
        e, gs = po.energy_grad_patches(w.w_half[0], w.dirty[0], comps, xis, True, kern)
        ds = [rng.normal(size=x.shape) for x in xis]
        h = 1e-5
        ep = po.energy_grad_patches(w.w_half[0], w.dirty[0], comps, [x + h * d for x, d in zip(xis, ds)], True, kern)[0]
        em = po.energy_grad_patches(w.w_half[0], w.dirty[0], comps, [x - h * d for x, d in zip(xis, ds)], True, kern)[0]
        lin = sum(np.sum(g * d) for g, d in zip(gs, ds))
        assert abs((ep - em) / (2 * h) - lin) <= 1e-6 * max(abs(lin), sum(np.linalg.norm(g) for g in gs))
        us = [rng.normal(size=x.shape) for x in xis]
        mu_ = po.metric_apply_patches(w.w_half[0], 32, 32, comps, xis, us, True, kern)
        md = po.metric_apply_patches(w.w_half[0], 32, 32, comps, xis, ds, True, kern)
        a, b = sum(np.sum(p * q) for p, q in zip(ds, mu_)), sum(np.sum(p * q) for p, q in zip(us, md))
        assert abs(a - b) <= 1e-11 * abs(a)
    # the sky is the sum of the inserted parts; one full-field component is the plain model of frs_oracle
    s, parts = po.sky_patches(comps, xis, 32, 32)
    ref = np.zeros((32, 32))
    ref[:, :] += parts[0]
    ref[4:20, 10:26] += parts[1]
    ref[20:28, 2:18] += parts[2]
    assert np.array_equal(s, ref)
    e1, g1 = po.energy_grad_patches(w.w_half[0], w.dirty[0], comps[:1], xis[:1])
    e0, g0 = fo.energy_grad(w.w_half, w.dirty, comps[0][0][None], [comps[0][1]], w.lognu, xis[0][None])
    assert abs(e1 - e0) <= 1e-12 * abs(e0) and np.max(np.abs(g1[0] - g0[0])) <= 1e-12 * np.max(np.abs(g0))


# ---------------------------------------------------------------------------------- the metrics against the Jacobian of their own sky
# Symmetry, M >= 1 and the reduction to a simpler model leave room for a consistent mistake in J and J^T together (the total
# instead of the diffuse sky at the point pixels; a dropped da . xi term).  Here J is assembled column by column from central
# differences of the very sky function the metric belongs to, M = J^T C J + 1 (Eq. 9 mode: J^T C N'^-1 C J + 1) is formed
# densely with frs_oracle's psf_apply / ninv_apply, and every column of it is compared with the metric applied to a unit vector.
def _dense_jacobian(sky_of, z, h=1e-3):
    """Five-point central differences (error O(h^4), rounding ~ 1e-16 / h): good to ~1e-10 of the sky's scale."""
    cols = []
    for i in range(z.size):
        e = np.zeros_like(z)
        e[i] = h
        d = (8.0 * (sky_of(z + e) - sky_of(z - e)) - (sky_of(z + 2 * e) - sky_of(z - 2 * e))) / (12.0 * h)
        cols.append(d.ravel())
    return np.stack(cols, axis=1)                                   # [npix, nlatent]


def _dense_metric(w_half_c, shape, jac, kern):
    def mid(col):
        c = fo.psf_apply(w_half_c, col.reshape(shape))
        if kern is not None:
            c = fo.psf_apply(w_half_c, fo.ninv_apply(kern, c))
        return c.ravel()
    cj = np.stack([mid(jac[:, i]) for i in range(jac.shape[1])], axis=1)
    return jac.T @ cj + np.eye(jac.shape[1])


def _kernels(w):
    return (None, fo.noise_kernel_from_psf(w.w_half[0], 1e-2 * float(fo.psf_from_weights(w.w_half[0])[0, 0])))


def test_full_model_metric_is_the_dense_jacobian_form_of_sky_full():
    n = 8
    w, hyper, xi, th, rng = _problem(n)
    pts = (np.array([[4, 4], [0, 7]]), 0.5, 0.05 * float(np.median(w.sky_true)))
    xp = np.array([0.8, -0.4])
    nx_, nt = xi.size, th.size
    z0 = np.concatenate([xi.ravel(), th, xp])
    sky_of = lambda z: po.sky_full(hyper, z[:nx_].reshape(n, n), z[nx_:nx_ + nt], pts, z[nx_ + nt:])[0]  # noqa: E731
    jac = _dense_jacobian(sky_of, z0)
    # the point columns of J are the flux derivative at the pixel and nothing else; the diffuse columns do NOT see the fluxes
    s, s_diff, _ = po.sky_full(hyper, xi, th, pts, xp)
    assert np.count_nonzero(np.abs(jac[:, nx_ + nt:]) > 1e-9 * np.max(np.abs(jac))) == 2
    for kern in _kernels(w):
        dense = _dense_metric(w.w_half[0], (n, n), jac, kern)
        for i in range(z0.size):
            e = np.zeros(z0.size)
            e[i] = 1.0
            ox, ot, op = po.metric_apply_full(w.w_half[0], hyper, xi, th, pts, xp, e[:nx_].reshape(n, n), e[nx_:nx_ + nt],
                                              e[nx_ + nt:], True, kern)
            col = np.concatenate([ox.ravel(), ot, op])
            assert np.max(np.abs(col - dense[:, i])) <= 1e-6 * np.max(np.abs(dense[:, i])), (i, kern is None)
    # the pin has teeth: the total sky in place of the diffuse one at the point pixels moves the metric far beyond the bound
    jbad = jac.copy()
    for (y, x), st, sd in zip(pts[0], [s[4, 4], s[0, 7]], [s_diff[4, 4], s_diff[0, 7]]):
        jbad[y * n + x, :nx_ + nt] *= st / sd
    bad = _dense_metric(w.w_half[0], (n, n), jbad, None)
    good = _dense_metric(w.w_half[0], (n, n), jac, None)
    assert np.max(np.abs(bad - good)) > 1e-3 * np.max(np.abs(good))


def test_joint_metric_is_the_dense_jacobian_form_of_sky_joint():
    n = 8
    w, hyper, xi, th, rng = _problem(n)
    nx_ = xi.size
    z0 = np.concatenate([xi.ravel(), th])
    sky_of = lambda z: po.sky_joint(None, hyper, z[:nx_].reshape(n, n), z[nx_:])[0]  # noqa: E731
    jac = _dense_jacobian(sky_of, z0)
    assert np.max(np.abs(jac[:, nx_:])) > 1e-3 * np.max(np.abs(jac))            # the theta columns (the da . xi term) are not small
    for kern in _kernels(w):
        dense = _dense_metric(w.w_half[0], (n, n), jac, kern)
        for i in range(z0.size):
            e = np.zeros(z0.size)
            e[i] = 1.0
            ox, ot = po.metric_apply_joint(w.w_half[0], hyper, xi, th, e[:nx_].reshape(n, n), e[nx_:], True, kern)
            col = np.concatenate([ox.ravel(), ot])
            assert np.max(np.abs(col - dense[:, i])) <= 1e-6 * np.max(np.abs(dense[:, i])), (i, kern is None)


def test_patch_metric_is_the_dense_jacobian_form_of_sky_patches():
    w = wl.make_config(1, n=16, seed=4)
    rng = np.random.default_rng(9)
    mu = float(np.log(np.median(w.sky_true)))
    comps = [(w.amp[0], mu - 1.0, 0, 0), (wl.make_config(1, n=8, seed=4).amp[0], mu, 4, 6)]       # the patch overlaps the background
    xis = [0.3 * rng.normal(size=c[0].shape) for c in comps]
    sizes = [x.size for x in xis]
    split = lambda z: [z[:sizes[0]].reshape(xis[0].shape), z[sizes[0]:].reshape(xis[1].shape)]  # noqa: E731
    z0 = np.concatenate([x.ravel() for x in xis])
    jac = _dense_jacobian(lambda z: po.sky_patches(comps, split(z), 16, 16)[0], z0)
    for kern in _kernels(w):
        dense = _dense_metric(w.w_half[0], (16, 16), jac, kern)
        for i in range(0, z0.size, 3):                                             # every third unit vector: both components
            e = np.zeros(z0.size)
            e[i] = 1.0
            outs = po.metric_apply_patches(w.w_half[0], 16, 16, comps, xis, split(e), True, kern)
            col = np.concatenate([o_.ravel() for o_ in outs])
            assert np.max(np.abs(col - dense[:, i])) <= 1e-6 * np.max(np.abs(dense[:, i])), (i, kern is None)
