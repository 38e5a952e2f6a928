"""ORACLE -- test infrastructure, not product code.

NEXT-3 of SURVEY.md section 8(f): the learned amplitude spectrum of the diffuse-emission prior and the inverse-gamma
point-source pixels (parameters of Table A.1 / B.1).  The paper defers the
definitions to Arras et al. (2021a), which is not in the container, so what is written out here is the reading
DESIGN.md lists as R17 (amplitude model), R18 (point sources) and R20 (several GPs on patches), in float64, in the order
of that reading.  Pins: tests/test_prior_oracle_pins.py.
Shares no code with the CUDA path; imported only by tests/.

R17 in one place (ny x nx harmonic grid, standard-normal latent vector theta):
  bins      b(pixel) = rint(|k|), |k| = sqrt(fy^2 + fx^2) in cycles per LONGER field side, f = min(k, n - k) scaled by
            nmax / n;  nb = max b + 1;  mult_b = pixels in bin b;  t_b = ln b (b >= 1)
  theta     [xi_fluct, xi_slope, xi_flex, xi_asp, xi_zm, zeta_1 .. zeta_{nb-2}, eta_1 .. eta_{nb-2}]
  hyper     (offset, zm_mean, zm_std, fl_mean, fl_std, sl_mean, sl_std, fx_mean, fx_std, as_mean, as_std)   Table A.1
  lognormal LN(xi; m, s) = m / sqrt(1 + (s/m)^2) * exp(sqrt(ln(1 + (s/m)^2)) xi): mean m, standard deviation s
  fluct = LN(xi_fluct), slope = sl_mean + sl_std xi_slope, flex = LN(xi_flex), asp = LN(xi_asp), zm = LN(xi_zm)
  walk      dev_1 = vel_1 = 0;  D_j = t_{j+1} - t_j;
            dev_{j+1} = dev_j + vel_j D_j + flex asp sqrt(D_j) eta_j;  vel_{j+1} = vel_j + flex sqrt(D_j) zeta_j
  spectrum  ln P_b = slope t_b + dev_b;  a_b = exp(ln P_b / 2);  S = sum_{b>=1} mult_b a_b^2
  amplitude A[pixel] = fluct a_b / sqrt(S) (b >= 1),  A[zero mode] = zm      =>  sum_pixels A^2 = fluct^2 + zm^2
  sky       s = exp(offset + H[A . xi])   (frs_oracle.sky with mu = offset)
"""
from __future__ import annotations

import numpy as np

NHYPER = 11
NSCALAR = 5          # xi_fluct, xi_slope, xi_flex, xi_asp, xi_zm


# ----------------------------------------------------------------------------------------------- bins
def bins(ny, nx):
    """b[ky, kx] = rint(|k|) (int64), mult[b], t[b] = ln b (t[0] unused = 0)."""
    nmax = max(ny, nx)
    fy = np.minimum(np.arange(ny), ny - np.arange(ny)) * (nmax // ny)
    fx = np.minimum(np.arange(nx), nx - np.arange(nx)) * (nmax // nx)
    k2 = fy[:, None].astype(np.int64) ** 2 + fx[None, :].astype(np.int64) ** 2
    b = np.rint(np.sqrt(k2.astype(np.float64))).astype(np.int64)
    nb = int(b.max()) + 1
    mult = np.bincount(b.ravel(), minlength=nb).astype(np.float64)
    t = np.zeros(nb)
    t[1:] = np.log(np.arange(1, nb))
    return b, mult, t


def ntheta(nb):
    return NSCALAR + 2 * (nb - 2)


# ----------------------------------------------------------------------------------------------- scalars
def lognormal(xi, mean, std):
    """Log-normal variable with the given mean and standard deviation as a function of a standard normal xi."""
    r = 1.0 + (std / mean) ** 2
    return mean / np.sqrt(r) * np.exp(np.sqrt(np.log(r)) * xi)


def unpack(theta, nb):
    theta = np.asarray(theta)
    n = nb - 2
    return theta[:NSCALAR], theta[NSCALAR:NSCALAR + n], theta[NSCALAR + n:NSCALAR + 2 * n]


# ----------------------------------------------------------------------------------------------- forward
def bin_amplitudes(theta, hyper, mult, t):
    """A_b for b = 0 .. nb-1 (the walk written as the plain loop of the reading).  Works for complex theta too
    (used by the complex-step derivative below), hence no float() casts."""
    nb = len(t)
    sc, zeta, eta = unpack(theta, nb)
    _, zm_m, zm_s, fl_m, fl_s, sl_m, sl_s, fx_m, fx_s, as_m, as_s = hyper
    fluct = lognormal(sc[0], fl_m, fl_s)
    slope = sl_m + sl_s * sc[1]
    flex = lognormal(sc[2], fx_m, fx_s)
    asp = lognormal(sc[3], as_m, as_s)
    zm = lognormal(sc[4], zm_m, zm_s)
    dtype = np.result_type(np.asarray(theta).dtype, np.float64)
    dev = np.zeros(nb, dtype)
    vel = np.zeros(nb, dtype)
    for j in range(1, nb - 1):
        d = t[j + 1] - t[j]
        dev[j + 1] = dev[j] + vel[j] * d + flex * asp * np.sqrt(d) * eta[j - 1]
        vel[j + 1] = vel[j] + flex * np.sqrt(d) * zeta[j - 1]
    a = np.zeros(nb, dtype)
    a[1:] = np.exp(0.5 * (slope * t[1:] + dev[1:]))
    s = np.sum(mult[1:] * a[1:] ** 2)
    out = np.zeros(nb, dtype)
    out[1:] = fluct * a[1:] / np.sqrt(s)
    out[0] = zm
    return out


def amplitude(theta, hyper, ny, nx):
    """A [ny, nx] (harmonic order) of the reading R17."""
    b, mult, t = bins(ny, nx)
    return bin_amplitudes(theta, hyper, mult, t)[b]


# ----------------------------------------------------------------------------------------------- derivatives
def amplitude_jvp(theta, dtheta, hyper, ny, nx, h=1e-30):
    """dA = (dA/dtheta) dtheta by the complex-step derivative of the forward function: exact to rounding and
    independent of any hand-derived formula (the forward map is analytic in theta)."""
    b, mult, t = bins(ny, nx)
    z = np.asarray(theta, np.complex128) + 1j * h * np.asarray(dtheta, np.float64)
    return (np.imag(bin_amplitudes(z, hyper, mult, t)) / h)[b]


def bin_jacobian(theta, hyper, mult, t):
    """Dense dA_b / dtheta_i [nb, ntheta], column by column with the complex step (small nb only)."""
    nb = len(t)
    n = ntheta(nb)
    jac = np.zeros((nb, n))
    for i in range(n):
        z = np.asarray(theta, np.complex128).copy()
        z[i] += 1e-30j
        jac[:, i] = np.imag(bin_amplitudes(z, hyper, mult, t)) / 1e-30
    return jac


def amplitude_vjp(theta, g_a, hyper, ny, nx):
    """g_theta = (dA/dtheta)^T g_A, the adjoint of the reading written out (reverse sweep of the walk)."""
    b, mult, t = bins(ny, nx)
    nb = len(t)
    g = np.bincount(b.ravel(), weights=np.asarray(g_a, np.float64).ravel(), minlength=nb)    # G_b = sum over the bin
    sc, zeta, eta = unpack(np.asarray(theta, np.float64), nb)
    _, zm_m, zm_s, fl_m, fl_s, sl_m, sl_s, fx_m, fx_s, as_m, as_s = hyper
    sig = lambda m, s: np.sqrt(np.log(1.0 + (s / m) ** 2))  # noqa: E731
    flex = lognormal(sc[2], fx_m, fx_s)
    asp = lognormal(sc[3], as_m, as_s)
    zm = lognormal(sc[4], zm_m, zm_s)
    a_b = bin_amplitudes(theta, hyper, mult, t)
    # A_b = fluct a_b / sqrt(S):  dA_b = A_b (dfluct / fluct + dlnP_b / 2 - dS / (2 S)),  dS / S = sum_b w_b dlnP_b
    q = a_b * g
    q[0] = 0.0
    qsum = np.sum(q)
    w = mult * a_b ** 2
    w[0] = 0.0
    w /= np.sum(w)                                        # = mult_b a_b^2 / S  (the fluct^2 cancels)
    lbar = 0.5 * q - 0.5 * qsum * w                       # adjoint of ln P_b
    out = np.zeros(ntheta(nb))
    out[0] = sig(fl_m, fl_s) * qsum
    out[1] = sl_s * np.sum(lbar * t)
    out[4] = zm * sig(zm_m, zm_s) * g[0]
    dbar = np.zeros(nb + 1)                               # D_b = sum_{b' >= b} lbar_b'
    for bb in range(nb - 1, 0, -1):
        dbar[bb] = dbar[bb + 1] + lbar[bb]
    vbar = np.zeros(nb + 1)                               # adjoint of vel_b
    fxbar = asbar = 0.0
    n = nb - 2
    for j in range(nb - 2, 0, -1):
        d = t[j + 1] - t[j]
        vbar[j] = vbar[j + 1] + d * dbar[j + 1]
        out[NSCALAR + n + (j - 1)] = flex * asp * np.sqrt(d) * dbar[j + 1]          # eta_j
        out[NSCALAR + (j - 1)] = flex * np.sqrt(d) * vbar[j + 1]                    # zeta_j
        fxbar += np.sqrt(d) * (asp * eta[j - 1] * dbar[j + 1] + zeta[j - 1] * vbar[j + 1])
        asbar += np.sqrt(d) * flex * eta[j - 1] * dbar[j + 1]
    out[2] = flex * sig(fx_m, fx_s) * fxbar
    out[3] = asp * sig(as_m, as_s) * asbar
    return out


# ----------------------------------------------------------------------------------------------- joint model
# Likelihood of DESIGN.md R1 (E_lh = 1/2 <s, C s> - <j, s>, single channel, one field) on the joint latent vector
# (xi, theta), prior 1/2 <xi, xi> + 1/2 <theta, theta>.  The convolution and the Hartley transform are the ones of
# frs_oracle (pinned there); what is new is the dependence of A on theta.
def _fo():
    from oracle import frs_oracle as fo
    return fo


def sky_joint(w_unused, hyper, xi, theta):
    fo = _fo()
    ny, nx = xi.shape
    a = amplitude(theta, hyper, ny, nx)
    return np.exp(hyper[0] + fo.hartley2(a * np.asarray(xi, np.float64))), a


def energy_grad_joint(w_half_c, dirty, hyper, xi, theta, with_prior=True, kern=None):
    """E(xi, theta), dE/dxi [ny, nx], dE/dtheta [ntheta].  kern = None: the N' = R' likelihood (R1); kern = K [ny, nx]:
    Eq. 9 with N'^-1 of Eq. 18 (R14), E_lh = 1/2 r^T N'^-1 r, r = j - C s."""
    fo = _fo()
    xi = np.asarray(xi, np.float64)
    theta = np.asarray(theta, np.float64)
    ny, nx = xi.shape
    s, a = sky_joint(None, hyper, xi, theta)
    cs = fo.psf_apply(w_half_c, s)
    if kern is None:
        e = 0.5 * np.sum(s * cs) - np.sum(np.asarray(dirty, np.float64) * s)
        h = fo.hartley2(s * (cs - dirty))
    else:
        r = np.asarray(dirty, np.float64) - cs
        u = fo.ninv_apply(kern, r)
        e = 0.5 * np.sum(r * u)
        h = -fo.hartley2(s * fo.psf_apply(w_half_c, u))
    g_xi = a * h
    g_th = amplitude_vjp(theta, xi * h, hyper, ny, nx)
    if with_prior:
        e += 0.5 * np.sum(xi * xi) + 0.5 * np.sum(theta * theta)
        g_xi = g_xi + xi
        g_th = g_th + theta
    return float(e), g_xi, g_th


def metric_apply_joint(w_half_c, hyper, xi, theta, dxi, dtheta, with_prior=True, kern=None):
    """Fisher metric J^T C J (+ 1) of the joint model applied to (dxi, dtheta); J = ds/d(xi, theta).
    kern given: J^T C N'^-1 C J (+ 1)."""
    fo = _fo()
    xi = np.asarray(xi, np.float64)
    ny, nx = xi.shape
    s, a = sky_joint(None, hyper, xi, theta)
    da = amplitude_jvp(theta, dtheta, hyper, ny, nx)
    dtau = fo.hartley2(a * np.asarray(dxi, np.float64) + da * xi)
    cj = fo.psf_apply(w_half_c, s * dtau)
    if kern is not None:
        cj = fo.psf_apply(w_half_c, fo.ninv_apply(kern, cj))
    h = fo.hartley2(s * cj)
    o_xi = a * h
    o_th = amplitude_vjp(theta, xi * h, hyper, ny, nx)
    if with_prior:
        o_xi = o_xi + dxi
        o_th = o_th + np.asarray(dtheta, np.float64)
    return o_xi, o_th


# ----------------------------------------------------------------------------------------------- point sources (R18)
# P:92 "pixels are independently modeled with an inverse gamma prior for their intensity ... the locations currently
# need to be manually set"; P:294 two such pixels in the core of Cygnus A.  The paper gives no formula; reading R18:
# flux_p = F^-1(Phi(xi_p)) with F the CDF of the inverse-gamma distribution pdf(x) ~ x^(-alpha-1) exp(-q / x) and Phi the
# standard normal CDF (so that xi_p is standard normal), added to the diffuse sky at pixel (y_p, x_p):
#   s = exp(offset + H[A xi]) + sum_p flux_p e_p.
# scipy's incomplete-gamma inverses are the library step (pinned in tests by the alpha = 1 closed form and by moments).
def point_flux(xi_p, alpha, q):
    from scipy import special
    xi_p = np.asarray(xi_p, np.float64)
    # F(x) = Q(alpha, q / x) (regularised upper incomplete gamma).  Solve in the tail that keeps precision:
    # xi >= 0: P(alpha, y) = Phi(-xi);  xi < 0: Q(alpha, y) = Phi(xi);  flux = q / y
    lo = special.gammaincinv(alpha, special.ndtr(-np.abs(xi_p)))          # for xi >= 0
    hi = special.gammainccinv(alpha, special.ndtr(-np.abs(xi_p)))         # for xi < 0
    return q / np.where(xi_p >= 0, lo, hi)


def point_flux_prime(xi_p, alpha, q):
    """d flux / d xi = phi(xi) / pdf(flux), pdf(x) = q^alpha / Gamma(alpha) x^(-alpha-1) exp(-q / x)."""
    from scipy import special
    xi_p = np.asarray(xi_p, np.float64)
    x = point_flux(xi_p, alpha, q)
    logpdf = alpha * np.log(q) - special.gammaln(alpha) - (alpha + 1.0) * np.log(x) - q / x
    return np.exp(-0.5 * xi_p ** 2 - 0.5 * np.log(2 * np.pi) - logpdf)


def sky_full(hyper, xi, theta_amp, pts, xi_pts):
    """Diffuse sky plus point sources.  pts = (yx [npts, 2] int, alpha, q)."""
    s, a = sky_joint(None, hyper, xi, theta_amp)
    s_diff = s.copy()
    yx, alpha, q = pts
    fl = point_flux(xi_pts, alpha, q)
    for (y, x), f in zip(yx, fl):
        s[y, x] += f
    return s, s_diff, a


def energy_grad_full(w_half_c, dirty, hyper, xi, theta_amp, pts, xi_pts, with_prior=True, kern=None):
    """E and its gradient with respect to (xi, theta_amp, xi_pts)."""
    fo = _fo()
    xi = np.asarray(xi, np.float64)
    theta_amp = np.asarray(theta_amp, np.float64)
    xi_pts = np.asarray(xi_pts, np.float64)
    ny, nx = xi.shape
    s, s_diff, a = sky_full(hyper, xi, theta_amp, pts, xi_pts)
    cs = fo.psf_apply(w_half_c, s)
    if kern is None:
        e = 0.5 * np.sum(s * cs) - np.sum(np.asarray(dirty, np.float64) * s)
        gs = cs - dirty                                   # dE / ds
    else:
        r = np.asarray(dirty, np.float64) - cs
        u = fo.ninv_apply(kern, r)
        e = 0.5 * np.sum(r * u)
        gs = -fo.psf_apply(w_half_c, u)
    h = fo.hartley2(s_diff * gs)
    g_xi = a * h
    g_th = amplitude_vjp(theta_amp, xi * h, hyper, ny, nx)
    yx, alpha, q = pts
    g_pt = point_flux_prime(xi_pts, alpha, q) * np.array([gs[y, x] for y, x in yx])
    if with_prior:
        e += 0.5 * np.sum(xi * xi) + 0.5 * np.sum(theta_amp ** 2) + 0.5 * np.sum(xi_pts ** 2)
        g_xi, g_th, g_pt = g_xi + xi, g_th + theta_amp, g_pt + xi_pts
    return float(e), g_xi, g_th, g_pt


def metric_apply_full(w_half_c, hyper, xi, theta_amp, pts, xi_pts, dxi, dtheta, dpts, with_prior=True, kern=None):
    fo = _fo()
    xi = np.asarray(xi, np.float64)
    ny, nx = xi.shape
    s, s_diff, a = sky_full(hyper, xi, theta_amp, pts, xi_pts)
    yx, alpha, q = pts
    fp = point_flux_prime(xi_pts, alpha, q)
    da = amplitude_jvp(theta_amp, dtheta, hyper, ny, nx)
    ds = s_diff * fo.hartley2(a * np.asarray(dxi, np.float64) + da * xi)          # J (dxi, dtheta, dpts)
    for (y, x), f, d in zip(yx, fp, np.asarray(dpts, np.float64)):
        ds[y, x] += f * d
    c = fo.psf_apply(w_half_c, ds)
    if kern is not None:
        c = fo.psf_apply(w_half_c, fo.ninv_apply(kern, c))
    h = fo.hartley2(s_diff * c)
    o_xi = a * h
    o_th = amplitude_vjp(theta_amp, xi * h, hyper, ny, nx)
    o_pt = fp * np.array([c[y, x] for y, x in yx])
    if with_prior:
        o_xi, o_th, o_pt = o_xi + dxi, o_th + np.asarray(dtheta, np.float64), o_pt + np.asarray(dpts, np.float64)
    return o_xi, o_th, o_pt


# ----------------------------------------------------------------------------------------------- several GPs on patches (R20)
# P:369 "We model each of these sources with a separate exponentiated Gaussian process ... a third Gaussian process model
# to represent all the background sources" (Fig. 10: two source patches inside a background field).  Reading R20: component k
# has its own grid (ny_k x nx_k), amplitude A_k, offset mu_k and excitations xi_k; its sky exp(mu_k + H_k[A_k xi_k]) is ADDED
# into the full field at the patch position (y0_k, x0_k); the components may overlap (the background covers everything).
#   s = sum_k insert_k( exp(mu_k + H_k[A_k xi_k]) ),   E = E_lh(s) + 1/2 sum_k <xi_k, xi_k>.
# comps: list of (amp_k [ny_k, nx_k], mu_k, y0_k, x0_k).
def sky_patches(comps, xis, ny, nx):
    fo = _fo()
    s = np.zeros((ny, nx))
    parts = []
    for (amp, mu, y0, x0), xi in zip(comps, xis):
        sk = np.exp(mu + fo.hartley2(np.asarray(amp, np.float64) * np.asarray(xi, np.float64)))
        parts.append(sk)
        s[y0:y0 + sk.shape[0], x0:x0 + sk.shape[1]] += sk
    return s, parts


def _dE_ds(w_half_c, dirty, s, kern):
    fo = _fo()
    cs = fo.psf_apply(w_half_c, s)
    if kern is None:
        return 0.5 * np.sum(s * cs) - np.sum(np.asarray(dirty, np.float64) * s), cs - dirty
    r = np.asarray(dirty, np.float64) - cs
    u = fo.ninv_apply(kern, r)
    return 0.5 * np.sum(r * u), -fo.psf_apply(w_half_c, u)


def energy_grad_patches(w_half_c, dirty, comps, xis, with_prior=True, kern=None):
    """E and the list of dE/dxi_k."""
    fo = _fo()
    ny, nx = dirty.shape
    s, parts = sky_patches(comps, xis, ny, nx)
    e, gs = _dE_ds(w_half_c, dirty, s, kern)
    grads = []
    for (amp, mu, y0, x0), xi, sk in zip(comps, xis, parts):
        g = np.asarray(amp, np.float64) * fo.hartley2(sk * gs[y0:y0 + sk.shape[0], x0:x0 + sk.shape[1]])
        if with_prior:
            e += 0.5 * np.sum(np.asarray(xi, np.float64) ** 2)
            g = g + xi
        grads.append(g)
    return float(e), grads


def metric_apply_patches(w_half_c, ny, nx, comps, xis, vs, with_prior=True, kern=None):
    """Fisher metric J^T C J (+ 1) (kern: J^T C N'^-1 C J) of the patch model applied to the list vs."""
    fo = _fo()
    _, parts = sky_patches(comps, xis, ny, nx)
    ds = np.zeros((ny, nx))
    for (amp, mu, y0, x0), v, sk in zip(comps, vs, parts):
        ds[y0:y0 + sk.shape[0], x0:x0 + sk.shape[1]] += sk * fo.hartley2(np.asarray(amp, np.float64) * np.asarray(v, np.float64))
    c = fo.psf_apply(w_half_c, ds)
    if kern is not None:
        c = fo.psf_apply(w_half_c, fo.ninv_apply(kern, c))
    outs = []
    for (amp, mu, y0, x0), v, sk in zip(comps, vs, parts):
        o_ = np.asarray(amp, np.float64) * fo.hartley2(sk * c[y0:y0 + sk.shape[0], x0:x0 + sk.shape[1]])
        outs.append(o_ + v if with_prior else o_)
    return outs
