"""ORACLE -- test infrastructure, not product code.

Plain, slow, float64 CPU statement of what the fast-resolve hot path computes, written
from the paper (`P:<n>` = /root/reference/PAPER.md line n) and from the readings listed in
DESIGN.md ("Readings", R1..R10 = SURVEY.md section 8(c) items c-1..c-10).  It shares no
code with the CUDA path and is imported only by tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.

Library primitives used as steps: numpy.fft (pinned in tests against the O(n^2) DFT written
out below and against the O(N^4) direct convolution), numpy.linalg.solve (CG pin only).

Pins: tests/test_oracle_pins.py (every function, incl. sky / log_sky / channel_coeff through the
hand-worked fixture tests/golden/hand_sky_two_fields.txt, the Eq. 9 / Eq. 15-18 functions, and the embedded
(non-power-of-two) functions of reading R19 through the O(N^4) direct sum and finite differences).
"parity unpinned": the absolute values of E and grad on real data -- the paper prints no operator
value (last pin row); they are pinned only through the identities tested there.

Shapes:  xi, amp  [nfield, ny, nx];  mu [nfield];  lognu [nchan];
         w_half   [nchan, My, nx+1]  (My = 2 ny, Mx = 2 nx; real >= 0 half spectrum of the PSF);
         dirty j, sky s  [nchan, ny, nx].
"""
from __future__ import annotations

import numpy as np

F64 = np.float64


# =============================================================================
# Definitions written out (used by the pins; O(n^2) / O(N^4))
# =============================================================================
def dft_naive(x, sign=-1):
    """X[k] = sum_n x[n] exp(sign 2 pi i k n / N) along the last axis -- the DFT definition."""
    x = np.asarray(x, dtype=np.complex128)
    n = x.shape[-1]
    k = np.arange(n)
    m = np.exp(sign * 2j * np.pi * np.outer(k, k) / n)
    return x @ m.T


def dft2_naive(x, sign=-1):
    return dft_naive(dft_naive(x, sign).swapaxes(-1, -2), sign).swapaxes(-1, -2)


def conv_direct(psf, x):
    """(PSF * x)[n] = sum_{n'} psf[(n - n') mod M] x[n'] for n, n' in the unpadded field.

    Linear (non-periodic) convolution of the N^2 field with a PSF twice the field size
    (P:174), PSF origin at index [0][0], negative offsets wrapped to M - d (reading R2)."""
    ny, nx = x.shape
    my, mx = psf.shape
    out = np.zeros((ny, nx))
    for y in range(ny):
        for xx in range(nx):
            acc = 0.0
            for yp in range(ny):
                for xp in range(nx):
                    acc += psf[(y - yp) % my, (xx - xp) % mx] * x[yp, xp]
            out[y, xx] = acc
    return out


# =============================================================================
# Padding and the PSF spectrum  (Eq. 14; readings R2-R4)
# =============================================================================
def pad(x):
    """P: write the ny x nx image into [0:ny, 0:nx] of a (2ny) x (2nx) zero array (R2)."""
    ny, nx = x.shape
    p = np.zeros((2 * ny, 2 * nx), dtype=F64)
    p[:ny, :nx] = x
    return p


def crop(p):
    """P^dagger: slice out the region not padded."""
    my, mx = p.shape
    return p[: my // 2, : mx // 2]


def full_spectrum(w_half_c):
    """Half grid [My, nx+1] -> full grid [My, Mx] by Hermitian symmetry W[-k] = W[k] (R4)."""
    my, nxp = w_half_c.shape
    mx = 2 * (nxp - 1)
    w = np.empty((my, mx), dtype=F64)
    w[:, :nxp] = w_half_c
    ky = (-np.arange(my)) % my
    for kx in range(nxp, mx):
        w[:, kx] = w_half_c[ky, mx - kx]
    return w


def psf_from_weights(w_half_c):
    """psf[x] = sum_k W[k] exp(+2 pi i k.x / M): unnormalised inverse DFT of W (R3).
    Hence psf[0] = sum W ("PSF peak = sum of weights")."""
    w = full_spectrum(np.asarray(w_half_c, dtype=F64))
    return np.real(np.fft.ifft2(w)) * w.size


def psf_spectrum_from_psf(psf, tol=1e-5):
    """set_psf semantics (R4): W = DFT(psf)/M^2 must be real and >= 0 up to tol * max W.
    Returns (w_half [My, nx+1], ok)."""
    psf = np.asarray(psf, dtype=F64)
    my, mx = psf.shape
    w = np.fft.fft2(psf) / psf.size
    top = np.max(np.abs(w.real))
    ok = bool(np.max(np.abs(w.imag)) <= tol * top and np.min(w.real) >= -tol * top)
    return np.maximum(w.real, 0.0)[:, : mx // 2 + 1], ok


def psf_apply(w_half_c, x):
    """C x = P^dagger FFT^-1[ FFT[I^PSF] . FFT[P x] ]   (Eq. 14)

    with the physical normalisation of R3:
    xhat[k] = sum_x (P x)[x] e^{-2 pi i k.x/M},  (C x)[x] = sum_k W[k] xhat[k] e^{+2 pi i k.x/M}.
    numpy's irfft2 divides by My*Mx, so that factor is multiplied back."""
    w = np.asarray(w_half_c, dtype=F64)
    p = pad(np.asarray(x, dtype=F64))
    y = np.fft.irfft2(w * np.fft.rfft2(p), s=p.shape) * p.size
    return crop(y)


def psf_apply_full(w_half_c, x):
    """Same operator through the full complex spectrum (no Hermitian shortcut)."""
    w = full_spectrum(np.asarray(w_half_c, dtype=F64))
    p = pad(np.asarray(x, dtype=F64))
    return crop(np.real(np.fft.ifft2(w * np.fft.fft2(p))) * p.size)


def quadratic_form_spectral(w_half_c, x):
    """<x, C x> = sum_k W[k] |xhat[k]|^2 over the full M^2 grid (no inverse FFT, no crop)."""
    w = full_spectrum(np.asarray(w_half_c, dtype=F64))
    xh = np.fft.fft2(pad(np.asarray(x, dtype=F64)))
    return float(np.sum(w * (xh.real ** 2 + xh.imag ** 2)))


# =============================================================================
# Correlated field ("Gaussian processes ... exponentiated"; reading R6)
# =============================================================================
def hartley2(z):
    """H z [x] = sum_k z[k] cas(2 pi k.x / N), cas = cos + sin;  = Re F - Im F with
    F[x] = sum_k z[k] e^{-2 pi i k.x/N}.  Real, symmetric, H o H = ny nx * identity."""
    f = np.fft.fft2(np.asarray(z, dtype=F64))
    return f.real - f.imag


def log_sky(xi, amp, mu):
    """tau_f = mu_f + H[A_f . xi_f]   (R6)"""
    xi = np.asarray(xi, dtype=F64)
    return np.stack([F64(mu[f]) + hartley2(np.asarray(amp[f], F64) * xi[f]) for f in range(xi.shape[0])])


def channel_coeff(nfield, lognu):
    """d tau_c / d tau_f:  [nchan, nfield] = (1, ln(nu_c/nu_0))."""
    lognu = np.asarray(lognu, dtype=F64)
    c = np.ones((lognu.shape[0], nfield), dtype=F64)
    if nfield == 2:
        c[:, 1] = lognu
    return c


def sky(xi, amp, mu, lognu):
    """s_c = exp( tau_I + ln(nu_c/nu_0) tau_alpha )  (single field: s = exp(tau))."""
    tau = log_sky(xi, amp, mu)
    co = channel_coeff(tau.shape[0], lognu)
    return np.exp(np.einsum("cf,fyx->cyx", co, tau))


# =============================================================================
# Energy, gradient, metric  (Eq. 9 with N' = R' = C, Eq. 10; readings R1, R8)
# =============================================================================
def energy_of_sky(w_half, dirty, s):
    """E_lh = sum_c 1/2 <s_c, C_c s_c> - <j_c, s_c>."""
    e = 0.0
    for c in range(s.shape[0]):
        cs = psf_apply(w_half[c], s[c])
        e += 0.5 * float(np.sum(s[c] * cs)) - float(np.sum(np.asarray(dirty[c], F64) * s[c]))
    return e


def energy(w_half, dirty, amp, mu, lognu, xi, with_prior=True):
    s = sky(xi, amp, mu, lognu)
    e = energy_of_sky(w_half, dirty, s)
    if with_prior:
        e += 0.5 * float(np.sum(np.asarray(xi, F64) ** 2))
    return e


def jvp(amp, mu, lognu, xi, v, s=None):
    """J v = s_c . sum_f coeff[c,f] H[A_f v_f]   (J = diag(s) H diag(A), R8)."""
    if s is None:
        s = sky(xi, amp, mu, lognu)
    v = np.asarray(v, dtype=F64)
    lin = np.stack([hartley2(np.asarray(amp[f], F64) * v[f]) for f in range(v.shape[0])])
    co = channel_coeff(v.shape[0], lognu)
    return s * np.einsum("cf,fyx->cyx", co, lin)


def vjp(amp, lognu, s, w):
    """J^T w = A_f . H[ sum_c coeff[c,f] s_c w_c ]   (H^T = H)."""
    nfield = amp.shape[0]
    co = channel_coeff(nfield, lognu)
    acc = np.einsum("cf,cyx->fyx", co, s * w)
    return np.stack([np.asarray(amp[f], F64) * hartley2(acc[f]) for f in range(nfield)])


def energy_grad(w_half, dirty, amp, mu, lognu, xi, with_prior=True):
    """(E, grad):  grad E_lh = J^T (C s - j);  + xi with the standard-normal prior."""
    xi = np.asarray(xi, dtype=F64)
    s = sky(xi, amp, mu, lognu)
    res = np.stack([psf_apply(w_half[c], s[c]) - np.asarray(dirty[c], F64) for c in range(s.shape[0])])
    e = 0.0
    for c in range(s.shape[0]):
        cs = res[c] + np.asarray(dirty[c], F64)
        e += 0.5 * float(np.sum(s[c] * cs)) - float(np.sum(np.asarray(dirty[c], F64) * s[c]))
    g = vjp(amp, lognu, s, res)
    if with_prior:
        e += 0.5 * float(np.sum(xi ** 2))
        g = g + xi
    return e, g


def sky_metric_apply(w_half, s, x):
    """'L1 apply': y_c = s_c . C_c (s_c . x_c) -- likelihood Fisher metric in log-sky space."""
    s = np.asarray(s, dtype=F64)
    x = np.asarray(x, dtype=F64)
    return np.stack([s[c] * psf_apply(w_half[c], s[c] * x[c]) for c in range(s.shape[0])])


def metric_apply(w_half, amp, mu, lognu, xi, v, with_prior=True, s=None):
    """'L2 apply': M v = J^T C J v (+ v): the Fisher / Gauss-Newton metric MGVI uses,
    the Fisher metric of a Gaussian likelihood with mean C s and covariance C (Eq. 10)."""
    if s is None:
        s = sky(xi, amp, mu, lognu)
    jv = jvp(amp, mu, lognu, xi, v, s=s)
    cj = np.stack([psf_apply(w_half[c], jv[c]) for c in range(s.shape[0])])
    out = vjp(amp, lognu, s, cj)
    if with_prior:
        out = out + np.asarray(v, dtype=F64)
    return out


# =============================================================================
# The likelihood the paper ran: Eq. 9 with the fitted noise kernel (Eq. 15-18; reading R14)
# =============================================================================
def noise_kernel_from_psf(w_half_c, eps):
    """K = exp(xi_bar) + eps of Eq. 16-17 for one channel, [ny, nx].

    Eq. 17: xi_bar minimises || N'(I_delta) - FFT^-1[(exp xi + eps) FFT(I_delta)] ||^2 with I_delta a point source in
    the centre of the field and N' = R'+ eps 1 (Eq. 11), R' = the PSF convolution C (Eq. 13).  |FFT(I_delta)| = 1 at
    every mode, so by Parseval the objective is sum_k |K[k] - K*[k]|^2 with K* = FFT(N' I_delta) conj FFT(I_delta),
    and the minimiser over REAL K is Re K*; exp xi > 0 makes eps the floor (reading R14: K = max(Re K*, eps))."""
    w = np.asarray(w_half_c, dtype=F64)
    ny, nx = w.shape[0] // 2, w.shape[1] - 1
    delta = np.zeros((ny, nx), dtype=F64)
    delta[ny // 2, nx // 2] = 1.0
    n_delta = psf_apply(w, delta) + eps * delta                      # N'(I_delta), Eq. 11 with Eq. 13
    kstar = np.fft.fft2(n_delta) * np.conj(np.fft.fft2(delta))
    return np.maximum(kstar.real, eps)


def ninv_apply(kern, x):
    """N'^-1 x = FFT^-1[ K^-1 . FFT x ] on the UNPADDED grid, periodic boundary (Eq. 18)."""
    return np.real(np.fft.ifft2(np.fft.fft2(np.asarray(x, dtype=F64)) / np.asarray(kern, dtype=F64)))


def energy_grad_eq9(w_half, kern, dirty, amp, mu, lognu, xi, with_prior=True):
    """E = sum_c 1/2 (j_c - C_c s_c)^T N'_c^-1 (j_c - C_c s_c)  (Eq. 9 without the s-independent ln|2 pi N'|),
    grad = -J^T C N'^-1 (j - C s);  + 1/2 <xi,xi>, + xi with the standard-normal prior."""
    xi = np.asarray(xi, dtype=F64)
    s = sky(xi, amp, mu, lognu)
    e = 0.0
    back = np.empty_like(s)
    for c in range(s.shape[0]):
        r = np.asarray(dirty[c], F64) - psf_apply(w_half[c], s[c])
        u = ninv_apply(kern[c], r)
        e += 0.5 * float(np.sum(r * u))
        back[c] = -psf_apply(w_half[c], u)                           # C is symmetric
    g = vjp(amp, lognu, s, back)
    if with_prior:
        e += 0.5 * float(np.sum(xi ** 2))
        g = g + xi
    return e, g


def metric_apply_eq9(w_half, kern, amp, mu, lognu, xi, v, with_prior=True, s=None):
    """M v = J^T C N'^-1 C J v (+ v): Fisher metric of the Gaussian likelihood of Eq. 9 (mean C s, covariance N')."""
    if s is None:
        s = sky(xi, amp, mu, lognu)
    jv = jvp(amp, mu, lognu, xi, v, s=s)
    t = np.stack([psf_apply(w_half[c], ninv_apply(kern[c], psf_apply(w_half[c], jv[c]))) for c in range(s.shape[0])])
    out = vjp(amp, lognu, s, t)
    if with_prior:
        out = out + np.asarray(v, dtype=F64)
    return out


# =============================================================================
# MGVI: posterior samples and the sample-averaged KL ("Metric Gaussian Variational Inference"; reading R15)
# =============================================================================
def ninv_sqrt_apply(kern, x):
    """N'^-1/2 x = FFT^-1[ K^-1/2 . FFT x ] (periodic, as Eq. 18): the symmetric square root of N'^-1."""
    return np.real(np.fft.ifft2(np.fft.fft2(np.asarray(x, dtype=F64)) / np.sqrt(np.asarray(kern, dtype=F64))))


def sample_source_eq9(w_half, kern, amp, lognu, s, eta_xi, eta_d):
    """m = eta_xi + J^T C N'^-1/2 eta_d  with white eta_xi [nfield,ny,nx], eta_d [nchan,ny,nx]:  Cov m = 1 + J^T C N'^-1 C J = M,
    the metric of Eq. 9 at the position with sky s (MGVI draws its samples as M^-1 m, Knollmueller & Ensslin 2019)."""
    t = np.stack([psf_apply(w_half[c], ninv_sqrt_apply(kern[c], eta_d[c])) for c in range(s.shape[0])])
    return np.asarray(eta_xi, dtype=F64) + vjp(amp, lognu, s, t)


def draw_sample_eq9(w_half, kern, amp, mu, lognu, xi, eta_xi, eta_d, cg_iters):
    """One posterior sample around xi: sigma = M(xi)^-1 m by `cg_iters` CG iterations from 0 (Cov sigma -> M^-1)."""
    s = sky(xi, amp, mu, lognu)
    m = sample_source_eq9(w_half, kern, amp, lognu, s, eta_xi, eta_d)
    sol = cg(lambda v: metric_apply_eq9(w_half, kern, amp, mu, lognu, xi, v, True, s=s), m, max_iter=cg_iters)
    return sol["x"], m


def kl_energy_grad_eq9(w_half, kern, dirty, amp, mu, lognu, xi, samples, mirrored=True):
    """Sample-averaged KL and its gradient: mean over the positions xi + sigma_i (and xi - sigma_i if mirrored) of
    E_tot and grad E_tot (Eq. 9 likelihood + standard-normal prior)."""
    xi = np.asarray(xi, dtype=F64)
    pos = [xi + np.asarray(sg, F64) for sg in samples] + ([xi - np.asarray(sg, F64) for sg in samples] if mirrored else [])
    e, g = 0.0, np.zeros_like(xi)
    for q in pos:
        ei, gi = energy_grad_eq9(w_half, kern, dirty, amp, mu, lognu, q, True)
        e += ei
        g += gi
    return e / len(pos), g / len(pos)


def kl_metric_apply_eq9(w_half, kern, amp, mu, lognu, xi, samples, v, mirrored=True):
    """Sample-averaged metric: mean over the same positions of M(xi +- sigma_i) v."""
    xi = np.asarray(xi, dtype=F64)
    pos = [xi + np.asarray(sg, F64) for sg in samples] + ([xi - np.asarray(sg, F64) for sg in samples] if mirrored else [])
    out = np.zeros_like(np.asarray(v, dtype=F64))
    for q in pos:
        out += metric_apply_eq9(w_half, kern, amp, mu, lognu, q, v, True)
    return out / len(pos)


# =============================================================================
# Major cycle with the exact response on a list of uv points (Eq. 1 coplanar, Alg. 1, Eq. 20-22; R16)
# =============================================================================
def exact_response(uv, x, my, mx):
    """R x: V_k = sum_pixels x[y][x] exp(-2 pi i (u_k x / Mx + v_k y / My)), (u, v) in cell units of the padded grid,
    NOT rounded to cells (Eq. 1 for a coplanar array, unit primary beam) -- the direct sum, O(nvis npix)."""
    x = np.asarray(x, dtype=F64)
    ny, nx = x.shape
    uv = np.asarray(uv, dtype=F64)
    ex = np.exp(-2j * np.pi * np.outer(uv[:, 0], np.arange(nx)) / mx)      # [nvis, nx]
    ey = np.exp(-2j * np.pi * np.outer(uv[:, 1], np.arange(ny)) / my)      # [nvis, ny]
    return np.einsum("ky,yx,kx->k", ey, x, ex)


def exact_adjoint(uv, wgt, vis, ny, nx, my, mx):
    """R^dagger N^-1 V with every visibility and its conjugate (the convention of the weight grid, R5):
    image[y][x] = sum_k 2 w_k Re( V_k exp(+2 pi i (u_k x / Mx + v_k y / My)) )."""
    uv = np.asarray(uv, dtype=F64)
    ex = np.exp(2j * np.pi * np.outer(uv[:, 0], np.arange(nx)) / mx)
    ey = np.exp(2j * np.pi * np.outer(uv[:, 1], np.arange(ny)) / my)
    return 2.0 * np.real(np.einsum("k,ky,kx->yx", np.asarray(wgt, F64) * np.asarray(vis, np.complex128), ey, ex))


def major_cycle_residual(uv, wgt, dirty_full, sky_i, my, mx):
    """d_{i+1} = I^D - R^dagger N^-1 R I_i with the exact response (Eq. 20, 22)."""
    ny, nx = np.asarray(sky_i).shape
    return np.asarray(dirty_full, F64) - exact_adjoint(uv, wgt, exact_response(uv, sky_i, my, mx), ny, nx, my, mx)


# =============================================================================
# Conjugate gradient (paper silent; reading R9: textbook Hestenes-Stiefel)
# =============================================================================
def cg_step(apply, x, r, p, rr):
    """One CG iteration from the state (x, r, p, rr=<r,r>); returns the new state and q, alpha, beta."""
    q = apply(p)
    pq = float(np.sum(p * q))
    alpha = rr / pq
    x1 = x + alpha * p
    r1 = r - alpha * q
    rr1 = float(np.sum(r1 * r1))
    beta = rr1 / rr
    p1 = r1 + beta * p
    return dict(x=x1, r=r1, p=p1, rr=rr1, q=q, pq=pq, alpha=alpha, beta=beta)


def cg(apply, b, x0=None, max_iter=20, rtol=0.0, keep=False):
    """x <- CG(M, b).  r0 = b - M x0, p0 = r0; stop at max_iter or ||r|| <= rtol ||b||.
    Returns dict(x, iters, res=[||r_0||..||r_k||], xs=[x_1..] if keep, phi=[phi(x_k)])."""
    b = np.asarray(b, dtype=F64)
    x = np.zeros_like(b) if x0 is None else np.asarray(x0, dtype=F64).copy()
    r = b - apply(x) if x0 is not None else b.copy()
    p = r.copy()
    rr = float(np.sum(r * r))
    bnorm = float(np.sqrt(np.sum(b * b)))
    res = [np.sqrt(rr)]
    xs, states = [], []
    it = 0
    while it < max_iter and not (rtol > 0 and np.sqrt(rr) <= rtol * bnorm):
        st = cg_step(apply, x, r, p, rr)
        if st["pq"] <= 0:
            raise FloatingPointError("CG breakdown: <p, M p> <= 0")
        x, r, p, rr = st["x"], st["r"], st["p"], st["rr"]
        it += 1
        res.append(np.sqrt(rr))
        if keep:
            xs.append(x.copy())
            states.append((st["alpha"], st["beta"]))
    return dict(x=x, iters=it, res=np.array(res), xs=xs, coeffs=states)


def cg_fp32_envelope(apply, b, max_iter=20, seed=1234):
    """fp64 CG whose operator output is multiplied by (1 + 2^-24 U(-1,1)) at every apply:
    the drift any fp32 operator shows in free-running CG (SURVEY 8(c)-9 finding ii).
    Returns rel-L2 distance of the perturbed iterates x_k from the unperturbed ones, k=1..max_iter."""
    rng = np.random.default_rng(seed)

    def noisy(v):
        o = apply(v)
        return o * (1.0 + 2.0 ** -24 * rng.uniform(-1.0, 1.0, o.shape))

    a = cg(apply, b, max_iter=max_iter, keep=True)
    n = cg(noisy, b, max_iter=max_iter, keep=True)
    return np.array([np.linalg.norm(xn - xa) / np.linalg.norm(xa) for xa, xn in zip(a["xs"], n["xs"])])


def newton_cg_step(w_half, dirty, amp, mu, lognu, xi, cg_iters=50):
    """'Outer KL step' with zero samples (reading R10): delta = CG(M(xi), -grad, cg_iters);
    xi <- xi + delta, halving delta up to 4 times while E_tot does not decrease."""
    xi = np.asarray(xi, dtype=F64)
    e0, g = energy_grad(w_half, dirty, amp, mu, lognu, xi, True)
    s = sky(xi, amp, mu, lognu)
    sol = cg(lambda v: metric_apply(w_half, amp, mu, lognu, xi, v, True, s=s), -g, max_iter=cg_iters)
    d = sol["x"]
    for _ in range(5):
        e1 = energy(w_half, dirty, amp, mu, lognu, xi + d, True)
        if e1 < e0:
            break
        d = 0.5 * d
    return xi + d, e0, e1


# =============================================================================
# Image sizes that are not powers of two (3600^2) by embedding -- DESIGN.md reading R19
# =============================================================================
# The convolution of Eq. 14 is a LINEAR convolution of the ny_i x nx_i image with the (2 ny_i) x (2 nx_i) PSF; any padded
# grid of at least twice the image size computes it exactly.  The correlated field lives on the embedding grid
# (ny x nx, the next power of two); the sky is its crop to the image, everything outside is not part of the model:
#   s = crop(exp(mu + H[A xi])),   E = 1/2 <s, C s> - <j, s> (+ 1/2 <xi, xi>),   C on the ny_i x nx_i image.
def embed(x, ny, nx):
    out = np.zeros(x.shape[:-2] + (ny, nx))
    out[..., :x.shape[-2], :x.shape[-1]] = x
    return out


def energy_grad_embedded(w_half_img, dirty_img, amp, mu, xi, with_prior=True):
    """w_half_img [2 ny_i, nx_i + 1], dirty_img [ny_i, nx_i]: the image-sized problem; amp, xi [ny, nx]: the field on the
    embedding grid.  Returns E and dE/dxi [ny, nx]."""
    xi = np.asarray(xi, dtype=F64)
    ny, nx = xi.shape
    nyi, nxi = dirty_img.shape
    s_full = np.exp(mu + hartley2(np.asarray(amp, F64) * xi))
    s = s_full[:nyi, :nxi]
    cs = psf_apply(w_half_img, s)
    e = 0.5 * np.sum(s * cs) - np.sum(np.asarray(dirty_img, F64) * s)
    g = np.asarray(amp, F64) * hartley2(embed(s * (cs - dirty_img), ny, nx))
    if with_prior:
        e += 0.5 * np.sum(xi * xi)
        g = g + xi
    return float(e), g


def metric_apply_embedded(w_half_img, nyi, nxi, amp, mu, xi, v, with_prior=True):
    xi = np.asarray(xi, dtype=F64)
    ny, nx = xi.shape
    s = np.exp(mu + hartley2(np.asarray(amp, F64) * xi))[:nyi, :nxi]
    jv = s * hartley2(np.asarray(amp, F64) * np.asarray(v, F64))[:nyi, :nxi]
    out = np.asarray(amp, F64) * hartley2(embed(s * psf_apply(w_half_img, jv), ny, nx))
    return out + v if with_prior else out
