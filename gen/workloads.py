"""Seeded synthetic workloads shaped like the paper's VLA / MeerKAT cases.

This module only *draws inputs* (uv coverage -> weight grid W, amplitude spectrum
A, a truth sky, a dirty image j).  It is consumed by the tests, the oracle runs and
the CUDA runs alike and deliberately imports neither `oracle/` nor the CUDA
package.  The few FFTs used to synthesise a statistically consistent dirty image
are direct calls of the numpy library routine.

Stand-in statement: these inputs replace the paper's VLA Cygnus A (P:285-292,
Tab. 1) and MeerKAT ESO 137-006 (Tab. 2) data sets, which are not
available; shapes follow BASELINE.json `configs` and SURVEY.md section 8(d).
`P:<n>` = line n of /root/reference/PAPER.md.

Recipe (fixed draw order from numpy.random.default_rng(seed):
uv -> xi* -> point sources -> noise), everything in float64 and rounded ONCE to
float32 at the end:

  * uv points in cell units of the padded grid (My, Mx) = (2 ny, 2 nx); a point is
    kept iff |u| < Mx/2 - 1/2 and |v| < My/2 - 1/2; it lands in cell
    (rint(v) mod My, rint(u) mod Mx); natural weighting W0[cell] += 1;
    W = W0 + flip(W0), flip(W0)[k] = W0[-k mod M] (a visibility and its conjugate).
  * amplitude spectrum A[k] = sigma_f a(|k|) / sqrt(sum_{k!=0} a^2), A[0] = sigma_0,
    a^2 = P(k), |k| from signed wrapped indices -> A even: A[-k] = A[k].
  * truth s* = exp(H[A xi*]) (+ envelope) + point sources, H = 2-D Hartley transform.
  * dirty j = C s* + n', Cov(n') = C, std(n') = sigma_rel * max(C s*): achieved by
    scaling the integer grid with one scalar w0 (Eq. 8-10).
"""
from __future__ import annotations

import dataclasses
import numpy as np


@dataclasses.dataclass
class Workload:
    name: str
    ny: int
    nx: int
    nchan: int
    nfield: int
    w_counts: np.ndarray   # [nchan, My, nx+1] float64 integer-valued half grid (before w0)
    w0: float
    w_half: np.ndarray     # [nchan, My, nx+1] float32 = fp32(w0 * w_counts)
    dirty: np.ndarray      # [nchan, ny, nx]   float32
    amp: np.ndarray        # [nfield, ny, nx]  float32
    mu: np.ndarray         # [nfield]          float32
    lognu: np.ndarray      # [nchan]           float32  ln(nu_c/nu_0)
    xi_true: np.ndarray    # [nfield, ny, nx]  float32  latent excitations of the diffuse truth
    sky_true: np.ndarray   # [nchan, ny, nx]   float32
    seed: int = 0

    @property
    def my(self):
        return 2 * self.ny

    @property
    def mx(self):
        return 2 * self.nx


# ----------------------------------------------------------------------------- uv sampling
def uv_gaussian(rng, npts, my, mx, sigma_frac):
    u = rng.normal(0.0, sigma_frac * mx, npts)
    v = rng.normal(0.0, sigma_frac * my, npts)
    return u, v


def uv_vla_like(rng, npts, my, mx, rmin=0.004, rmax=0.45):
    """'27-antenna-style' radial density with a central hole (config 2)."""
    r = rmin + (rmax - rmin) * rng.uniform(0.0, 1.0, npts) ** 2
    th = rng.uniform(0.0, 2.0 * np.pi, npts)
    return r * mx * np.cos(th), r * my * np.sin(th)


def uv_mixture(rng, npts, my, mx, s_core=0.05, s_tail=0.4, frac_core=0.7):
    """MeerKAT-like dense core + long-baseline tail (configs 3-5)."""
    core = rng.uniform(0.0, 1.0, npts) < frac_core
    sig = np.where(core, s_core, s_tail)
    u = rng.normal(0.0, 1.0, npts) * sig * mx
    v = rng.normal(0.0, 1.0, npts) * sig * my
    return u, v


def grid_weights(u, v, my, mx):
    """uv points -> Hermitian-symmetrised integer count grid W [My, Mx] (float64)."""
    keep = (np.abs(u) < mx / 2 - 0.5) & (np.abs(v) < my / 2 - 0.5)
    iu = np.rint(u[keep]).astype(np.int64) % mx
    iv = np.rint(v[keep]).astype(np.int64) % my
    w0 = np.bincount(iv * mx + iu, minlength=my * mx).astype(np.float64).reshape(my, mx)
    flip = np.roll(w0[::-1, ::-1], (1, 1), axis=(0, 1))      # flip[k] = w0[-k mod M]
    return w0 + flip


# ----------------------------------------------------------------------------- prior spectrum
def k_radius(ny, nx):
    n = max(ny, nx)
    ky = np.fft.fftfreq(ny, d=1.0 / ny) * (n / ny)           # signed wrapped index
    kx = np.fft.fftfreq(nx, d=1.0 / nx) * (n / nx)
    return np.sqrt(ky[:, None] ** 2 + kx[None, :] ** 2)


def amplitude_spectrum(ny, nx, kind, sigma_f, sigma_0=0.1, k0=4.0):
    """A[k] (float64), even in k.  kind: 'lorentz4' P=(1+k/k0)^-4 | 'pow3.5' P=k^-3.5."""
    k = k_radius(ny, nx)
    with np.errstate(divide="ignore"):
        if kind == "lorentz4":
            p = (1.0 + k / k0) ** -4.0
        elif kind == "pow3.5":
            p = np.where(k > 0, k, 1.0) ** -3.5
        else:
            raise ValueError(kind)
    p[0, 0] = 0.0
    a = np.sqrt(p)
    a *= sigma_f / np.sqrt(np.sum(a * a))
    a[0, 0] = sigma_0
    return a


def _hartley2(z):
    f = np.fft.fft2(z)
    return f.real - f.imag


# ----------------------------------------------------------------------------- data synthesis
def _conv_counts(w_half_counts, s, ny, nx):
    my, mx = 2 * ny, 2 * nx
    p = np.zeros((my, mx))
    p[:ny, :nx] = s
    return (np.fft.irfft2(w_half_counts * np.fft.rfft2(p), s=(my, mx)) * (my * mx))[:ny, :nx]


def _noise_counts(w_half_counts, eta, ny, nx):
    my, mx = 2 * ny, 2 * nx
    return (np.fft.irfft2(np.sqrt(w_half_counts) * np.fft.rfft2(eta), s=(my, mx))
            * np.sqrt(my * mx))[:ny, :nx]


def build(name, ny, nx, *, uv_kind, npts, spectrum, sigma_f, points, sigma_rel=1e-3,
          envelope=None, nchan=1, seed=0, sigma_0=0.1):
    """Generic builder; `make_config` maps BASELINE.json's five configs onto it.

    points = (count, mode): mode 'lognormal10' (flux = exp(N(ln(10 median), 1))),
    'x100' (100 x median), 'powerlaw' (dN/dS ~ S^-1.8 on [Smin, 1e3 Smin], Smin = median).
    """
    rng = np.random.default_rng(seed)
    my, mx = 2 * ny, 2 * nx
    nfield = 2 if nchan > 1 else 1
    # 1. uv -> W ---------------------------------------------------------------
    if uv_kind == "gauss":
        u, v = uv_gaussian(rng, npts, my, mx, 0.25)
    elif uv_kind == "vla":
        u, v = uv_vla_like(rng, npts, my, mx)
    elif uv_kind == "mix":
        u, v = uv_mixture(rng, npts, my, mx)
    else:
        raise ValueError(uv_kind)
    if nchan == 1:
        lognu = np.zeros(1)
        wc = grid_weights(u, v, my, mx)[None, :, : nx + 1]
    else:
        nu = 0.9 + 0.8 * np.arange(nchan) / (nchan - 1)        # GHz
        nu0 = 1.3
        lognu = np.log(nu / nu0)
        wc = np.stack([grid_weights(u * f, v * f, my, mx)[:, : nx + 1] for f in nu / nu0])
    # 2. prior + truth -----------------------------------------------------------
    amp = np.empty((nfield, ny, nx))
    mu = np.zeros(nfield)
    amp[0] = amplitude_spectrum(ny, nx, spectrum, sigma_f, sigma_0)
    if nfield == 2:
        amp[1] = amplitude_spectrum(ny, nx, spectrum, 0.2, sigma_0)
        mu[1] = -0.7
    xi = rng.normal(0.0, 1.0, (nfield, ny, nx))
    tau = np.stack([mu[f] + _hartley2(amp[f] * xi[f]) for f in range(nfield)])
    if nfield == 1:
        sky = np.exp(tau[0])[None]
    else:
        sky = np.exp(tau[0][None] + lognu[:, None, None] * tau[1][None])
    if envelope == "two_lobe":
        yy, xx = np.mgrid[0:ny, 0:nx]
        sg = max(ny, nx) / 10.0
        env = sum(np.exp(-0.5 * (((yy - ny / 2) / sg) ** 2 + ((xx - cx) / sg) ** 2))
                  for cx in (nx / 2 - nx / 5, nx / 2 + nx / 5))
        sky = sky * env[None]
    # 3. point sources -------------------------------------------------------------
    npnt, mode = points
    med = float(np.median(sky[0]))
    py = rng.integers(0, ny, npnt)
    px = rng.integers(0, nx, npnt)
    if mode == "lognormal10":
        flux = np.exp(rng.normal(np.log(10.0 * med), 1.0, npnt))
    elif mode == "x100":
        flux = np.full(npnt, 100.0 * med) * (1.0 + 0.0 * rng.uniform(size=npnt))
    elif mode == "powerlaw":
        q = rng.uniform(0.0, 1.0, npnt)
        a = 1.0 - 1.8
        smin, smax = med, 1e3 * med
        flux = (smin ** a + q * (smax ** a - smin ** a)) ** (1.0 / a)
    else:
        raise ValueError(mode)
    for c in range(nchan):
        spec = np.exp(-0.7 * lognu[c])
        np.add.at(sky[c], (py, px), flux * spec)
    # 4. dirty image ----------------------------------------------------------------
    sig = [_conv_counts(wc[c], sky[c], ny, nx) for c in range(nchan)]
    peak = max(float(np.max(s)) for s in sig)
    w0 = float(np.mean(np.sum(_full_sum(wc), axis=0))) / (sigma_rel * peak) ** 2
    dirty = np.empty((nchan, ny, nx))
    for c in range(nchan):
        eta = rng.normal(0.0, 1.0, (my, mx))
        dirty[c] = w0 * sig[c] + np.sqrt(w0) * _noise_counts(wc[c], eta, ny, nx)
    f32 = np.float32
    return Workload(name=name, ny=ny, nx=nx, nchan=nchan, nfield=nfield, w_counts=wc, w0=w0,
                    w_half=(w0 * wc).astype(f32), dirty=dirty.astype(f32), amp=amp.astype(f32),
                    mu=mu.astype(f32), lognu=lognu.astype(f32), xi_true=xi.astype(f32),
                    sky_true=sky.astype(f32), seed=seed)


def _full_sum(wc):
    """Sum over the FULL grid of each channel's half grid [nchan, My, nx+1] -> [1, nchan]."""
    nxp = wc.shape[-1]
    inner = wc[..., 1: nxp - 1].sum(axis=(-1, -2))
    edge = wc[..., 0].sum(axis=-1) + wc[..., nxp - 1].sum(axis=-1)
    return (2.0 * inner + edge)[None]


_CONFIGS = {
    1: dict(n=128, uv_kind="gauss", npts=20_000, spectrum="lorentz4", sigma_f=1.0,
            points=(20, "lognormal10")),
    2: dict(n=512, uv_kind="vla", npts=200_000, spectrum="lorentz4", sigma_f=2.0,
            points=(5, "x100"), envelope="two_lobe"),
    3: dict(n=2048, uv_kind="mix", npts=5_000_000, spectrum="pow3.5", sigma_f=1.0,
            points=(200, "lognormal10")),
    4: dict(n=4096, uv_kind="mix", npts=20_000_000, spectrum="pow3.5", sigma_f=1.0,
            points=(1000, "powerlaw")),
    5: dict(n=1024, uv_kind="mix", npts=1_000_000, spectrum="pow3.5", sigma_f=1.0,
            points=(100, "lognormal10"), nchan=16),
}


def make_config(i, seed=0, n=None, ny=None, nx=None, sigma_rel=1e-3, nchan=None, npts=None):
    """BASELINE.json config i (1..5).  n / ny,nx / nchan / npts override the size so tests can
    run the same recipe at a size the oracle finishes in seconds (uv counts scale with area)."""
    c = dict(_CONFIGS[i])
    n0 = c.pop("n")
    ny = ny or n or n0
    nx = nx or n or n0
    if npts is None:
        npts = max(2000, int(c["npts"] * (ny * nx) / float(n0 * n0)))
    c["npts"] = npts
    if nchan is not None:
        c["nchan"] = nchan
    name = f"config{i}_{ny}x{nx}" + (f"x{c['nchan']}ch" if c.get("nchan", 1) > 1 else "")
    return build(name, ny, nx, sigma_rel=sigma_rel, seed=seed, **c)
