"""Several Gaussian processes on patches (Fig. 10; reading R20), composed from C-ABI calls.

    s = sum_k insert_k( exp(mu_k + H_k[A_k xi_k]) ),    E = E_lh(s) + 1/2 sum_k <xi_k, xi_k>

`field` is the Context of the full field (PSF, dirty image, likelihood mode); every component has a Context of its own
on its own power-of-two grid with its amplitude set, and a position (y0, x0) in the field.  This module holds no arithmetic
of the method: sums, products and transforms all happen inside the library (frs_sky_forward, frs_patch_insert_add,
frs_sky_energy_grad, frs_patch_crop, frs_latent_vjp / _jvp, frs_psf_apply, frs_ninv_apply); Python only orders the calls
and owns the device buffers.
"""
from __future__ import annotations


class PatchModel:
    def __init__(self, field, components):
        """components: list of (ctx_k, y0_k, x0_k); ctx_k.set_amplitude(...) already called."""
        import torch
        self.torch, self.field, self.comps = torch, field, list(components)
        dev = field.device
        self.sky = torch.zeros(1, field.ny, field.nx, device=dev)
        self.gsky = torch.zeros_like(self.sky)
        self.tmp = torch.zeros_like(self.sky)
        self.parts = [torch.zeros(1, c.ny, c.nx, device=dev) for c, _, _ in self.comps]
        self.crops = [torch.zeros(1, c.ny, c.nx, device=dev) for c, _, _ in self.comps]
        self.mode = 0

    def set_likelihood(self, mode):
        self.field.set_likelihood(mode)
        self.mode = int(mode)

    def _forward(self, xis):
        self.sky.zero_()
        for (c, y0, x0), xi, part in zip(self.comps, xis, self.parts):
            c.sky_forward(xi, part)                              # sets the component's position
            self.field.patch_insert_add(part, y0, x0, self.sky)

    def sky_forward(self, xis):
        self._forward(xis)
        return self.sky

    def energy_grad(self, xis, grads, with_prior=True):
        """E (host float) and dE/dxi_k into grads[k]."""
        self._forward(xis)
        e = self.field.sky_energy_grad(self.sky, self.gsky)
        for (c, y0, x0), xi, g, crop in zip(self.comps, xis, grads, self.crops):
            self.field.patch_crop(self.gsky, y0, x0, crop)
            c.latent_vjp(crop, g, add=xi if with_prior else None)
            if with_prior:
                e += 0.5 * c.dot(xi, xi)
        return e

    def metric_apply(self, vs, outs, with_prior=True):
        """Fisher metric at the position of the last energy_grad / sky_forward."""
        self.tmp.zero_()
        for (c, y0, x0), v, crop in zip(self.comps, vs, self.crops):
            c.latent_jvp(v, crop)
            self.field.patch_insert_add(crop, y0, x0, self.tmp)
        self.field.psf_apply(self.tmp, self.gsky)                # C J v
        if self.mode == 1:
            self.field.ninv_apply(self.gsky, self.tmp)           # N'^-1 C J v
            self.field.psf_apply(self.tmp, self.gsky)            # C N'^-1 C J v
        for (c, y0, x0), v, o, crop in zip(self.comps, vs, outs, self.crops):
            self.field.patch_crop(self.gsky, y0, x0, crop)
            c.latent_vjp(crop, o, add=v if with_prior else None)
        return outs
