"""ctypes binding of include/frs.h -- argument marshalling only (same names as the C ABI)."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libfrs.so")

FRS_OK, FRS_EINVAL, FRS_ESTATE, FRS_ENOTPSD, FRS_ECUDA, FRS_EBREAKDOWN = 0, -1, -2, -3, -4, -5
_CODES = {-1: "FRS_EINVAL", -2: "FRS_ESTATE", -3: "FRS_ENOTPSD", -4: "FRS_ECUDA", -5: "FRS_EBREAKDOWN"}

_vp, _i, _f, _d = C.c_void_p, C.c_int, C.c_float, C.c_double
# name -> (restype, argtypes): every symbol include/frs.h declares
EXPORTS = {
    "frs_create": (_i, [_i, _i, _i, _i, _vp, C.POINTER(_vp)]),
    "frs_destroy": (None, [_vp]),
    "frs_last_error": (C.c_char_p, [_vp]),
    "frs_version": (C.c_char_p, []),
    "frs_set_psf": (_i, [_vp, _vp]),
    "frs_set_psf_weights": (_i, [_vp, _vp]),
    "frs_set_dirty": (_i, [_vp, _vp]),
    "frs_set_amplitude": (_i, [_vp, _i, _vp, C.POINTER(_f)]),
    "frs_set_channel_lognu": (_i, [_vp, C.POINTER(_f)]),
    "frs_sky_forward": (_i, [_vp, _vp, _vp]),
    "frs_psf_apply": (_i, [_vp, _vp, _vp]),
    "frs_sky_metric_apply": (_i, [_vp, _vp, _vp]),
    "frs_set_sky": (_i, [_vp, _vp]),
    "frs_energy_grad": (_i, [_vp, _vp, _i, _vp, C.POINTER(_d), _vp]),
    "frs_metric_apply": (_i, [_vp, _vp, _i, _vp]),
    "frs_cg_solve": (_i, [_vp, _vp, _vp, _i, _f, _i, C.POINTER(_i), C.POINTER(_d), _vp]),
    "frs_cg_read_state": (_i, [_vp, _vp, _vp, _vp, C.POINTER(_d)]),
    "frs_cg_load": (_i, [_vp, _vp, _vp, _d]),
    "frs_cg_step": (_i, [_vp, _vp, _i]),
    "frs_cg_step_begin": (_i, [_vp, C.POINTER(_vp)]),
    "frs_cg_step_end": (_i, [_vp, _vp, _i]),
    "frs_set_noise_kernel": (_i, [_vp, _f]),
    "frs_set_noise_kernel_array": (_i, [_vp, _vp]),
    "frs_get_noise_kernel": (_i, [_vp, _vp]),
    "frs_ninv_apply": (_i, [_vp, _vp, _vp]),
    "frs_set_likelihood": (_i, [_vp, _i]),
    "frs_set_cuda_graphs": (_i, [_vp, _i]),
    "frs_set_fused_passes": (_i, [_vp, _i]),
    "frs_sky_energy_grad": (_i, [_vp, _vp, C.POINTER(_d), _vp]),
    "frs_dot": (_i, [_vp, _vp, _vp, C.c_longlong, C.POINTER(_d)]),
    "frs_dot_noalloc": (_i, [_i, _vp, _vp, _vp, C.c_longlong, _vp]),
    "frs_dot_noalloc_last_error": (C.c_char_p, []),
    "frs_latent_jvp": (_i, [_vp, _vp, _vp]),
    "frs_latent_vjp": (_i, [_vp, _vp, _vp, _vp]),
    "frs_patch_insert_add": (_i, [_vp, _vp, _i, _i, _i, _i, _vp]),
    "frs_patch_crop": (_i, [_vp, _vp, _i, _i, _i, _i, _vp]),
    "frs_set_psf_embedded": (_i, [_vp, _vp, _i, _i]),
    "frs_set_field_of_view": (_i, [_vp, _i, _i]),
    "frs_amp_model_size": (_i, [_i, _i, C.POINTER(_i), C.POINTER(_i)]),
    "frs_set_amplitude_model": (_i, [_vp, C.POINTER(_f)]),
    "frs_amplitude_forward": (_i, [_vp, _vp, _vp]),
    "frs_amplitude_jvp": (_i, [_vp, _vp, _vp]),
    "frs_amplitude_vjp": (_i, [_vp, _vp, _vp]),
    "frs_set_point_sources": (_i, [_vp, _i, C.POINTER(_i), _f, _f]),
    "frs_energy_grad_joint": (_i, [_vp, _vp, _vp, _i, C.POINTER(_d), _vp, _vp]),
    "frs_metric_apply_joint": (_i, [_vp, _vp, _vp, _i, _vp, _vp]),
    "frs_draw_sample": (_i, [_vp, _vp, _vp, _i, _f, _vp, C.POINTER(_i)]),
    "frs_kl_energy_grad": (_i, [_vp, _vp, _vp, _i, _i, _vp, C.POINTER(_d), _vp]),
    "frs_kl_metric_apply": (_i, [_vp, _vp, _vp, _i, _i, _vp, _vp]),
    "frs_exact_response": (_i, [_vp, _vp, _i, _vp, _vp]),
    "frs_exact_adjoint": (_i, [_vp, _vp, _vp, _i, _vp, _vp]),
    "frs_major_cycle_residual": (_i, [_vp, _vp, _vp, _i, _vp, _vp, _vp]),
    "frs_sky_metric_apply_host": (_i, [_vp, _vp, _vp]),
    "frs_psf_apply_host": (_i, [_vp, _vp, _vp]),
    "frs_sky_metric_apply_host_batch": (_i, [_vp, _i, C.POINTER(_vp), C.POINTER(_vp)]),
    "frs_launch_count": (C.c_longlong, [_vp]),
    "frs_profile_enable": (_i, [_vp, _i]),
    "frs_debug_check_guards": (_i, [_vp, C.POINTER(_i)]),
    "frs_profile_read": (_i, [_vp, C.POINTER(_d), C.POINTER(C.c_longlong)]),
    "frs_selftest_fft_host": (_i, [_i, _i, _vp, _vp]),
    "frs_selftest_tma_geometry": (_i, [_i, _i, C.POINTER(_i)]),
    "frs_selftest_dif_host": (_i, [_i, _i, _vp, _vp]),
    "frs_selftest_dif_exchange": (_i, [_i, C.POINTER(_i)]),
    "frs_selftest_tcgen05_stage": (_i, [_i, _i, _i, C.POINTER(_d)]),
}

_lib = None


class FrsError(RuntimeError):
    def __init__(self, code, msg=""):
        self.code = code
        super().__init__(f"{_CODES.get(code, code)}: {msg}")


def load_library(path=LIB_PATH):
    """dlopen libfrs.so and declare every prototype.  Raises if the library is not built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise FileNotFoundError(f"{path} not built -- run `python -m paper_2406_09144_b200.build` "
                                "(there is no CPU fallback)")
    lib_ = C.CDLL(path)
    for name, (res, args) in EXPORTS.items():
        fn = getattr(lib_, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib_
    return lib_


def lib():
    return load_library()


def selftest_fft_host(x, inverse=False):
    """CPU replay of the kernels' FFT stage logic (complex64 [n])."""
    x = np.ascontiguousarray(x, dtype=np.complex64)
    out = np.empty_like(x)
    rc = lib().frs_selftest_fft_host(x.shape[0], int(inverse), x.ctypes.data, out.ctypes.data)
    if rc != 0:
        raise FrsError(rc, "selftest")
    return out


def selftest_dif_host(x, inverse=False):
    """CPU replay of the DIF/DIT core of the column convolution (complex64 [n], natural order both sides)."""
    x = np.ascontiguousarray(x, dtype=np.complex64)
    out = np.empty_like(x)
    rc = lib().frs_selftest_dif_host(x.shape[0], int(inverse), x.ctypes.data, out.ctypes.data)
    if rc != 0:
        raise FrsError(rc, "selftest_dif_host")
    return out


def selftest_dif_exchange(n):
    """(worst bank-conflict degree, unordered hazards, out-of-range slots, slots used, slots allocated,
    frequency-map defects) of the DIF core's exchange pattern."""
    out = (_i * 6)()
    rc = lib().frs_selftest_dif_exchange(int(n), out)
    if rc != 0:
        raise FrsError(rc, "selftest_dif_exchange")
    return tuple(int(v) for v in out)


def selftest_tcgen05_stage(n_out=64, mmas_per_commit=24, iters=2000):
    """SM cycles per tcgen05.mma kind::tf32 (M = 128, K = 8, N = n_out) -- the tensor-core measurement of DESIGN.md section 5."""
    out = _d(0.0)
    rc = lib().frs_selftest_tcgen05_stage(int(n_out), int(mmas_per_commit), int(iters), C.byref(out))
    if rc != 0:
        raise FrsError(rc, "selftest_tcgen05_stage")
    return out.value


def _ptr(t, dtype=None, numel=None, name="tensor"):
    if t is None:
        return None
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous CUDA tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"{name}: expected dtype {dtype}, got {t.dtype}")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{name}: expected {numel} elements, got {t.numel()}")
    return t.data_ptr()


def selftest_tma_geometry(nf, rows):
    """(box_bins, bin_copies, box_pairs, col_copies, xbuf_slots, rows_use_tma) of csrc/tmap.h."""
    out = (_i * 6)()
    rc = lib().frs_selftest_tma_geometry(int(nf), int(rows), out)
    if rc != 0:
        raise FrsError(rc, "selftest_tma_geometry")
    return tuple(int(v) for v in out)


FRS_DOT_NOALLOC_MAX_N = 1 << 28


def dot_noalloc(a, b, d_out, stream=None):
    """frs_dot_noalloc: d_out[0] = <a, b> in fp64 for callers that must not allocate on the device (a framework allocator
    owns the GPU's memory, or a cudaMalloc would stall the other streams of a latency-bound loop).  Needs no Context; the
    library's only scratch is a fixed array in its device code, shared by every call on the device -- so calls that can
    overlap on the GPU race.  a, b: CUDA float32 tensors of equal length (a multiple of 4, at most FRS_DOT_NOALLOC_MAX_N);
    d_out: a CUDA float64 tensor of one element on the same device, written on `stream` (default: torch's current
    stream) without synchronising.  Marshalling only."""
    import torch
    pa, pb = _ptr(a, torch.float32, None, "a"), _ptr(b, torch.float32, a.numel(), "b")
    po = _ptr(d_out, torch.float64, 1, "d_out")
    if b.device != a.device or d_out.device != a.device:
        raise ValueError("a, b and d_out must live on one device")
    if stream is None:
        stream = torch.cuda.current_stream(a.device)
    rc = lib().frs_dot_noalloc(a.device.index, stream.cuda_stream, pa, pb, a.numel(), po)
    if rc != 0:
        raise FrsError(rc, lib().frs_dot_noalloc_last_error().decode())


class _DevicePtr:
    """Minimal __cuda_array_interface__ carrier so that torch can view library-owned device memory."""

    def __init__(self, ptr, shape):
        self.__cuda_array_interface__ = {"data": (int(ptr), False), "shape": tuple(shape), "typestr": "<f4", "version": 2}


def _device_view(ptr, shape, device):
    import torch
    return torch.as_tensor(_DevicePtr(ptr, shape), device=device)


class Context:
    """frs_ctx wrapper.  Methods mirror the C calls and take torch CUDA float32 tensors."""

    def __init__(self, ny, nx, nchan=1, device=0, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the fast-resolve hot path has no CPU fallback")
        self.torch = torch
        self.ny, self.nx, self.nchan, self.nfield = ny, nx, nchan, 0
        self.device = torch.device("cuda", device)
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        self.stream = stream
        self._h = _vp()
        rc = lib().frs_create(ny, nx, nchan, device, _vp(stream.cuda_stream), C.byref(self._h))
        if rc != 0:
            raise FrsError(rc, "frs_create")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().frs_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc):
        if rc != 0:
            raise FrsError(rc, lib().frs_last_error(self._h).decode())

    @property
    def npix(self):
        return self.ny * self.nx

    @property
    def f32(self):
        return self.torch.float32

    def new_image(self):
        return self.torch.empty((self.nchan, self.ny, self.nx), dtype=self.f32, device=self.device)

    def new_latent(self):
        return self.torch.empty((self.nfield, self.ny, self.nx), dtype=self.f32, device=self.device)

    # ---- setup
    def set_psf(self, psf):
        self._ck(lib().frs_set_psf(self._h, _ptr(psf, self.f32, self.nchan * 4 * self.npix, "psf")))

    def set_psf_weights(self, w_half):
        self._ck(lib().frs_set_psf_weights(
            self._h, _ptr(w_half, self.f32, self.nchan * 2 * self.ny * (self.nx + 1), "w_half")))

    def set_dirty(self, j):
        self._ck(lib().frs_set_dirty(self._h, _ptr(j, self.f32, self.nchan * self.npix, "dirty")))

    def set_amplitude(self, amp, mu):
        nfield = amp.shape[0]
        mu_arr = (_f * nfield)(*[float(m) for m in mu])
        self._ck(lib().frs_set_amplitude(self._h, nfield, _ptr(amp, self.f32, nfield * self.npix, "amp"), mu_arr))
        self.nfield = nfield

    def set_channel_lognu(self, lognu):
        arr = (_f * self.nchan)(*[float(v) for v in lognu])
        self._ck(lib().frs_set_channel_lognu(self._h, arr))

    def set_sky(self, sky):
        self._ck(lib().frs_set_sky(self._h, _ptr(sky, self.f32, self.nchan * self.npix, "sky")))

    # ---- Eq. 9 with the fitted noise kernel
    def set_noise_kernel(self, eps=None, kern=None):
        if kern is not None:
            self._ck(lib().frs_set_noise_kernel_array(self._h, _ptr(kern, self.f32, self.nchan * self.npix, "kern")))
        else:
            self._ck(lib().frs_set_noise_kernel(self._h, float(eps)))

    def get_noise_kernel(self):
        k = self.new_image()
        self._ck(lib().frs_get_noise_kernel(self._h, k.data_ptr()))
        return k

    def ninv_apply(self, x, y):
        self._ck(lib().frs_ninv_apply(self._h, _ptr(x, self.f32, self.nchan * self.npix, "x"),
                                      _ptr(y, self.f32, self.nchan * self.npix, "y")))
        return y

    def set_likelihood(self, mode):
        self._ck(lib().frs_set_likelihood(self._h, int(mode)))

    # ---- learned amplitude spectrum (NEXT-3, reading R17)
    def set_amplitude_model(self, hyper):
        h = (_f * 11)(*[float(x) for x in hyper])
        self._ck(lib().frs_set_amplitude_model(self._h, h))
        nb, nt = _i(0), _i(0)
        self._ck(lib().frs_amp_model_size(self.ny, self.nx, C.byref(nb), C.byref(nt)))
        self.nfield, self.nb, self.ntheta = 1, nb.value, nt.value

    def set_point_sources(self, yx, alpha, q):
        """yx: sequence of (y, x) pixels; the joint calls then take theta = [amplitude part | one latent per pixel]."""
        flat = [int(v) for p in yx for v in p]
        arr = (_i * max(1, len(flat)))(*flat)
        self._ck(lib().frs_set_point_sources(self._h, len(flat) // 2, arr, float(alpha), float(q)))
        self.npts = len(flat) // 2

    @property
    def ntheta_joint(self):
        return self.ntheta + getattr(self, "npts", 0)

    def amplitude_forward(self, theta, amp_out=None):
        self._ck(lib().frs_amplitude_forward(self._h, _ptr(theta, self.f32, None, "theta"),
                                             _ptr(amp_out, self.f32, self.npix, "amp_out")))

    def amplitude_jvp(self, dtheta, d_amp):
        self._ck(lib().frs_amplitude_jvp(self._h, _ptr(dtheta, self.f32, self.ntheta, "dtheta"), _ptr(d_amp, self.f32, self.npix, "d_amp")))

    def amplitude_vjp(self, g_amp, g_theta):
        self._ck(lib().frs_amplitude_vjp(self._h, _ptr(g_amp, self.f32, self.npix, "g_amp"), _ptr(g_theta, self.f32, self.ntheta, "g_theta")))

    def energy_grad_joint(self, xi, theta, grad_xi, grad_theta, with_prior=True):
        e = _d(0.0)
        self._ck(lib().frs_energy_grad_joint(self._h, _ptr(xi, self.f32, self.npix, "xi"), _ptr(theta, self.f32, self.ntheta_joint, "theta"),
                                             int(with_prior), C.byref(e), _ptr(grad_xi, self.f32, self.npix, "grad_xi"),
                                             _ptr(grad_theta, self.f32, self.ntheta_joint, "grad_theta")))
        return e.value

    def metric_apply_joint(self, dxi, dtheta, out_xi, out_theta, with_prior=True):
        self._ck(lib().frs_metric_apply_joint(self._h, _ptr(dxi, self.f32, self.npix, "dxi"), _ptr(dtheta, self.f32, self.ntheta_joint, "dtheta"),
                                              int(with_prior), _ptr(out_xi, self.f32, self.npix, "out_xi"),
                                              _ptr(out_theta, self.f32, self.ntheta_joint, "out_theta")))

    # ---- images smaller than the (power-of-two) grid: embedding, reading R19
    def set_psf_embedded(self, psf_img, ny_img, nx_img):
        self._ck(lib().frs_set_psf_embedded(self._h, _ptr(psf_img, self.f32, self.nchan * 4 * ny_img * nx_img, "psf_img"),
                                            int(ny_img), int(nx_img)))

    def set_field_of_view(self, ny_img, nx_img):
        self._ck(lib().frs_set_field_of_view(self._h, int(ny_img), int(nx_img)))

    # ---- building blocks of composed sky models (several GPs on patches, reading R20)
    def sky_energy_grad(self, sky, grad_sky):
        e = _d(0.0)
        self._ck(lib().frs_sky_energy_grad(self._h, _ptr(sky, self.f32, self.nchan * self.npix, "sky"), C.byref(e),
                                           _ptr(grad_sky, self.f32, self.nchan * self.npix, "grad_sky")))
        return e.value

    def dot(self, a, b):
        out = _d(0.0)
        self._ck(lib().frs_dot(self._h, _ptr(a, self.f32, None, "a"), _ptr(b, self.f32, a.numel(), "b"), a.numel(), C.byref(out)))
        return out.value

    def latent_jvp(self, v, dsky):
        self._ck(lib().frs_latent_jvp(self._h, _ptr(v, self.f32, self.npix, "v"), _ptr(dsky, self.f32, self.npix, "dsky")))

    def latent_vjp(self, w_sky, out, add=None):
        self._ck(lib().frs_latent_vjp(self._h, _ptr(w_sky, self.f32, self.npix, "w_sky"), _ptr(add, self.f32, self.npix, "add"),
                                      _ptr(out, self.f32, self.npix, "out")))

    def patch_insert_add(self, patch, y0, x0, field):
        nyp, nxp = patch.shape[-2], patch.shape[-1]
        self._ck(lib().frs_patch_insert_add(self._h, _ptr(patch, self.f32, nyp * nxp, "patch"), nyp, nxp, int(y0), int(x0),
                                            _ptr(field, self.f32, self.npix, "field")))

    def patch_crop(self, field, y0, x0, patch):
        nyp, nxp = patch.shape[-2], patch.shape[-1]
        self._ck(lib().frs_patch_crop(self._h, _ptr(field, self.f32, self.npix, "field"), nyp, nxp, int(y0), int(x0),
                                      _ptr(patch, self.f32, nyp * nxp, "patch")))

    def set_fused_passes(self, on):
        self._ck(lib().frs_set_fused_passes(self._h, int(bool(on))))

    def set_cuda_graphs(self, on):
        self._ck(lib().frs_set_cuda_graphs(self._h, int(bool(on))))

    # ---- major cycle (exact response on uv points; images are single-channel [ny][nx])
    def exact_response(self, uv, x, vis):
        nvis = uv.shape[0]
        self._ck(lib().frs_exact_response(self._h, _ptr(uv, self.f32, 2 * nvis, "uv"), nvis, _ptr(x, self.f32, self.npix, "x"),
                                          _ptr(vis, self.f32, 2 * nvis, "vis")))
        return vis

    def exact_adjoint(self, uv, wgt, vis, y):
        nvis = uv.shape[0]
        self._ck(lib().frs_exact_adjoint(self._h, _ptr(uv, self.f32, 2 * nvis, "uv"), _ptr(wgt, self.f32, nvis, "wgt"), nvis,
                                         _ptr(vis, self.f32, 2 * nvis, "vis"), _ptr(y, self.f32, self.npix, "y")))
        return y

    def major_cycle_residual(self, uv, wgt, dirty_full, sky, d_next):
        nvis = uv.shape[0]
        self._ck(lib().frs_major_cycle_residual(self._h, _ptr(uv, self.f32, 2 * nvis, "uv"), _ptr(wgt, self.f32, nvis, "wgt"), nvis,
                                                _ptr(dirty_full, self.f32, self.npix, "dirty_full"),
                                                _ptr(sky, self.f32, self.npix, "sky"), _ptr(d_next, self.f32, self.npix, "d_next")))
        return d_next

    # ---- MGVI
    def draw_sample(self, eta_xi, eta_d, sample, max_iter, rtol=0.0):
        it = _i(0)
        self._ck(lib().frs_draw_sample(self._h, _ptr(eta_xi, self.f32, self.nfield * self.npix, "eta_xi"),
                                       _ptr(eta_d, self.f32, self.nchan * self.npix, "eta_d"), int(max_iter), float(rtol),
                                       _ptr(sample, self.f32, self.nfield * self.npix, "sample"), C.byref(it)))
        return it.value

    def kl_energy_grad(self, xi, samples, grad, mirrored=True):
        h = _d(0.0)
        ns = samples.shape[0]
        self._ck(lib().frs_kl_energy_grad(self._h, _ptr(xi, self.f32, self.nfield * self.npix, "xi"),
                                          _ptr(samples, self.f32, ns * self.nfield * self.npix, "samples"), ns, int(mirrored),
                                          None, C.byref(h), _ptr(grad, self.f32, self.nfield * self.npix, "grad")))
        return h.value

    def kl_metric_apply(self, xi, samples, v, out, mirrored=True):
        ns = samples.shape[0]
        self._ck(lib().frs_kl_metric_apply(self._h, _ptr(xi, self.f32, self.nfield * self.npix, "xi"),
                                           _ptr(samples, self.f32, ns * self.nfield * self.npix, "samples"), ns, int(mirrored),
                                           _ptr(v, self.f32, self.nfield * self.npix, "v"),
                                           _ptr(out, self.f32, self.nfield * self.npix, "out")))
        return out

    # ---- hot path
    def sky_forward(self, xi, sky=None):
        self._ck(lib().frs_sky_forward(self._h, _ptr(xi, self.f32, self.nfield * self.npix, "xi"),
                                       _ptr(sky, self.f32, self.nchan * self.npix, "sky")))
        return sky

    def psf_apply(self, x, y):
        self._ck(lib().frs_psf_apply(self._h, _ptr(x, self.f32, self.nchan * self.npix, "x"),
                                     _ptr(y, self.f32, self.nchan * self.npix, "y")))
        return y

    def sky_metric_apply(self, x, y):
        self._ck(lib().frs_sky_metric_apply(self._h, _ptr(x, self.f32, self.nchan * self.npix, "x"),
                                            _ptr(y, self.f32, self.nchan * self.npix, "y")))
        return y

    def energy_grad(self, xi, grad, with_prior=True, d_energy=None, host_energy=True):
        h = _d(0.0)
        self._ck(lib().frs_energy_grad(self._h, _ptr(xi, self.f32, self.nfield * self.npix, "xi"), int(with_prior),
                                       _ptr(d_energy, self.torch.float64, 1, "d_energy"),
                                       C.byref(h) if host_energy else None,
                                       _ptr(grad, self.f32, self.nfield * self.npix, "grad")))
        return h.value if host_energy else None

    def metric_apply(self, v, out, with_prior=True):
        self._ck(lib().frs_metric_apply(self._h, _ptr(v, self.f32, self.nfield * self.npix, "v"), int(with_prior),
                                        _ptr(out, self.f32, self.nfield * self.npix, "out")))
        return out

    def cg_solve(self, b, x, max_iter, rtol=0.0, with_prior=True, res_history=None):
        it, rn = _i(0), _d(0.0)
        if res_history is not None and res_history.numel() < max_iter + 1:
            raise ValueError("res_history needs max_iter + 1 doubles")
        self._ck(lib().frs_cg_solve(self._h, _ptr(b, self.f32, self.nfield * self.npix, "b"),
                                    _ptr(x, self.f32, self.nfield * self.npix, "x"), int(max_iter), float(rtol),
                                    int(with_prior), C.byref(it), C.byref(rn),
                                    _ptr(res_history, self.torch.float64, None, "res_history")))
        return it.value, rn.value

    def cg_load(self, r, p, rr):
        self._ck(lib().frs_cg_load(self._h, _ptr(r, self.f32, self.nfield * self.npix, "r"),
                                   _ptr(p, self.f32, self.nfield * self.npix, "p"), float(rr)))

    def cg_step(self, x, with_prior=True):
        self._ck(lib().frs_cg_step(self._h, _ptr(x, self.f32, self.nfield * self.npix, "x"), int(with_prior)))

    def cg_step_begin(self):
        """Likelihood part q = J^T C J p of this context's channels; returns q as a tensor VIEW of the
        ctx-owned device buffer (to be summed over ranks in place), see frs_cg_step_begin."""
        q = _vp()
        self._ck(lib().frs_cg_step_begin(self._h, C.byref(q)))
        return _device_view(q.value, (self.nfield, self.ny, self.nx), self.device)

    def cg_step_end(self, x, with_prior=True):
        self._ck(lib().frs_cg_step_end(self._h, _ptr(x, self.f32, self.nfield * self.npix, "x"), int(with_prior)))

    def cg_read_state(self):
        """Copies of the ctx-owned r, p, q (torch) and the scalar block (numpy float64[8]:
        rr, pq, rr_new, alpha, beta, breakdown, bb, -) after a cg_step / cg_solve."""
        r, p, q = self.new_latent(), self.new_latent(), self.new_latent()
        sc = (_d * 8)()
        self._ck(lib().frs_cg_read_state(self._h, r.data_ptr(), p.data_ptr(), q.data_ptr(), sc))
        return r, p, q, np.array(list(sc), dtype=np.float64)

    # ---- host-buffer entry points (torch CPU tensors, ideally pinned)
    def sky_metric_apply_host(self, x_host, y_host):
        self._ck(lib().frs_sky_metric_apply_host(self._h, _vp(x_host.data_ptr()), _vp(y_host.data_ptr())))
        return y_host

    def sky_metric_apply_host_batch(self, x_hosts, y_hosts):
        """Lists of (pinned) CPU tensors; copies and kernels of neighbouring items overlap inside the library."""
        n = len(x_hosts)
        xs = (_vp * max(1, n))(*[x.data_ptr() for x in x_hosts])
        ys = (_vp * max(1, n))(*[y.data_ptr() for y in y_hosts])
        self._ck(lib().frs_sky_metric_apply_host_batch(self._h, n, xs, ys))
        return y_hosts

    def psf_apply_host(self, x_host, y_host):
        self._ck(lib().frs_psf_apply_host(self._h, _vp(x_host.data_ptr()), _vp(y_host.data_ptr())))
        return y_host

    def check_guards(self):
        """(arrays with a corrupted guard zone, arrays under guard); needs FRS_GUARD=1 in the environment at construction."""
        n = _i(0)
        bad = lib().frs_debug_check_guards(self._h, C.byref(n))
        if bad < 0:
            raise FrsError(-1, "frs_debug_check_guards")
        return bad, n.value

    # ---- instrumentation
    def launch_count(self):
        return int(lib().frs_launch_count(self._h))

    def profile_enable(self, on=True):
        self._ck(lib().frs_profile_enable(self._h, int(on)))

    def profile_read(self):
        ms = (_d * 5)()
        n = (C.c_longlong * 5)()
        self._ck(lib().frs_profile_read(self._h, ms, n))
        names = ["conv_rows_fwd", "conv_cols", "conv_rows_inv", "hart_rows", "hart_cols"]
        return {k: (ms[i], int(n[i])) for i, k in enumerate(names)}
