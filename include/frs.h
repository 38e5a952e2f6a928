/* frs.h -- C ABI of the fast-resolve hot path on B200 (sm_100a).
 *
 * The library evaluates the PSF-convolution likelihood of fast-resolve (arXiv 2406.09144),
 *     E(s) = 1/2 s^T (PSF * s) - j^T s,        s = exp(correlated field),
 * its gradient and its Fisher-metric-vector product, and solves M x = b by conjugate gradients.
 * Citations `P:<n>` are lines of the paper text; `R<k>` are the
 * readings listed in DESIGN.md for points the paper leaves open.
 *
 * That energy is Eq. 9 of the paper in the limit N' = R' (likelihood mode 0, the default and the one the headline
 * benchmark times: one padded PSF convolution per metric apply).  The paper's literal likelihood with the separately
 * fitted noise kernel (Eq. 15-18: three convolutions per metric apply) is mode 1, frs_set_likelihood.  Further families of
 * calls, each in its own section below: MGVI samples and the sample-averaged KL; the major-cycle residual with an exact
 * response on uv points; the learned amplitude spectrum with the joint latent vector (xi, theta) and inverse-gamma
 * point-source pixels; building blocks for several Gaussian processes on patches; images that are not a power of two by
 * embedding; host-buffer entry points; instrumentation and self-tests.
 *
 * Conventions (all calls)
 *   - frs_ctx owns the PSF spectrum, dirty image, amplitude spectra, the cached sky of the current
 *     position and all scratch.  The caller owns every array it passes; set_* calls COPY.
 *   - Unless a name ends in `_host`, array arguments are DEVICE pointers to contiguous float32,
 *     16-byte aligned, on the ctx's device.  Scalars documented "host" are host pointers.
 *   - Layout: images [nchan][ny][nx] row-major (x fastest); latent arrays [nfield][ny][nx] indexed
 *     by harmonic mode (ky, kx) in DFT order; PSF half spectrum [nchan][2ny][nx+1].
 *   - Calls enqueue work on the ctx's stream and return; they synchronise only where a host output
 *     is requested (documented per call).  One ctx per stream; a ctx is not thread-safe.
 *   - Input and output arrays of one call must not overlap unless stated.
 *   - Return value: 0 on success, a negative FRS_E* code otherwise.  No exceptions cross the ABI.
 *   - ny, nx: powers of two in [32, 4096]; nchan >= 1; nfield in {1, 2}.
 */
#ifndef FRS_H
#define FRS_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct frs_ctx frs_ctx;

#define FRS_OK 0
#define FRS_EINVAL (-1)     /* bad size, NULL or misaligned pointer */
#define FRS_ESTATE (-2)     /* call order: e.g. metric_apply before a position / PSF was set */
#define FRS_ENOTPSD (-3)    /* PSF spectrum has a significant negative or imaginary part */
#define FRS_ECUDA (-4)      /* CUDA runtime error; text via frs_last_error */
#define FRS_EBREAKDOWN (-5) /* CG met <p, M p> <= 0 */

/* Create a context for images of ny x nx pixels, nchan frequency channels, on CUDA device `device`,
 * enqueuing on `stream` (a cudaStream_t; NULL = the legacy default stream).  The number of latent
 * fields is fixed later by frs_set_amplitude.  Allocates all tables; scratch is allocated lazily. */
int frs_create(int ny, int nx, int nchan, int device, void* stream, frs_ctx** out);
void frs_destroy(frs_ctx* ctx);
/* Text of the last error of this ctx (never NULL; owned by the ctx). */
const char* frs_last_error(const frs_ctx* ctx);
/* Library version / build string (static storage). */
const char* frs_version(void);

/* ---- setup (untimed) ---------------------------------------------------------------------- */

/* PSF given in image space: psf [nchan][2ny][2nx], origin at [0][0], negative offsets wrapped
 * (R2).  Computes W = DFT(psf)/(4 ny nx) with a direct O(M^2 log M) transform on the device and
 * requires max|Im W| <= 1e-5 max W and min Re W >= -1e-5 max W, else FRS_ENOTPSD (R4; P:191:
 * a covariance kernel must be real and positive).  Stores max(Re W, 0).  Synchronises. */
int frs_set_psf(frs_ctx* ctx, const float* psf);
/* PSF given as its real, non-negative half spectrum W [nchan][2ny][nx+1] (the gridded, Hermitian-
 * symmetrised visibility weights; P:180 'FFT[I^PSF]', R3: (C x)[n] = sum_k W[k] xhat[k] e^{+2 pi i k.n/M},
 * so the PSF peak equals sum W).  Negative entries -> FRS_ENOTPSD.  Synchronises. */
int frs_set_psf_weights(frs_ctx* ctx, const float* w_half);

/* ---- images that are not a power of two (3600^2) by embedding; reading R19 ----
 * Eq. 14 is a LINEAR convolution of the ny_img x nx_img image with a PSF twice its size: any padded grid of at least
 * twice the image computes it exactly.  The context is created on the next power of two (ny, nx); every image-sized
 * array of the other calls stays [ny][nx] with the image in its corner [0, ny_img) x [0, nx_img); the correlated field
 * lives on the whole grid and the sky is its crop: frs_sky_forward / frs_set_sky zero it outside the image, and with it
 * every fused . s of the gradient and the metric.  (Mode 1 applies Eq. 18 on the embedding grid.) */

/* psf_img: device [nchan][2 ny_img][2 nx_img], origin at [0][0], negative offsets wrapped.  Copies it to the offsets
 * |dy| < ny_img, |dx| < nx_img of the context's padded grid (zero elsewhere), takes its spectrum as frs_set_psf does --
 * but keeps the sign of Re W (the truncated PSF is real and even, not a covariance on the larger grid; FRS_ENOTPSD only
 * for max|Im W| > 1e-5 max W) -- and sets the field of view.  Synchronises. */
int frs_set_psf_embedded(frs_ctx* ctx, const float* psf_img, int ny_img, int nx_img);
/* The sky is zero outside [0, ny_img) x [0, nx_img) from now on (ny_img = ny, nx_img = nx: whole grid again).  For PSFs
 * given as weights on the context's own padded grid.  Invalidates the cached position. */
int frs_set_field_of_view(frs_ctx* ctx, int ny_img, int nx_img);

/* Dirty image j = I^D [nchan][ny][nx]  (Eq. 6, Eq. 8).  For major cycles pass
 * j_eff = d_i + C s_{i-1} (Eq. 21, R13). */
int frs_set_dirty(frs_ctx* ctx, const float* j);
/* Correlated-field model (R6): amplitude spectra A [nfield][ny][nx] (real >= 0, even in k) and
 * offsets mu [nfield] (HOST pointer).  nfield = 1: s = exp(mu + H[A xi]);  nfield = 2:
 * s_c = exp(tau_0 + lognu_c tau_1).  Invalidates the cached position. */
int frs_set_amplitude(frs_ctx* ctx, int nfield, const float* amp, const float* mu_host);
/* ln(nu_c / nu_0) per channel, HOST pointer [nchan]; only used when nfield == 2. */
int frs_set_channel_lognu(frs_ctx* ctx, const float* lognu_host);

/* ---- hot path -------------------------------------------------------------------------------- */

/* s = exp(correlated field of xi): sets the position, caches s inside the ctx and, if `sky` is
 * not NULL, also writes it there [nchan][ny][nx]  (R6). */
int frs_sky_forward(frs_ctx* ctx, const float* xi, float* sky);
/* y = C x: zero-pad, FFT, multiply by W, inverse FFT, crop (Eq. 14). x, y [nchan][ny][nx]. */
int frs_psf_apply(frs_ctx* ctx, const float* x, float* y);
/* 'L1 apply', the headline operator: y = s . C (s . x) at the cached position -- the likelihood
 * Fisher metric in log-sky coordinates (Eq. 10, R8).  Needs a prior frs_sky_forward /
 * frs_energy_grad / frs_set_sky. */
int frs_sky_metric_apply(frs_ctx* ctx, const float* x, float* y);
/* Set the cached sky directly (copy), bypassing the correlated-field model. */
int frs_set_sky(frs_ctx* ctx, const float* sky);
/* E = sum_c 1/2 <s_c, C_c s_c> - <j_c, s_c> (+ 1/2 <xi, xi> if with_prior) and its gradient
 * grad [nfield][ny][nx] = J^T (C s - j) (+ xi)   (Eq. 9 with N' = R', R1, R8).
 * d_energy: device double (may be NULL); h_energy: host double (may be NULL; non-NULL makes the
 * call synchronise).  Sets the position to xi. */
int frs_energy_grad(frs_ctx* ctx, const float* xi, int with_prior, double* d_energy, double* h_energy, float* grad);
/* 'L2 apply': out = J^T C J v (+ v if with_prior) at the cached position -- the MGVI metric
 * (R8).  v, out [nfield][ny][nx]. */
int frs_metric_apply(frs_ctx* ctx, const float* v, int with_prior, float* out);
/* Solve M x = b by textbook CG (R9).  x: in = x0, out = solution.  Runs until max_iter or
 * ||r|| <= rtol ||b|| (rtol = 0: exactly max_iter iterations, fully asynchronous until the end).
 * The stopping test is evaluated on the DEVICE after every iteration; once it holds, the vector updates of the
 * iterations still enqueued are no-ops, so x is exactly the iterate at which the test was met.  With rtol > 0 the
 * host reads the flag every 8 iterations only to stop enqueueing (up to 7 wasted metric applies, no change of x).
 * h_iters (host, may be NULL): iterations done.  h_resnorm (host, may be NULL): final ||r||.
 * d_res_history (DEVICE double [max_iter+1], may be NULL): ||r_k|| (constant after the stopping point).
 * Synchronises at the end.  FRS_EBREAKDOWN if <p, M p> <= 0 was met (x is the last good iterate). */
int frs_cg_solve(frs_ctx* ctx, const float* b, float* x, int max_iter, float rtol, int with_prior,
                 int* h_iters, double* h_resnorm, double* d_res_history);
/* frs_cg_solve (and the solves inside frs_draw_sample) run iteration 0 with plain launches and replay every later
 * iteration as ONE captured CUDA graph (the iteration index lives on the device), rebuilt only when a frozen argument
 * (x, with_prior, likelihood mode, history pointer, rtol, number of fields) changes.  on = 0 turns that off (plain
 * launches throughout: what the profiling events of frs_profile_enable need, and the comparison arm of bench.py).
 * The results are the same kernels on the same data either way.  Default: on. */
int frs_set_cuda_graphs(frs_ctx* ctx, int on);
/* In the latent-space calls (single channel, one field, no point sources, row length 1024 .. 4096) the last pass of the
 * convolution and the row pass of the Hartley transform that follows run as ONE kernel: s . C(...) goes from registers
 * straight into the half-length row transform instead of through memory.  on = 0: the two separate passes (same
 * arithmetic; the fp64 energy sums are added in another order).  Default: on. */
int frs_set_fused_passes(frs_ctx* ctx, int on);
/* Copy out the CG state of the last frs_cg_solve / frs_cg_step: r, p, q (DEVICE pointers,
 * [nfield][ny][nx] each, any may be NULL) and the scalar block scal_host (HOST double[8], may be NULL:
 * rr, pq, rr_new, alpha, beta, breakdown, bb, -).  Synchronises. */
int frs_cg_read_state(frs_ctx* ctx, float* r, float* p, float* q, double* scal_host);
/* One CG iteration on caller-visible state (teacher-forced parity, R9): given x, and the ctx's
 * r, p and rr (loaded with frs_cg_load), computes q = M p, alpha, x, r, beta, p. */
int frs_cg_load(frs_ctx* ctx, const float* r, const float* p, double rr_host);
int frs_cg_step(frs_ctx* ctx, float* x, int with_prior);
/* The same iteration split around the one exchange step of a channel-sharded run (each
 * rank holds a subset of the channels, latent vectors are replicated).  frs_cg_step_begin computes
 * the likelihood part q = J^T C J p of THIS context's channels (no prior term) into ctx-owned storage
 * and returns its DEVICE pointer in *d_q ([nfield][ny][nx]); the caller sums q over the ranks in place
 * (ncclAllReduce on the ctx's stream); frs_cg_step_end adds the prior term (q += p if with_prior) and
 * finishes the iteration exactly as frs_cg_step (alpha, x, r, beta, p).  Errors as frs_cg_step. */
int frs_cg_step_begin(frs_ctx* ctx, float** d_q);
int frs_cg_step_end(frs_ctx* ctx, float* x, int with_prior);

/* ---- the likelihood the paper ran: Eq. 9 with the separately fitted noise kernel ----------------
 * P:154 (Eq. 9), P:162 (Eq. 11), P:186-206 (Eq. 15-18); reading R14.
 *   E_lh = 1/2 (j - C s)^T N'^-1 (j - C s),  N'^-1 x = FFT^-1[ K^-1 . FFT x ]  on the UNPADDED ny x nx grid, periodic
 *   (Eq. 18), K = exp(xi_bar) + eps real, even and >= eps (Eq. 16);  Fisher metric J^T C N'^-1 C J (+ 1).
 * The default likelihood of every call above is its N' = R' limit (mode 0). */

/* Fit K to the PSF that is set (Eq. 17, closed form by Parseval: K = max(Re[FFT(N' I_delta) conj FFT(I_delta)], eps),
 * I_delta a point source at (ny/2, nx/2), N' = C + eps 1).  eps > 0 (same units as the PSF).  Errors: FRS_ESTATE
 * without a PSF, FRS_EINVAL for eps <= 0.  A later frs_set_psf* discards the kernel and returns to mode 0. */
int frs_set_noise_kernel(frs_ctx* ctx, float eps);
/* Or supply K directly: device [nchan][ny][nx], harmonic (DFT) order, strictly positive and even (K[-k] = K[k] to
 * 1e-5 relative), else FRS_ENOTPSD.  Copied. */
int frs_set_noise_kernel_array(frs_ctx* ctx, const float* kern);
/* Copy of the kernel in use, device [nchan][ny][nx]. */
int frs_get_noise_kernel(frs_ctx* ctx, float* kern);
/* y = N'^-1 x (sky space, [nchan][ny][nx]); x == y allowed. */
int frs_ninv_apply(frs_ctx* ctx, const float* x, float* y);
/* mode 0: E = 1/2 s^T C s - j^T s, metric J^T C J (+1)   (N' = R' limit, R1)
 * mode 1: Eq. 9 with N'^-1 of Eq. 18, metric J^T C N'^-1 C J (+1); needs a noise kernel (else FRS_ESTATE).
 * Affects frs_energy_grad, frs_metric_apply, frs_cg_solve / _step / _step_begin. */
int frs_set_likelihood(frs_ctx* ctx, int mode);

/* ---- NEXT-3: learned amplitude spectrum of the diffuse-emission prior (parameters of Table A.1 / B.1,
 * P:536-566; the paper defers the definition to Arras et al. 2021a -- DESIGN.md reading R17 states the one built) ----
 * The amplitude A of frs_set_amplitude becomes a function of a standard-normal latent vector theta:
 *   radial bins b(mode) = rint(|k|) (cycles per longer field side), nb bins, t_b = ln b;
 *   theta = [xi_fluct, xi_slope, xi_flex, xi_asp, xi_zm, zeta_1..zeta_{nb-2}, eta_1..eta_{nb-2}]  (ntheta = 5 + 2 (nb - 2));
 *   fluct, flex, asp, zm log-normal with the given mean / std, slope = mean + std xi_slope;
 *   dev_1 = vel_1 = 0, dev_{j+1} = dev_j + vel_j D_j + flex asp sqrt(D_j) eta_j, vel_{j+1} = vel_j + flex sqrt(D_j) zeta_j,
 *   D_j = t_{j+1} - t_j;  ln P_b = slope t_b + dev_b;  a_b = exp(ln P_b / 2);  A = fluct a_b / sqrt(sum mult_b a_b^2) on
 *   bin b >= 1, A = zm on the zero mode;  sky = exp(offset + H[A . xi]).
 * Single channel, one field.  The spectrum (a few thousand bins) is evaluated in fp64 on the device; A is fp32. */

/* Host arithmetic only: number of bins and length of theta for an ny x nx grid (either pointer may be NULL). */
int frs_amp_model_size(int ny, int nx, int* nb, int* ntheta);
/* hyper_host: HOST float[11] = offset, zero-mode mean, std, fluctuations mean, std, loglogavgslope mean, std,
 * flexibility mean, std, asperity mean, std (the rows of Table A.1).  Builds the bin index of the grid on first use.
 * Switches the context to nfield = 1 with mu = offset and invalidates amplitude and position; frs_set_amplitude
 * switches back.  Errors: FRS_ESTATE for nchan != 1, FRS_EINVAL for a non-positive log-normal mean or a negative std. */
int frs_set_amplitude_model(frs_ctx* ctx, const float* hyper_host);
/* A(theta) becomes the context's amplitude (theta: device float[ntheta], copied); amp_out: device [ny][nx] or NULL.
 * Invalidates the cached position. */
int frs_amplitude_forward(frs_ctx* ctx, const float* theta, float* amp_out);
/* d_amp [ny][nx] = (dA/dtheta) dtheta and g_theta [ntheta] = (dA/dtheta)^T g_amp at the theta of the last forward. */
int frs_amplitude_jvp(frs_ctx* ctx, const float* dtheta, float* d_amp);
int frs_amplitude_vjp(frs_ctx* ctx, const float* g_amp, float* g_theta);
/* Inverse-gamma point-source pixels ("pixels independently modeled with an inverse gamma prior ... locations
 * manually set"; reading R18): flux_p = F^-1(Phi(xi_p)), F the CDF of pdf(x) ~ x^(-alpha-1) exp(-q / x), is
 * added to the diffuse sky at pixel (y_p, x_p).  yx_host: HOST int[npts][2]; npts = 0 removes them; npts <= 1024.
 * With point sources set, theta of the joint calls below is [amplitude part (frs_amp_model_size) | xi_p, p < npts] and
 * so are grad_theta, dtheta, out_theta; frs_sky_forward adds the fluxes of the last joint position (xi_p = 0 before
 * one), and every latent-space call uses the diffuse sky as the Jacobian of the diffuse part at those pixels.
 * Errors: FRS_EINVAL (pixel outside the field of view, repeated pixel, alpha or q <= 0), FRS_ESTATE for nchan != 1.
 * frs_set_field_of_view / frs_set_psf_embedded return FRS_EINVAL, changing nothing, if a point set earlier would fall outside. */
int frs_set_point_sources(frs_ctx* ctx, int npts, const int* yx_host, float alpha, float q);
/* Energy of the likelihood in use (frs_set_likelihood) at the joint position (xi, theta), prior 1/2 <xi,xi> + 1/2
 * <theta,theta> if with_prior, and its gradient with respect to both (grad_xi [ny][nx], grad_theta [ntheta]).
 * Sets the joint position.  h_energy: host double or NULL (non-NULL synchronises). */
int frs_energy_grad_joint(frs_ctx* ctx, const float* xi, const float* theta, int with_prior, double* h_energy, float* grad_xi,
                          float* grad_theta);
/* Fisher metric of the joint model at the joint position: (out_xi, out_theta) = J^T C J (dxi, dtheta) (+ (dxi, dtheta)),
 * J = d sky / d (xi, theta) = diag(s) H [diag(A) . + diag(xi) dA/dtheta .]   (mode 1: C N'^-1 C in the middle).
 * FRS_ESTATE without a joint position. */
int frs_metric_apply_joint(frs_ctx* ctx, const float* dxi, const float* dtheta, int with_prior, float* out_xi, float* out_theta);

/* ---- building blocks of composed sky models: several Gaussian processes on patches ("each of these sources with a
 * separate exponentiated Gaussian process ... a third Gaussian process model for the background", Fig. 10; R20) ----
 * s = sum_k insert_k( exp(mu_k + H_k[A_k xi_k]) ): one context per component (its own power-of-two grid, amplitude, offset) and
 * one context of the full field that owns PSF, dirty image and likelihood.  These calls are the two halves the fused calls
 * above combine; `PatchModel` in paper_2406_09144_b200/patches.py strings them together (no arithmetic in Python). */

/* Likelihood energy (NO prior term) of a caller-supplied sky and its derivative with respect to the sky:
 * mode 0: E = 1/2 <s, C s> - <j, s>, grad_sky = C s - j;  mode 1: E = 1/2 r^T N'^-1 r, grad_sky = -C N'^-1 r, r = j - C s.
 * sky, grad_sky: device [nchan][ny][nx], natural orientation.  Sets the sky as frs_set_sky does.  h_energy: host double
 * or NULL (non-NULL synchronises). */
int frs_sky_energy_grad(frs_ctx* ctx, const float* sky, double* h_energy, float* grad_sky);
/* Jacobian of one log-normal field at the cached position (frs_sky_forward), single channel, one field:
 * dsky [ny][nx] = s . H[A v]   and   out [ny][nx] = A . H[s . w_sky] (+ add if non-NULL). */
int frs_latent_jvp(frs_ctx* ctx, const float* v, float* dsky);
int frs_latent_vjp(frs_ctx* ctx, const float* w_sky, const float* add, float* out);
/* *h_out = <a, b> over n device floats (n a multiple of 4, 16-byte aligned), accumulated in fp64 in a fixed order (the prior
 * terms 1/2 <xi_k, xi_k> of a composed model).  Synchronises. */
int frs_dot(frs_ctx* ctx, const float* a, const float* b, long long n, double* h_out);
/* field [ny][nx] of THIS context: field[y0 + y][x0 + x] += patch[y][x], patch [nyp][nxp]; and the crop patch = field[...].
 * FRS_EINVAL if the patch does not lie inside the field. */
int frs_patch_insert_add(frs_ctx* ctx, const float* patch, int nyp, int nxp, int y0, int x0, float* field);
int frs_patch_crop(frs_ctx* ctx, const float* field, int nyp, int nxp, int y0, int x0, float* patch);

/* ---- MGVI: posterior samples and the sample-averaged KL (reading R15) ------------
 * MGVI approximates the posterior by N(xi, M(xi)^-1), M the metric above, and minimises the KL estimated on samples
 * xi +- sigma_i, sigma_i ~ N(0, M^-1).  The random numbers are INPUTS (white N(0,1) arrays drawn by the caller). */

/* One sample at the cached position (Eq. 9 likelihood, mode 1, only): m = eta_xi + J^T C N'^-1/2 eta_d has covariance M;
 * sample = M^-1 m by CG from 0 (max_iter, rtol as frs_cg_solve).  eta_xi [nfield][ny][nx], eta_d [nchan][ny][nx] white
 * noise (device); sample [nfield][ny][nx].  h_iters (host, may be NULL).  Synchronises.  Errors: FRS_ESTATE in mode 0
 * (the square root of C needs noise on the padded grid: not provided) or without a position. */
int frs_draw_sample(frs_ctx* ctx, const float* eta_xi, const float* eta_d, int max_iter, float rtol, float* sample, int* h_iters);
/* Sample-averaged KL and gradient: mean over the positions xi + sigma_i (and xi - sigma_i if mirrored) of E_tot and
 * grad E_tot (likelihood of the current mode + prior).  samples: device [nsamples][nfield][ny][nx].  Energy outputs
 * as frs_energy_grad.  Leaves the cached position at xi. */
int frs_kl_energy_grad(frs_ctx* ctx, const float* xi, const float* samples, int nsamples, int mirrored, double* d_energy,
                       double* h_energy, float* grad);
/* out = mean over the same positions of M(xi +- sigma_i) v (with the prior term): the metric of the KL's Newton-CG step.
 * Recomputes the sky at every position (2 nsamples sky evaluations and metric applies per call).  Leaves the position at xi. */
int frs_kl_metric_apply(frs_ctx* ctx, const float* xi, const float* samples, int nsamples, int mirrored, const float* v, float* out);

/* ---- major cycle: exact response on a list of uv points (Alg. 1, Eq. 20-22; Eq. 1; reading R16) ----
 * One channel at a time: images are [ny][nx] (any channel of a context), ny, nx <= 1024 (direct sums, O(nvis npix);
 * else FRS_EINVAL).  uv: DEVICE float [nvis][2] = (u, v) in cell units of the padded (2ny x 2nx) grid, NOT rounded to
 * cells; wgt: DEVICE float [nvis] = N^-1 (natural weighting: the scale w0 of the weight grid); vis: DEVICE float
 * [nvis][2] = (Re, Im).  A minor cycle on the residual d_i uses frs_set_dirty(d_i + C s_{i-1}) (R13). */

/* vis = R x:  V_k = sum_pixels x[y][x] exp(-2 pi i (u_k x / (2 nx) + v_k y / (2 ny))). */
int frs_exact_response(frs_ctx* ctx, const float* uv, int nvis, const float* x, float* vis);
/* y = R^dagger N^-1 vis, each visibility with its conjugate (the convention of the weight grid, R5):
 * y[y][x] = sum_k 2 w_k Re(V_k exp(+2 pi i (u_k x / (2 nx) + v_k y / (2 ny)))).  The dirty image is frs_exact_adjoint(V). */
int frs_exact_adjoint(frs_ctx* ctx, const float* uv, const float* wgt, int nvis, const float* vis, float* y);
/* d_next = dirty_full - R^dagger N^-1 R sky   (Eq. 20, 22).  d_next may alias dirty_full. */
int frs_major_cycle_residual(frs_ctx* ctx, const float* uv, const float* wgt, int nvis, const float* dirty_full, const float* sky,
                             float* d_next);

/* ---- host-buffer entry points (end-to-end measurements: copies are part of the call) -------- */

/* y = s . C (s . x) with x, y in HOST memory (pinned or pageable), [nchan][ny][nx].
 * Copies x to the device, runs frs_sky_metric_apply, copies y back, synchronises. */
int frs_sky_metric_apply_host(frs_ctx* ctx, const float* x_host, float* y_host);
/* n independent applies y_k = s . C (s . x_k) with HOST buffers (x_hosts, y_hosts: host arrays of n host pointers; the
 * buffers should be pinned, pageable memory makes the copies synchronous).  The copies of neighbouring items overlap the
 * kernels: host -> device of item k + 1 and device -> host of item k - 1 run on two copy streams of the context while
 * item k computes (two device buffers each way), so the throughput is that of the slowest of the three.  The same x or y
 * buffer may appear again only two items later.  Synchronises at the end. */
int frs_sky_metric_apply_host_batch(frs_ctx* ctx, int n, const float* const* x_hosts, float* const* y_hosts);
/* y = C x with HOST buffers. */
int frs_psf_apply_host(frs_ctx* ctx, const float* x_host, float* y_host);

/* ---- an entry point that allocates nothing ------------------------------------------------------
 * Everything above needs a frs_ctx, and a context allocates device memory: tables in frs_create, the scratch arrays on
 * first use.  Some callers cannot afford a single cudaMalloc: a process whose framework allocator (PyTorch's caching
 * allocator, say) has already taken the GPU's memory for itself, so that an allocation made behind its back fails or
 * eats into what it planned with; and a latency-bound loop -- a sharded CG between two all-reduces -- in which
 * cudaMalloc / cudaFree would hold up every stream of the device.  For them the inner product of frs_dot (the prior
 * terms 1/2 <xi_k, xi_k> of a composed model, the scalars of a CG written by the caller) exists in a second form that
 * needs no context and calls no cudaMalloc, cudaFree or other allocating routine.  Its only scratch, one fp64 partial sum
 * per CTA, is a fixed 9 472-byte array inside the library's device code; every GPU that loads libfrs.so holds that array
 * until the process exits. */

/* Largest n frs_dot_noalloc accepts: 2^28 floats = 1 GiB per operand, 8 x the largest latent vector of this library
 * (2 fields x 4096^2).  The scratch itself never overflows -- at most 1184 CTAs stride over the data, whatever n -- so
 * this is the range the entry point is specified and tested for, and anything larger is refused rather than run. */
#define FRS_DOT_NOALLOC_MAX_N (1LL << 28)

/* *d_out = <a, b> over n floats, products and sums in fp64 in the fixed order of frs_dot (the same bits).
 *   device : CUDA device ordinal (0 .. 63) that holds a, b and d_out; made current on the calling thread, as every frs_*
 *            call does with its context's device.
 *   stream : cudaStream_t on that device (NULL = the legacy default stream).  The two kernels are enqueued there and the
 *            call returns without synchronising; d_out is valid once the stream reaches that point.
 *   a, b   : DEVICE float32 [n], 16-byte aligned, owned by the caller, read only.  n: positive multiple of 4.
 *   d_out  : DEVICE double, 8-byte aligned, owned by the caller.
 * Set-up: the FIRST call on each device looks up where the scratch array lives on that device (once, under a lock).
 * Make that first call during initialisation, before any stream capture is begun on the thread.
 * Sharing: every call on a device uses the same scratch array, on whatever stream.  The array keeps what the last call
 * wrote; no slot is read before the same call has written it, so nothing has to be cleared between calls.  But two calls
 * whose kernels can overlap on the GPU (different streams without an event between them, or two host threads) race on
 * it and both results are garbage: order them on one stream or with events.
 * Errors (text via frs_dot_noalloc_last_error): FRS_EINVAL for a NULL or misaligned pointer, n <= 0, n not a multiple
 * of 4, n > FRS_DOT_NOALLOC_MAX_N ("beyond the maximum"), device outside 0 .. 63; FRS_ECUDA for a CUDA error.  Nothing
 * is enqueued when an error is returned. */
int frs_dot_noalloc(int device, void* stream, const float* a, const float* b, long long n, double* d_out);
/* Text of the calling thread's last frs_dot_noalloc error (static thread-local storage, never NULL). */
const char* frs_dot_noalloc_last_error(void);

/* ---- instrumentation ---------------------------------------------------------------------------- */

/* Number of kernels this ctx has launched since creation (monotone). */
long long frs_launch_count(const frs_ctx* ctx);
/* When enabled, every FFT pass is bracketed by CUDA events on the ctx's stream.  frs_profile_read
 * synchronises and returns accumulated milliseconds and launch counts per pass kind:
 * 0 rows_fwd (conv), 1 conv_cols, 2 rows_inv, 3 rows_fwd (Hartley), 4 hart_cols.  Resets on read.
 * While enabled, CG iterations run as plain launches and the latent-space calls use the two separate passes instead of the
 * fused inverse + Hartley row pass (frs_set_fused_passes), so that every pass has its own bracket: the per-pass times are
 * those of the unfused sequence, not of the production path (time that one from outside, as bench.py does). */
int frs_profile_enable(frs_ctx* ctx, int on);
/* Debug aid (compute-sanitizer is not available on every pool): with the environment variable FRS_GUARD=1 set when
 * frs_create runs, every array the context owns is allocated between two 4 KB guard zones filled with a byte pattern.
 * Returns the number of arrays whose guard zones have been written to (0 = clean; -1 on error), *n_arrays (may be NULL) the
 * number of arrays under guard (0 without FRS_GUARD).  Synchronises the device. */
int frs_debug_check_guards(frs_ctx* ctx, int* n_arrays);
int frs_profile_read(frs_ctx* ctx, double ms[5], long long launches[5]);

/* ---- self-test of host-replayable index logic (no GPU needed) -------------------------------- */

/* Replays the register/shared-memory FFT stage logic thread by thread on the CPU for an n-point
 * transform (n a power of two in [16, 4096]); in/out: interleaved complex float [n]. */
int frs_selftest_fft_host(int n, int inverse, const float* in, float* out);
/* The same for the second FFT core (csrc/fft_dif.cuh: forward decimated in frequency, inverse decimated in
 * time, spectrum in a permuted order), n a power of two in [256, 4096].  Forward: natural order in, the
 * permuted spectrum sorted to natural order out; inverse: natural frequency order in, natural time order out. */
int frs_selftest_dif_host(int n, int inverse, const float* in, float* out);
/* Lane-by-lane analysis of that core's shared-memory exchange over two consecutive columns.  out (HOST int[6]):
 * worst bank-conflict degree of any 128-bit access (1 = none), number of cross-thread read/write hazards not
 * ordered by a barrier (block barrier, or warp sync between lanes of one warp), out-of-range slots, slots
 * used, slots allocated, defects of the register <-> frequency map (0 = bijection). */
int frs_selftest_dif_exchange(int n, int* out);
/* Geometry of the TMA tensor copies that feed the row and column passes (csrc/tmap.h), for rows of nf
 * bins and columns of `rows` samples (powers of two, nf >= 16, rows >= 32; else FRS_EINVAL).  out (HOST
 * int[6]): bins per row-gather copy, copies per row pair, row pairs per column copy, copies per column,
 * 16-byte slots of the exchange buffer the row gather lands in, 1 if rows of nf bins use TMA. */
int frs_selftest_tma_geometry(int nf, int rows, int* out);

/* The tensor-core measurement north_star asks for before a DFT-as-GEMM stage may be used (needs a GPU; FRS_ECUDA without):
 * SM cycles per tcgen05.mma kind::tf32 instruction of shape M = 128, K = 8, N = n_out (32 or 64), operands in shared
 * memory, accumulator in TMEM, one CTA per SM, `mmas_per_commit` instructions per commit/wait, `iters` repetitions.
 * A radix-16 stage of one column pair with the 3-term TF32 split is 24 such instructions at N = 64. */
int frs_selftest_tcgen05_stage(int n_out, int mmas_per_commit, int iters, double* clk_per_mma);

#ifdef __cplusplus
}
#endif
#endif /* FRS_H */
