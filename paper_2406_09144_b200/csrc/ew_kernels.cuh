// ew_kernels.cuh -- elementwise maps, deterministic single-order reductions and the CG vector
// updates.  All reductions: fp64 products and sums, one partial per
// CTA written to a buffer, summed afterwards in a fixed order by one CTA (no float atomics), so a
// result does not depend on scheduling.
#pragma once
#include <cuda_runtime.h>

namespace frs {

constexpr int kEwThreads = 256;
constexpr int kRedThreads = 256;

__device__ __forceinline__ double block_sum(double x) {
    __shared__ double red[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) red[w] = x;
    __syncthreads();
    double y = 0.0;
    if (w == 0) {
        const int nw = blockDim.x >> 5;
        y = l < nw ? red[l] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) y += __shfl_down_sync(0xffffffffu, y, o);
    }
    return y;   // valid in thread 0
}

// s[c][i] = exp(tau0[i] + lognu[c] tau1[i])   (tau already contains mu; reading R6)
__global__ void sky_kernel(const float* __restrict__ tau, const float* __restrict__ lognu, float* __restrict__ s,
                           size_t npix, int nfield, int nchan) {
    const size_t i4 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i4 * 4 >= npix) return;
    const float4 t0 = reinterpret_cast<const float4*>(tau)[i4];
    float4 t1 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (nfield == 2) t1 = reinterpret_cast<const float4*>(tau + npix)[i4];
    for (int c = 0; c < nchan; ++c) {
        const float l = nfield == 2 ? lognu[c] : 0.f;
        float4 o;
        o.x = expf(fmaf(l, t1.x, t0.x)); o.y = expf(fmaf(l, t1.y, t0.y));
        o.z = expf(fmaf(l, t1.z, t0.z)); o.w = expf(fmaf(l, t1.w, t0.w));
        reinterpret_cast<float4*>(s + (size_t)c * npix)[i4] = o;
    }
}

// img[c][i] = s[c][i] (lin0[i] + lognu[c] lin1[i])      (J v without the Hartley map)
__global__ void jvp_combine_kernel(const float* __restrict__ lin, const float* __restrict__ s,
                                   const float* __restrict__ lognu, float* __restrict__ img,
                                   size_t npix, int nfield, int nchan) {
    const size_t i4 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i4 * 4 >= npix) return;
    const float4 t0 = reinterpret_cast<const float4*>(lin)[i4];
    float4 t1 = make_float4(0.f, 0.f, 0.f, 0.f);
    if (nfield == 2) t1 = reinterpret_cast<const float4*>(lin + npix)[i4];
    for (int c = 0; c < nchan; ++c) {
        const float l = nfield == 2 ? lognu[c] : 0.f;
        const float4 sv = reinterpret_cast<const float4*>(s + (size_t)c * npix)[i4];
        float4 o;
        o.x = sv.x * fmaf(l, t1.x, t0.x); o.y = sv.y * fmaf(l, t1.y, t0.y);
        o.z = sv.z * fmaf(l, t1.z, t0.z); o.w = sv.w * fmaf(l, t1.w, t0.w);
        reinterpret_cast<float4*>(img + (size_t)c * npix)[i4] = o;
    }
}

// acc[f][i] = sum_c coeff[c][f] img[c][i], channels summed in index order   (J^T without H, A)
__global__ void vjp_combine_kernel(const float* __restrict__ img, const float* __restrict__ lognu,
                                   float* __restrict__ acc, size_t npix, int nfield, int nchan) {
    const size_t i4 = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i4 * 4 >= npix) return;
    float4 a0 = make_float4(0.f, 0.f, 0.f, 0.f), a1 = a0;
    for (int c = 0; c < nchan; ++c) {
        const float4 w = reinterpret_cast<const float4*>(img + (size_t)c * npix)[i4];
        a0.x += w.x; a0.y += w.y; a0.z += w.z; a0.w += w.w;
        if (nfield == 2) {
            const float l = lognu[c];
            a1.x = fmaf(l, w.x, a1.x); a1.y = fmaf(l, w.y, a1.y); a1.z = fmaf(l, w.z, a1.z); a1.w = fmaf(l, w.w, a1.w);
        }
    }
    reinterpret_cast<float4*>(acc)[i4] = a0;
    if (nfield == 2) reinterpret_cast<float4*>(acc + npix)[i4] = a1;
}

// partials[blockIdx.x] = sum over this CTA's slice of a[i] b[i]
__global__ void __launch_bounds__(kRedThreads) dot_partial_kernel(const float* __restrict__ a, const float* __restrict__ b,
                                                                  size_t n, double* __restrict__ partials) {
    double acc = 0.0;
    const size_t n4 = n / 4;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        const float4 x = reinterpret_cast<const float4*>(a)[i], y = reinterpret_cast<const float4*>(b)[i];
        acc += (double)x.x * y.x + (double)x.y * y.y + (double)x.z * y.z + (double)x.w * y.w;
    }
    acc = block_sum(acc);
    if (threadIdx.x == 0) partials[blockIdx.x] = acc;
}

// out[k] = scale[k] * sum_{i<n} partials[i*stride + k] for k < nk, fixed order; one CTA.
// Optional combination for the energy:  energy = 0.5*S0 - S1 + 0.5*prior
__global__ void __launch_bounds__(kRedThreads) reduce_final_kernel(const double* __restrict__ partials, int n, int stride,
                                                                   int k, double* __restrict__ out) {
    double acc = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) acc += partials[(size_t)i * stride + k];
    acc = block_sum(acc);
    if (threadIdx.x == 0) *out = acc;
}

// sc: device scalars.  E = 0.5 sc[kSC] - sc[kJS] + 0.5 with_prior sc[kXX]
__global__ void energy_final_kernel(const double* __restrict__ sc_sc, const double* __restrict__ sc_js,
                                    const double* __restrict__ sc_xx, int with_prior, double* __restrict__ e) {
    *e = 0.5 * (*sc_sc) - (*sc_js) + (with_prior ? 0.5 * (*sc_xx) : 0.0);
}

// ---- noise kernel of Eq. 16-17 (reading R14) from the transposed Hartley transform HT[kx][ky] of t = C I_delta, I_delta at
// (ny/2, nx/2):  Re FFT(t)[k] = (H[k] + H[-k]) / 2, conj FFT(I_delta)[k] = (-1)^(ky+kx), + eps from the eps I_delta term:
//   K = max((-1)^(ky+kx) (H[k] + H[-k]) / 2 + eps, eps);   kern[ky][kx] = K;  kinv = 1 / (K ny nx) in both orientations
__global__ void noise_kernel_finish_kernel(const float* __restrict__ ht, float eps, float* __restrict__ kern,
                                           float* __restrict__ kinv_n, float* __restrict__ kinv_t, float* __restrict__ kisq_n,
                                           int ny, int nx) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x, npix = (size_t)ny * nx;
    if (i >= npix) return;
    const size_t b = blockIdx.y * npix;
    const int ky = (int)(i / nx), kx = (int)(i % nx);
    const int my = (ny - ky) % ny, mx = (nx - kx) % nx;
    const float h = ht[b + (size_t)kx * ny + ky], hm = ht[b + (size_t)mx * ny + my];
    const float sgn = ((ky + kx) & 1) ? -1.f : 1.f;
    const float k = fmaxf(fmaf(sgn * 0.5f, h + hm, eps), eps);
    kern[b + i] = k;
    const float inv = 1.0f / (k * (float)ny * (float)nx);
    kinv_n[b + i] = inv;
    kinv_t[b + (size_t)kx * ny + ky] = inv;
    kisq_n[b + i] = rsqrtf(k) / ((float)ny * (float)nx);          // N'^-1/2 (MGVI sample source, R15)
}
// a caller-supplied kernel: flags non-positive / NaN entries and departures from K[-k] = K[k] beyond 1e-5 max-free relative
__global__ void noise_kernel_from_array_kernel(const float* __restrict__ kern, float* __restrict__ kinv_n,
                                               float* __restrict__ kinv_t, float* __restrict__ kisq_n, int ny, int nx,
                                               int* __restrict__ bad) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x, npix = (size_t)ny * nx;
    if (i >= npix) return;
    const size_t b = blockIdx.y * npix;
    const int ky = (int)(i / nx), kx = (int)(i % nx);
    const float k = kern[b + i], km = kern[b + (size_t)((ny - ky) % ny) * nx + (nx - kx) % nx];
    if (!(k > 0.f) || !(fabsf(k - km) <= 1e-5f * fmaxf(k, km))) atomicExch(bad, 1);
    const float inv = 1.0f / (k * (float)ny * (float)nx);
    kinv_n[b + i] = inv;
    kinv_t[b + (size_t)kx * ny + ky] = inv;
    kisq_n[b + i] = rsqrtf(k) / ((float)ny * (float)nx);
}
// out = x + sgn y  (a position xi +- sigma of the sample-averaged KL), n a multiple of 4
__global__ void __launch_bounds__(kEwThreads) add_scaled_kernel(const float* __restrict__ x, const float* __restrict__ y, float sgn,
                                                                 float* __restrict__ out, size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i * 4 >= n) return;
    const float4 a = reinterpret_cast<const float4*>(x)[i], b = reinterpret_cast<const float4*>(y)[i];
    reinterpret_cast<float4*>(out)[i] = make_float4(fmaf(sgn, b.x, a.x), fmaf(sgn, b.y, a.y), fmaf(sgn, b.z, a.z), fmaf(sgn, b.w, a.w));
}
// acc = (first ? 0 : acc) + w g ;  the energies likewise in fp64: e_acc = (first ? 0 : e_acc) + w e
__global__ void __launch_bounds__(kEwThreads) accumulate_kernel(float* __restrict__ acc, const float* __restrict__ g, float w, int first,
                                                                 size_t n, double* __restrict__ e_acc, const double* __restrict__ e) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0 && e_acc) *e_acc = (first ? 0.0 : *e_acc) + (double)w * (*e);
    if (i * 4 >= n) return;
    const float4 b = reinterpret_cast<const float4*>(g)[i];
    float4 a = first ? make_float4(0.f, 0.f, 0.f, 0.f) : reinterpret_cast<float4*>(acc)[i];
    a.x = fmaf(w, b.x, a.x); a.y = fmaf(w, b.y, a.y); a.z = fmaf(w, b.z, a.z); a.w = fmaf(w, b.w, a.w);
    reinterpret_cast<float4*>(acc)[i] = a;
}
__global__ void set_delta_kernel(float* __restrict__ img, size_t npix, size_t pos) { img[blockIdx.x * npix + pos] = 1.0f; }
// a *= b, n a multiple of 4
__global__ void __launch_bounds__(kEwThreads) mul_inplace_kernel(float* __restrict__ a, const float* __restrict__ b, size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i * 4 >= n) return;
    float4 x = reinterpret_cast<float4*>(a)[i];
    const float4 y = reinterpret_cast<const float4*>(b)[i];
    x.x *= y.x; x.y *= y.y; x.z *= y.z; x.w *= y.w;
    reinterpret_cast<float4*>(a)[i] = x;
}
// E = 0.5 <r, N'^-1 r> + 0.5 with_prior <xi, xi>
__global__ void energy9_final_kernel(const double* __restrict__ ru, const double* __restrict__ xx, int with_prior,
                                     double* __restrict__ e) {
    *e = 0.5 * (*ru) + (with_prior ? 0.5 * (*xx) : 0.0);
}

// ---- CG (reading R9).  scal[0]=rr, [1]=pq, [2]=rr_new, [3]=alpha, [4]=beta, [5]=breakdown flag, [6]=<b,b>, [7]=done flag;
// scal[kIters] = completed iterations.  The stopping test runs on the DEVICE (cg_shift_kernel): once `done` is set the
// vector updates of the iterations still enqueued turn into no-ops, so the host never has to synchronise inside the loop
// and x is exactly the iterate at which the criterion was met.
enum { kRR = 0, kPQ = 1, kRRNew = 2, kAlpha = 3, kBeta = 4, kBreak = 5, kBB = 6, kDone = 7, kNScal = 8, kIters = 12, kStep = 13 };

// r = b - q ; p = r ; partial <r,r>       (q = M x0, or q == nullptr for x0 = 0)
__global__ void __launch_bounds__(kRedThreads) cg_init_kernel(const float* __restrict__ b, const float* __restrict__ q,
                                                              float* __restrict__ r, float* __restrict__ p, size_t n,
                                                              double* __restrict__ partials) {
    double acc = 0.0;
    const size_t n4 = n / 4;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        float4 x = reinterpret_cast<const float4*>(b)[i];
        if (q) {
            const float4 y = reinterpret_cast<const float4*>(q)[i];
            x.x -= y.x; x.y -= y.y; x.z -= y.z; x.w -= y.w;
        }
        reinterpret_cast<float4*>(r)[i] = x;
        reinterpret_cast<float4*>(p)[i] = x;
        acc += (double)x.x * x.x + (double)x.y * x.y + (double)x.z * x.z + (double)x.w * x.w;
    }
    acc = block_sum(acc);
    if (threadIdx.x == 0) partials[blockIdx.x] = acc;
}

// alpha = rr/pq ; x += alpha p ; r -= alpha q ; partial <r,r>
__global__ void __launch_bounds__(kRedThreads) cg_update_xr_kernel(float* __restrict__ x, float* __restrict__ r,
                                                                   const float* __restrict__ p, const float* __restrict__ q,
                                                                   size_t n, double* __restrict__ scal,
                                                                   double* __restrict__ partials) {
    if (scal[kDone] != 0.0) return;               // stopped: x, r and the partial sums stay as they are
    const double pq = scal[kPQ];
    const double alpha_d = pq > 0.0 ? scal[kRR] / pq : 0.0;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        scal[kAlpha] = alpha_d;
        if (!(pq > 0.0)) scal[kBreak] = 1.0;
    }
    const float alpha = (float)alpha_d;
    double acc = 0.0;
    const size_t n4 = n / 4;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        float4 xv = reinterpret_cast<float4*>(x)[i], rv = reinterpret_cast<float4*>(r)[i];
        const float4 pv = reinterpret_cast<const float4*>(p)[i], qv = reinterpret_cast<const float4*>(q)[i];
        xv.x = fmaf(alpha, pv.x, xv.x); xv.y = fmaf(alpha, pv.y, xv.y); xv.z = fmaf(alpha, pv.z, xv.z); xv.w = fmaf(alpha, pv.w, xv.w);
        rv.x = fmaf(-alpha, qv.x, rv.x); rv.y = fmaf(-alpha, qv.y, rv.y); rv.z = fmaf(-alpha, qv.z, rv.z); rv.w = fmaf(-alpha, qv.w, rv.w);
        reinterpret_cast<float4*>(x)[i] = xv;
        reinterpret_cast<float4*>(r)[i] = rv;
        acc += (double)rv.x * rv.x + (double)rv.y * rv.y + (double)rv.z * rv.z + (double)rv.w * rv.w;
    }
    acc = block_sum(acc);
    if (threadIdx.x == 0) partials[blockIdx.x] = acc;
}

// beta = rr_new/rr ; p = r + beta p ; then rr <- rr_new (done by the last-launched thread 0 after use)
__global__ void __launch_bounds__(kEwThreads) cg_update_p_kernel(float* __restrict__ p, const float* __restrict__ r, size_t n,
                                                                 const double* __restrict__ scal, double* __restrict__ beta_out) {
    if (scal[kDone] != 0.0) return;
    const double rr = scal[kRR];
    const double beta_d = rr > 0.0 ? scal[kRRNew] / rr : 0.0;
    if (blockIdx.x == 0 && threadIdx.x == 0) *beta_out = beta_d;
    const float beta = (float)beta_d;
    const size_t n4 = n / 4;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        const float4 rv = reinterpret_cast<const float4*>(r)[i];
        float4 pv = reinterpret_cast<float4*>(p)[i];
        pv.x = fmaf(beta, pv.x, rv.x); pv.y = fmaf(beta, pv.y, rv.y); pv.z = fmaf(beta, pv.z, rv.z); pv.w = fmaf(beta, pv.w, rv.w);
        reinterpret_cast<float4*>(p)[i] = pv;
    }
}

// q += p (prior term of the metric, added after the cross-rank sum of the likelihood part)
__global__ void __launch_bounds__(kEwThreads) add_inplace_kernel(float* __restrict__ q, const float* __restrict__ p, size_t n) {
    const size_t i = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) * 4;
    if (i + 3 < n) {
        float4 a = *reinterpret_cast<float4*>(q + i);
        const float4 b = *reinterpret_cast<const float4*>(p + i);
        a.x += b.x; a.y += b.y; a.z += b.z; a.w += b.w;
        *reinterpret_cast<float4*>(q + i) = a;
    } else {
        for (size_t j = i; j < n; ++j) q[j] += p[j];
    }
}
// end of iteration k (k = 0: initialisation): rr <- rr_new, count it, and decide whether to stop:
// ||r||^2 <= rtol2 <b,b>  (rtol2 = 0: never)  or  breakdown <p, M p> <= 0.
// k < 0: the iteration index is the device-side counter scal[kStep] + 1, so that one captured iteration (a CUDA graph
// whose kernel arguments are frozen) can be replayed for every k.
__global__ void cg_shift_kernel(double* __restrict__ scal, double* __restrict__ hist, int k, double rtol2) {
    if (k < 0) k = (int)scal[kStep] + 1;
    scal[kStep] = (double)k;
    if (scal[kDone] == 0.0) {
        scal[kRR] = scal[kRRNew];
        scal[kIters] = (double)k;
        if (scal[kBreak] != 0.0 || (rtol2 > 0.0 && scal[kRRNew] <= rtol2 * scal[kBB])) scal[kDone] = 1.0;
    }
    if (hist) hist[k] = sqrt(scal[kRR]);
}

}  // namespace frs
