// kernels.cuh -- the FFT passes of the fast-resolve hot path.
//
// Data layouts:
//   image      real  [nb][ny][nx]                      row-major, x fastest
//   spectrum T cplx  [nb][ntile][ny][2]                column-pair tiles: tile m holds columns
//                                                       kx = 2m, 2m+1 of the row-transformed
//                                                       array, ntile = NF/2 + 1 (kx = 0..NF; the
//                                                       odd slot of the last tile is zero)
//   weights Wt real  [nb][ntile][2][ny][2]             parity (even/odd ky), q, column-in-tile
//
// Passes:
//   rows_fwd   real rows -> half spectrum (R2C through a half-length complex FFT), PAD = the row
//              is zero-extended nx -> 2 nx (Eq. 14 'FFT[P I]'), optional fused multiply
//   conv_cols  per column: zero-padded FFT (even/odd split) . W . inverse FFT, cropped (Eq. 14)
//   rows_inv   half spectrum -> real rows, cropped to the first nx samples (P:182 'P^dagger'),
//              fused epilogues (x s, energy/residual)
//   hart_cols  second pass of the 2-D Hartley transform of the correlated field (reading R6)
#pragma once
#include "fft_core.cuh"

namespace frs {

template <int NF, int ROLES>
struct Geo {
    static constexpr int P = NF / kE;                                  // threads per transform pair
    static constexpr int GT = P * ROLES;                               // threads per group
    static constexpr int THREADS = GT >= 64 ? GT : 64;
    static constexpr int G = THREADS / GT;                             // groups per CTA
    static constexpr int SMEM = G * ROLES * 2 * xbuf_len(NF) * (int)sizeof(float2);
};

__device__ __forceinline__ float2 ldg2(const float* p) { return __ldg(reinterpret_cast<const float2*>(p)); }
__device__ __forceinline__ float4 ldg4(const void* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

// ------------------------------------------------------------------------------------------------
struct RowsFwdArgs {
    const float* in;      // [nb][ny][nxr]
    const float* mul;     // optional [nb or 1][ny][nxr] multiplier (s or A); nullptr = none
    float2* out;          // [nb][ntile][ny][2]
    int ny;               // rows
    size_t in_bstride, mul_bstride, out_bstride;   // elements (float / float / float2)
    float scale;
    const float2* tw;     // stage twiddles for NF
    const float2* twist;  // exp(-2 pi i k/(2 NF)), k = 0..NF
};

// One group (P threads) transforms rows y0, y0+1 together (two transforms per thread share the
// twiddle fetches and turn the 16-byte tile slots into 32-byte sectors).
template <int NF, bool PAD>
__global__ void __launch_bounds__(Geo<NF, 1>::THREADS, (Geo<NF, 1>::THREADS >= 256 ? 2 : 4))
rows_fwd_kernel(RowsFwdArgs a) {
    using GEO = Geo<NF, 1>;
    constexpr int P = GEO::P;
    constexpr int NXR = PAD ? NF : 2 * NF;        // real samples per row
    constexpr int NE = PAD ? kE / 2 : kE;         // canonical slots that hold data
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / P, p = threadIdx.x % P;
    float2* bufs = smem + (size_t)g * 2 * xbuf_len(NF);
    const int rp = blockIdx.x * GEO::G + g;       // row pair
    const int b = blockIdx.y;
    const bool live = 2 * rp < a.ny;
    const int y0 = 2 * rp;

    float2 v[2][kE];
#pragma unroll
    for (int e = 0; e < kE; ++e) { v[0][e] = make_float2(0.f, 0.f); v[1][e] = make_float2(0.f, 0.f); }
    if (live) {
        const float* r0 = a.in + b * a.in_bstride + (size_t)y0 * NXR;
#pragma unroll
        for (int e = 0; e < NE; ++e) {
            const int n = p + e * P;
            v[0][e] = ldg2(r0 + 2 * n);
            v[1][e] = ldg2(r0 + NXR + 2 * n);
        }
        if (a.mul) {
            const float* m0 = a.mul + b * a.mul_bstride + (size_t)y0 * NXR;
#pragma unroll
            for (int e = 0; e < NE; ++e) {
                const int n = p + e * P;
                float2 ma = ldg2(m0 + 2 * n), mb = ldg2(m0 + NXR + 2 * n);
                v[0][e].x *= ma.x; v[0][e].y *= ma.y;
                v[1][e].x *= mb.x; v[1][e].y *= mb.y;
            }
        }
    }
    group_fft<NF, false, 2>(v, p, bufs, a.tw);
    canon_scatter<NF>(v[0], p, bufs);
    canon_scatter<NF>(v[1], p, bufs + xbuf_len(NF));
    __syncthreads();
    if (live) {
        // X[k] * (scale) = (Z[k] + conj Z[NF-k]) - i twist[k] (Z[k] - conj Z[NF-k]),  k = 0..NF
        constexpr int NTILE = NF / 2 + 1;
        float4* ob = reinterpret_cast<float4*>(a.out + b * a.out_bstride);
        for (int m = p; m < NTILE; m += P) {
            float2 res[2][2];
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                const int k = 2 * m + c;
                const int ik = k & (NF - 1), im = (NF - k) & (NF - 1);
                const float2 w = (k <= NF) ? __ldg(a.twist + k) : make_float2(0.f, 0.f);
#pragma unroll
                for (int t = 0; t < 2; ++t) {
                    const float2* zb = bufs + t * xbuf_len(NF);
                    const float2 za = zb[xpad(ik)], zm = cconj(zb[xpad(im)]);
                    const float2 s = cadd(za, zm), d = cmul(csub(za, zm), w);
                    float2 x = make_float2((s.x + d.y) * a.scale, (s.y - d.x) * a.scale);
                    if (k > NF) x = make_float2(0.f, 0.f);
                    res[t][c] = x;
                }
            }
            float4* o = ob + (size_t)m * a.ny + y0;
            o[0] = make_float4(res[0][0].x, res[0][0].y, res[0][1].x, res[0][1].y);
            o[1] = make_float4(res[1][0].x, res[1][0].y, res[1][1].x, res[1][1].y);
        }
    }
}

// ------------------------------------------------------------------------------------------------
struct ConvColsArgs {
    float2* t;            // [nb][ntile][NF][2] in place
    const float* wt;      // [nb][ntile][2][NF][2]
    int ntile;
    size_t t_bstride, w_bstride;
    const float2* tw;
    const float2* twist;  // exp(-2 pi i n/(2 NF))
};

// Group = 2 roles x P threads; role 0 owns the even output bins of the length-2NF transform of the
// zero-extended column, role 1 the odd bins (input pre-multiplied by twist^n).  After . W and the
// inverse transforms:  y[n] = IFFT_NF(E')[n] + conj(twist^n) IFFT_NF(O')[n].
template <int NF>
__global__ void __launch_bounds__(Geo<NF, 2>::THREADS, (Geo<NF, 2>::THREADS >= 512 ? 1 : 2))
conv_cols_kernel(ConvColsArgs a) {
    using GEO = Geo<NF, 2>;
    constexpr int P = GEO::P;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / (2 * P), role = (threadIdx.x / P) & 1, p = threadIdx.x % P;
    float2* gb = smem + (size_t)g * 4 * xbuf_len(NF);
    float2* bufs = gb + role * 2 * xbuf_len(NF);
    const int m = blockIdx.x * GEO::G + g;
    const int b = blockIdx.y;
    const bool live = m < a.ntile;

    float2 v[2][kE];
    float4* tile = reinterpret_cast<float4*>(a.t + b * a.t_bstride) + (size_t)m * NF;
    if (live) {
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const float4 x = ldg4(tile + p + e * P);
            v[0][e] = make_float2(x.x, x.y);
            v[1][e] = make_float2(x.z, x.w);
        }
        if (role) {
#pragma unroll
            for (int e = 0; e < kE; ++e) {
                const float2 w = __ldg(a.twist + p + e * P);
                v[0][e] = cmul(v[0][e], w);
                v[1][e] = cmul(v[1][e], w);
            }
        }
    } else {
#pragma unroll
        for (int e = 0; e < kE; ++e) { v[0][e] = make_float2(0.f, 0.f); v[1][e] = make_float2(0.f, 0.f); }
    }
    group_fft<NF, false, 2>(v, p, bufs, a.tw);
    if (live) {
        const float2* w = reinterpret_cast<const float2*>(a.wt + b * a.w_bstride) + ((size_t)m * 2 + role) * NF;
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const float2 ww = __ldg(w + p + e * P);
            v[0][e] = cscale(v[0][e], ww.x);
            v[1][e] = cscale(v[1][e], ww.y);
        }
    }
    group_fft<NF, true, 2>(v, p, bufs, a.tw);
    // combine the two roles through role 1's (now idle) exchange buffers: [transform][e][p]
    float2* cb = gb + 2 * xbuf_len(NF);
    if (role) {
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const float2 w = __ldg(a.twist + p + e * P);
            cb[e * P + p] = cmulc(v[0][e], w);
            cb[xbuf_len(NF) + e * P + p] = cmulc(v[1][e], w);
        }
    }
    __syncthreads();
    if (!role && live) {
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const float2 o0 = cb[e * P + p], o1 = cb[xbuf_len(NF) + e * P + p];
            tile[p + e * P] = make_float4(v[0][e].x + o0.x, v[0][e].y + o0.y, v[1][e].x + o1.x, v[1][e].y + o1.y);
        }
    }
}

// ------------------------------------------------------------------------------------------------
enum RowsInvMode { kPlain = 0, kMulS = 1, kEnergy = 2 };

struct RowsInvArgs {
    const float2* t;      // [nb][ntile][ny][2]
    float* out;           // [nb][ny][NF]
    const float* s;       // [nb][ny][NF]  (kMulS, kEnergy)
    const float* j;       // [nb][ny][NF]  (kEnergy)
    double* partials;     // [gridDim.y][gridDim.x][2]  (kEnergy): sum s*c, sum j*s
    int ny, mode;
    size_t t_bstride, img_bstride;
    const float2* tw;
    const float2* twist;
};

template <int NF>
__global__ void __launch_bounds__(Geo<NF, 1>::THREADS, (Geo<NF, 1>::THREADS >= 256 ? 2 : 4))
rows_inv_kernel(RowsInvArgs a) {
    using GEO = Geo<NF, 1>;
    constexpr int P = GEO::P;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / P, p = threadIdx.x % P;
    float2* bufs = smem + (size_t)g * 2 * xbuf_len(NF);
    const int rp = blockIdx.x * GEO::G + g;
    const int b = blockIdx.y;
    const bool live = 2 * rp < a.ny;
    const int y0 = 2 * rp;
    constexpr int NTILE = NF / 2 + 1;

    if (live) {
        const float4* tb = reinterpret_cast<const float4*>(a.t + b * a.t_bstride);
        for (int m = p; m < NTILE; m += P) {
            const float4* q = tb + (size_t)m * a.ny + y0;
            const float4 r0 = ldg4(q), r1 = ldg4(q + 1);
            const int k = 2 * m;
            bufs[xpad(k)] = make_float2(r0.x, r0.y);
            bufs[xbuf_len(NF) + xpad(k)] = make_float2(r1.x, r1.y);
            if (k + 1 <= NF) {
                bufs[xpad(k + 1)] = make_float2(r0.z, r0.w);
                bufs[xbuf_len(NF) + xpad(k + 1)] = make_float2(r1.z, r1.w);
            }
        }
    }
    __syncthreads();
    // Z'[k] = (Y[k] + conj Y[NF-k]) + i conj(twist[k]) (Y[k] - conj Y[NF-k]),  k = 0..NF-1
    float2 v[2][kE];
#pragma unroll
    for (int e = 0; e < kE; ++e) {
        const int k = p + e * P;
        const float2 w = __ldg(a.twist + k);
#pragma unroll
        for (int t = 0; t < 2; ++t) {
            const float2* yb = bufs + t * xbuf_len(NF);
            float2 ya = make_float2(0.f, 0.f), ym = ya;
            if (live) { ya = yb[xpad(k)]; ym = cconj(yb[xpad(NF - k)]); }
            const float2 s = cadd(ya, ym), d = cmulc(csub(ya, ym), w);
            v[t][e] = make_float2(s.x - d.y, s.y + d.x);
        }
    }
    __syncthreads();
    group_fft<NF, true, 2>(v, p, bufs, a.tw);

    double acc_sc = 0.0, acc_js = 0.0;
    if (live) {
#pragma unroll
        for (int t = 0; t < 2; ++t) {
            const size_t row = b * a.img_bstride + (size_t)(y0 + t) * NF;
#pragma unroll
            for (int e = 0; e < kE / 2; ++e) {
                const int n = p + e * P;
                float2 c = v[t][e];
                if (a.mode == kMulS) {
                    const float2 s = ldg2(a.s + row + 2 * n);
                    c.x *= s.x; c.y *= s.y;
                } else if (a.mode == kEnergy) {
                    const float2 s = ldg2(a.s + row + 2 * n), j = ldg2(a.j + row + 2 * n);
                    acc_sc += (double)(s.x * c.x) + (double)(s.y * c.y);
                    acc_js += (double)(j.x * s.x) + (double)(j.y * s.y);
                    c.x = s.x * (c.x - j.x); c.y = s.y * (c.y - j.y);
                }
                *reinterpret_cast<float2*>(a.out + row + 2 * n) = c;
            }
        }
    }
    if (a.mode == kEnergy) {
        // fixed-order block reduction: warp shuffle tree, then warp 0 over the per-warp sums
        __shared__ double red[2][32];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            acc_sc += __shfl_down_sync(0xffffffffu, acc_sc, o);
            acc_js += __shfl_down_sync(0xffffffffu, acc_js, o);
        }
        const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
        if (l == 0) { red[0][w] = acc_sc; red[1][w] = acc_js; }
        __syncthreads();
        if (w == 0) {
            const int nw = blockDim.x >> 5;
            double x = l < nw ? red[0][l] : 0.0, y = l < nw ? red[1][l] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                x += __shfl_down_sync(0xffffffffu, x, o);
                y += __shfl_down_sync(0xffffffffu, y, o);
            }
            if (l == 0) {
                double* ps = a.partials + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * 2;
                ps[0] = x; ps[1] = y;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
struct HartColsArgs {
    const float2* t;      // [nb][ntile][NF][2], columns x = 0..nx/2 of the row-transformed field
    float* out;           // [nb][NF][nx]
    const float* mul;     // optional [nb][NF][nx]: out = mul * H + add
    const float* add;     // optional [nb][NF][nx]
    const float* offset;  // optional device [nb]: out = H + offset[b]   (mu)
    int nx;
    size_t t_bstride, img_bstride;
    const float2* tw;
};

// F[y][x] = column FFT; H[y][x] = Re F - Im F and H[(-y) mod ny][nx - x] = Re F + Im F  (reading R6)
template <int NF>
__global__ void __launch_bounds__(Geo<NF, 1>::THREADS, (Geo<NF, 1>::THREADS >= 256 ? 2 : 4))
hart_cols_kernel(HartColsArgs a) {
    using GEO = Geo<NF, 1>;
    constexpr int P = GEO::P;
    extern __shared__ float2 smem[];
    const int g = threadIdx.x / P, p = threadIdx.x % P;
    float2* bufs = smem + (size_t)g * 2 * xbuf_len(NF);
    const int ntile = a.nx / 4 + 1;
    const int m = blockIdx.x * GEO::G + g;
    const int b = blockIdx.y;
    const bool live = m < ntile;

    float2 v[2][kE];
    if (live) {
        const float4* tile = reinterpret_cast<const float4*>(a.t + b * a.t_bstride) + (size_t)m * NF;
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const float4 x = ldg4(tile + p + e * P);
            v[0][e] = make_float2(x.x, x.y);
            v[1][e] = make_float2(x.z, x.w);
        }
    } else {
#pragma unroll
        for (int e = 0; e < kE; ++e) { v[0][e] = make_float2(0.f, 0.f); v[1][e] = make_float2(0.f, 0.f); }
    }
    group_fft<NF, false, 2>(v, p, bufs, a.tw);
    if (live) {
        const size_t base = b * a.img_bstride;
        const float off = a.offset ? __ldg(a.offset + b) : 0.f;
        const int half = a.nx / 2;
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const int y = p + e * P, ym = (NF - y) & (NF - 1);
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                const int x = 2 * m + c;
                if (x > half) continue;
                const float2 f = v[c][e];
                size_t i0 = base + (size_t)y * a.nx + x;
                float h0 = f.x - f.y + off;
                if (a.mul) h0 *= __ldg(a.mul + i0);
                if (a.add) h0 += __ldg(a.add + i0);
                a.out[i0] = h0;
                if (x > 0 && x < half) {
                    size_t i1 = base + (size_t)ym * a.nx + (a.nx - x);
                    float h1 = f.x + f.y + off;
                    if (a.mul) h1 *= __ldg(a.mul + i1);
                    if (a.add) h1 += __ldg(a.add + i1);
                    a.out[i1] = h1;
                }
            }
        }
    }
}

}  // namespace frs
