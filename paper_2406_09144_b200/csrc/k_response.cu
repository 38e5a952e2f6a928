// k_response.cu -- exact (ungridded) response on a list of uv points, by direct sums: the major cycle of Alg. 1
// (Eq. 20-22; Eq. 1 for a coplanar array; reading R16).
//   R x       : V_k = sum_pixels x[y][x] exp(-2 pi i (u_k x / Mx + v_k y / My))                 (exact_degrid)
//   R^+ N^-1 V: img[y][x] = sum_k 2 w_k Re(V_k exp(+2 pi i (u_k x / Mx + v_k y / My)))          (exact_grid)
// (u, v) in cell units of the padded grid, not rounded to cells.  Both sums use the separability of the plane wave
// (per visibility nx + ny phase factors instead of nx ny), phases reduced in fp64 before the fp32 sincospi, fp64
// accumulation across rows / visibilities.  Cost O(nvis npix): meant for the sizes of configs 1-2 (a production major
// cycle at 4096^2 needs a gridder, SURVEY 2.1 -- out of scope).
#include <cuda_runtime.h>
#include "response.h"

namespace frs {

// exp(i pi t) for a phase of t half-turns given in fp64
__device__ __forceinline__ float2 cis_pi(double t) {
    t -= 2.0 * rint(0.5 * t);
    float s, c;
    sincospif((float)t, &s, &c);
    return make_float2(c, s);
}

constexpr int kVB = 4;        // visibilities per block (degrid)
constexpr int kRespThreads = 256;

// grid: ceil(nvis / kVB); dynamic smem: kVB (nx + ny) float2
__global__ void __launch_bounds__(kRespThreads) exact_degrid_kernel(const float2* __restrict__ uv, int nvis, const float* __restrict__ img,
                                                                    int ny, int nx, float2* __restrict__ vis) {
    extern __shared__ float2 ph[];
    float2* ex = ph;                       // [kVB][nx]
    float2* ey = ph + kVB * nx;            // [kVB][ny]
    const int k0 = blockIdx.x * kVB;
    const double ifx = -2.0 / (2.0 * nx), ify = -2.0 / (2.0 * ny);
    for (int i = threadIdx.x; i < kVB * nx; i += blockDim.x) {
        const int v = i / nx, x = i - v * nx;
        ex[i] = k0 + v < nvis ? cis_pi(ifx * (double)uv[k0 + v].x * x) : make_float2(0.f, 0.f);
    }
    for (int i = threadIdx.x; i < kVB * ny; i += blockDim.x) {
        const int v = i / ny, y = i - v * ny;
        ey[i] = k0 + v < nvis ? cis_pi(ify * (double)uv[k0 + v].y * y) : make_float2(0.f, 0.f);
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
    double tr[kVB], ti[kVB];
#pragma unroll
    for (int v = 0; v < kVB; ++v) tr[v] = ti[v] = 0.0;
    for (int y = warp; y < ny; y += nwarp) {
        float pr[kVB], pi[kVB];
#pragma unroll
        for (int v = 0; v < kVB; ++v) pr[v] = pi[v] = 0.f;
        const float* row = img + (size_t)y * nx;
        for (int x = lane; x < nx; x += 32) {
            const float a = row[x];
#pragma unroll
            for (int v = 0; v < kVB; ++v) {
                const float2 e = ex[v * nx + x];
                pr[v] = fmaf(a, e.x, pr[v]);
                pi[v] = fmaf(a, e.y, pi[v]);
            }
        }
#pragma unroll
        for (int v = 0; v < kVB; ++v) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                pr[v] += __shfl_down_sync(0xffffffffu, pr[v], o);
                pi[v] += __shfl_down_sync(0xffffffffu, pi[v], o);
            }
            if (lane == 0) {
                const float2 e = ey[v * ny + y];
                tr[v] += (double)pr[v] * e.x - (double)pi[v] * e.y;
                ti[v] += (double)pr[v] * e.y + (double)pi[v] * e.x;
            }
        }
    }
    __shared__ double red[kRespThreads / 32][kVB][2];
    if (lane == 0)
#pragma unroll
        for (int v = 0; v < kVB; ++v) { red[warp][v][0] = tr[v]; red[warp][v][1] = ti[v]; }
    __syncthreads();
    if (threadIdx.x < kVB && k0 + threadIdx.x < nvis) {
        double sr = 0.0, si = 0.0;
        for (int w = 0; w < nwarp; ++w) { sr += red[w][threadIdx.x][0]; si += red[w][threadIdx.x][1]; }
        vis[k0 + threadIdx.x] = make_float2((float)sr, (float)si);
    }
}

constexpr int kTile = 32, kKC = 64;
// grid: (ceil(nx/32), ceil(ny/32)); block 256 = 32 (x) x 8 (y), 4 rows per thread
__global__ void __launch_bounds__(kRespThreads) exact_grid_kernel(const float2* __restrict__ uv, const float* __restrict__ wgt,
                                                                  const float2* __restrict__ vis, int nvis, int ny, int nx,
                                                                  const float* __restrict__ base, float sign, float* __restrict__ out) {
    __shared__ float2 cx[kKC][kTile];      // exp(+2 pi i u x / Mx)
    __shared__ float2 cy[kKC][kTile];      // 2 w V exp(+2 pi i v y / My)
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int x0 = blockIdx.x * kTile, y0 = blockIdx.y * kTile;
    const double ifx = 2.0 / (2.0 * nx), ify = 2.0 / (2.0 * ny);
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (int kc = 0; kc < nvis; kc += kKC) {
        __syncthreads();
        for (int i = threadIdx.x; i < kKC * kTile; i += blockDim.x) {
            const int kk = i / kTile, t = i - kk * kTile, k = kc + kk;
            if (k < nvis) {
                const float2 p = uv[k];
                cx[kk][t] = cis_pi(ifx * (double)p.x * (x0 + t));
                const float2 e = cis_pi(ify * (double)p.y * (y0 + t)), v = vis[k];
                const float w2 = 2.0f * wgt[k];
                cy[kk][t] = make_float2(w2 * (v.x * e.x - v.y * e.y), w2 * (v.x * e.y + v.y * e.x));
            } else {
                cx[kk][t] = cy[kk][t] = make_float2(0.f, 0.f);
            }
        }
        __syncthreads();
        float part[4] = {0.f, 0.f, 0.f, 0.f};     // one chunk in fp32, chunks accumulated in fp64
#pragma unroll 8
        for (int kk = 0; kk < kKC; ++kk) {
            const float2 a = cx[kk][tx];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float2 b = cy[kk][ty + 8 * j];
                part[j] = fmaf(b.x, a.x, fmaf(-b.y, a.y, part[j]));
            }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[j] += (double)part[j];
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int x = x0 + tx, y = y0 + ty + 8 * j;
        if (x < nx && y < ny) {
            const size_t i = (size_t)y * nx + x;
            out[i] = (float)((base ? (double)base[i] : 0.0) + (double)sign * acc[j]);
        }
    }
}

int launch_exact_degrid(cudaStream_t st, const float* uv, int nvis, const float* img, int ny, int nx, float* vis) {
    const int smem = kVB * (nx + ny) * (int)sizeof(float2);
    static int cache[64] = {};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return (int)cudaErrorInvalidDevice;
    if (!cache[dev]) {
        cudaError_t e = cudaFuncSetAttribute(exact_degrid_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kVB * 2048 * (int)sizeof(float2));
        if (e != cudaSuccess) return (int)e;
        cache[dev] = 1;
    }
    exact_degrid_kernel<<<(nvis + kVB - 1) / kVB, kRespThreads, smem, st>>>(reinterpret_cast<const float2*>(uv), nvis, img, ny, nx,
                                                                           reinterpret_cast<float2*>(vis));
    return (int)cudaGetLastError();
}
int launch_exact_grid(cudaStream_t st, const float* uv, const float* wgt, const float* vis, int nvis, int ny, int nx,
                      const float* base, float sign, float* out) {
    dim3 grid((nx + kTile - 1) / kTile, (ny + kTile - 1) / kTile);
    exact_grid_kernel<<<grid, kRespThreads, 0, st>>>(reinterpret_cast<const float2*>(uv), wgt, reinterpret_cast<const float2*>(vis), nvis,
                                                     ny, nx, base, sign, out);
    return (int)cudaGetLastError();
}

}  // namespace frs
