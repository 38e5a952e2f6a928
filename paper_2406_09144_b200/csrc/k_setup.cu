// k_setup.cu -- untimed setup: PSF -> weight-spectrum layout (P:180 'FFT[I^PSF]' precomputed)
#include "launch.h"
#include "setup.h"
namespace frs {

// Column pass of the full (not zero-padded) 2NF-point DFT of the row-transformed PSF by one
// decimation-in-frequency step: even bins = FFT_NF(x[n] + x[n+NF]), odd = FFT_NF((x[n] - x[n+NF]) twist^n).
template <int NF>
__global__ void __launch_bounds__(Geo<NF, 2>::THREADS, Geo<NF, 2>::MINB)
psf_cols_kernel(PsfColsArgs a) {
    using GEO = Geo<NF, 2>;
    constexpr int P = GEO::P;
    extern __shared__ __align__(128) float4 smem4[];
    float4* tws = smem4;
    const int g = threadIdx.x / (2 * P), role = (threadIdx.x / P) & 1, p = threadIdx.x % P;
    float4* buf = smem4 + GEO::TW + ((size_t)g * 2 + role) * xbuf_len(NF);
    load_twiddles<NF>(tws, a.tw);
    __syncthreads();
    const int m = blockIdx.x * GEO::G + g;
    const int b = blockIdx.y;
    const bool live = m < a.ntile;
    C2 v[kE];
#pragma unroll
    for (int e = 0; e < kE; ++e) v[e] = c2zero();
    if (live) {
        // columns 2m, 2m+1 of the row-transformed PSF (2 NF rows, block layout of tmap.h)
        const float2* c0 = a.t + b * spec_batch_stride(2 * NF, a.ncols - 1, kPairBins);
        const bool two = 2 * m + 1 < a.ncols;
        auto at = [&](int c, int y) { return ldg2(reinterpret_cast<const float*>(c0 + spec_index(2 * NF, 2 * m + c, y, kPairBins))); };
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const int n = p + e * P;
            const float2 z = make_float2(0.f, 0.f);
            const float2 a0 = at(0, n), a1 = at(0, n + NF);
            const float2 b0 = two ? at(1, n) : z, b1 = two ? at(1, n + NF) : z;
            if (!role) {
                v[e] = c2make(make_float2(a0.x + a1.x, a0.y + a1.y), make_float2(b0.x + b1.x, b0.y + b1.y));
            } else {
                const float2 w = __ldg(a.twist + n);
                v[e] = c2make(cmul(make_float2(a0.x - a1.x, a0.y - a1.y), w), cmul(make_float2(b0.x - b1.x, b0.y - b1.y), w));
            }
        }
    }
    pair_fft<NF, false>(v, p, buf, tws, GEO::bar(g));
    float max_im = 0.f, min_re = 0.f, max_re = 0.f;
    if (live) {
        float* w = a.wt + b * a.w_bstride + (size_t)m * 2 * NF * 2 + role;      // [c][q][parity = role]
#pragma unroll
        for (int e = 0; e < kE; ++e) {
            const float re0 = v[e].re.x * a.scale, re1 = v[e].re.y * a.scale;
            max_im = fmaxf(max_im, fmaxf(fabsf(v[e].im.x), fabsf(v[e].im.y)) * a.scale);
            min_re = fminf(min_re, fminf(re0, re1));
            max_re = fmaxf(max_re, fmaxf(re0, re1));
            w[(size_t)(p + e * P) * 2] = 0.5f * fmaxf(re0, a.floor);
            w[(size_t)(NF + p + e * P) * 2] = 0.5f * fmaxf(re1, a.floor);
        }
    }
    __shared__ float red[3][32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        max_im = fmaxf(max_im, __shfl_down_sync(0xffffffffu, max_im, o));
        min_re = fminf(min_re, __shfl_down_sync(0xffffffffu, min_re, o));
        max_re = fmaxf(max_re, __shfl_down_sync(0xffffffffu, max_re, o));
    }
    const int wid = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) { red[0][wid] = max_im; red[1][wid] = min_re; red[2][wid] = max_re; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < (int)(blockDim.x >> 5); ++i) {
            max_im = fmaxf(max_im, red[0][i]); min_re = fminf(min_re, red[1][i]); max_re = fmaxf(max_re, red[2][i]);
        }
        float* s = a.stats + ((size_t)b * gridDim.x + blockIdx.x) * 3;
        s[0] = max_im; s[1] = min_re; s[2] = max_re;
    }
}

template <int NF>
static int run(cudaStream_t st, const PsfColsArgs& a, int nb, int* grid_x) {
    using GEO = Geo<NF, 2>;
    static int cache[kMaxDevices] = {};
    int unused = 0;
    if (int e = persistent_ctas(cache, psf_cols_kernel<NF>, GEO::THREADS, GEO::SMEM, &unused)) return e;
    dim3 grid((a.ntile + GEO::G - 1) / GEO::G, nb);
    if (grid_x) *grid_x = grid.x;
    if (a.t) psf_cols_kernel<NF><<<grid, GEO::THREADS, GEO::SMEM, st>>>(a);
    return (int)cudaGetLastError();
}
int launch_psf_cols(cudaStream_t st, int nf, const PsfColsArgs& a, int nb, int* grid_x) {
#define CALL(N) return run<N>(st, a, nb, grid_x)
    FRS_DISPATCH_NF(nf, CALL)
#undef CALL
    return 0;
}

// w_half [nb][2ny][nx+1]  ->  wt [nb][ntile][c][q][par] = 0.5 * W[2q+par][2m+c]  (0 beyond kx = nx)
__global__ void weights_layout_kernel(const float* __restrict__ w_half, float* __restrict__ wt, int ny, int nx,
                                      int* __restrict__ neg_flag) {
    const int ntile = nx / 2 + 1;
    const size_t per = (size_t)ntile * 2 * ny * 2;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= per) return;
    const int b = blockIdx.y;
    const int par = i & 1;
    const int q = (i >> 1) % ny;
    const int c = ((i >> 1) / ny) & 1;
    const int m = (int)((i >> 1) / ny / 2);
    const int kx = 2 * m + c, ky = 2 * q + par;
    float v = 0.f;
    if (kx <= nx) {
        const float* wb = w_half + (size_t)b * (2 * ny) * (nx + 1);
        v = wb[(size_t)ky * (nx + 1) + kx];
        if (!(v >= 0.f)) atomicExch(neg_flag, 1);
        // Hermitian symmetry W[-k] = W[k] (R4) is implied by the half grid everywhere except on the self-conjugate
        // columns kx = 0 and kx = nx, where both members of a pair are stored: they must agree, or the natural and the
        // transposed orientation of the operator would silently differ
        if (kx == 0 || kx == nx) {
            const float m = wb[(size_t)((2 * ny - ky) % (2 * ny)) * (nx + 1) + kx];
            if (!(fabsf(v - m) <= 1e-5f * fmaxf(fabsf(v), fabsf(m)))) atomicExch(neg_flag, 2);
        }
    }
    wt[(size_t)b * per + i] = 0.5f * v;
}
int launch_weights_layout(cudaStream_t st, const float* w_half, float* wt, int ny, int nx, int nb, int* neg_flag) {
    const size_t per = (size_t)(nx / 2 + 1) * 2 * ny * 2;
    dim3 grid((unsigned)((per + 255) / 256), nb);
    weights_layout_kernel<<<grid, 256, 0, st>>>(w_half, wt, ny, nx, neg_flag);
    return (int)cudaGetLastError();
}

// Weight table of the transposed orientation (image [nx][ny]): rows are transformed along y (tiles over
// ky = 2m+c, 0..ny), columns along x (padded bins kx = 2q+par, q < nx):
//   wtT[m][c][q][par] = 0.5 W[ky][kx],  W[ky][kx] = W[(-ky) mod 2ny][2nx - kx] for kx > nx  (Hermitian, R4)
__device__ __forceinline__ float wt_lookup(const float* wt, int ny, int ky, int kx) {   // kx <= nx
    return wt[(((size_t)(kx >> 1) * 2 + (kx & 1)) * ny + (ky >> 1)) * 2 + (ky & 1)];
}
__global__ void weights_transpose_kernel(const float* __restrict__ wt, float* __restrict__ wtT, int ny, int nx) {
    const int ntT = ny / 2 + 1;
    const size_t perT = (size_t)ntT * 2 * nx * 2, per = (size_t)(nx / 2 + 1) * 2 * ny * 2;
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= perT) return;
    const int b = blockIdx.y;
    const int par = i & 1;
    const int q = (i >> 1) % nx;
    const int c = ((i >> 1) / nx) & 1;
    const int m = (int)((i >> 1) / nx / 2);
    const int ky = 2 * m + c, kx = 2 * q + par;
    float v = 0.f;
    if (ky <= ny) {
        const float* w = wt + (size_t)b * per;
        v = kx <= nx ? wt_lookup(w, ny, ky, kx) : wt_lookup(w, ny, (2 * ny - ky) % (2 * ny), 2 * nx - kx);
    }
    wtT[(size_t)b * perT + i] = v;
}
int launch_weights_transpose(cudaStream_t st, const float* wt, float* wtT, int ny, int nx, int nb) {
    const size_t perT = (size_t)(ny / 2 + 1) * 2 * nx * 2;
    dim3 grid((unsigned)((perT + 255) / 256), nb);
    weights_transpose_kernel<<<grid, 256, 0, st>>>(wt, wtT, ny, nx);
    return (int)cudaGetLastError();
}

// Column pass on the DIF/DIT core (fft_dif.cuh): register e of thread t multiplies frequency freq_index(t, e), and reads
// its weight pair from slot e P + t of the column -- permute every column of a weight table into that order, in place.
template <int NF>
__global__ void weights_permute_kernel(float2* __restrict__ wt, int cols) {
    extern __shared__ float2 colbuf[];
    float2* w = wt + ((size_t)blockIdx.y * cols + blockIdx.x) * NF;
    for (int i = threadIdx.x; i < NF; i += blockDim.x) colbuf[i] = w[i];
    __syncthreads();
    for (int i = threadIdx.x; i < NF; i += blockDim.x) w[i] = colbuf[Dif<NF>::freq_index(i % Dif<NF>::P, i / Dif<NF>::P)];
}
template <int NF>
static int run_permute(cudaStream_t st, float* wt, int cols, int nb) {
    weights_permute_kernel<NF><<<dim3(cols, nb), 256, NF * sizeof(float2), st>>>(reinterpret_cast<float2*>(wt), cols);
    return (int)cudaGetLastError();
}
int launch_weights_permute(cudaStream_t st, float* wt, int nf, int cols, int nb) {
    switch (nf) {
        case 256: return run_permute<256>(st, wt, cols, nb);
        case 512: return run_permute<512>(st, wt, cols, nb);
        case 1024: return run_permute<1024>(st, wt, cols, nb);
        case 2048: return run_permute<2048>(st, wt, cols, nb);
        case 4096: return run_permute<4096>(st, wt, cols, nb);
        default: return (int)cudaErrorInvalidValue;
    }
}

__global__ void transpose_kernel(const float* __restrict__ in, float* __restrict__ out, int rows, int cols) {
    __shared__ float tile[32][33];
    const size_t base = (size_t)blockIdx.z * rows * cols;
    const int x = blockIdx.x * 32 + threadIdx.x;
#pragma unroll
    for (int j = 0; j < 32; j += 8) {
        const int y = blockIdx.y * 32 + threadIdx.y + j;
        if (x < cols && y < rows) tile[threadIdx.y + j][threadIdx.x] = in[base + (size_t)y * cols + x];
    }
    __syncthreads();
    const int ox = blockIdx.y * 32 + threadIdx.x;
#pragma unroll
    for (int j = 0; j < 32; j += 8) {
        const int oy = blockIdx.x * 32 + threadIdx.y + j;
        if (ox < rows && oy < cols) out[base + (size_t)oy * rows + ox] = tile[threadIdx.x][threadIdx.y + j];
    }
}
int launch_transpose(cudaStream_t st, const float* in, float* out, int rows, int cols, int nb) {
    dim3 grid((cols + 31) / 32, (rows + 31) / 32, nb), block(32, 8);
    transpose_kernel<<<grid, block, 0, st>>>(in, out, rows, cols);
    return (int)cudaGetLastError();
}

__global__ void embed_psf_kernel(const float* __restrict__ small, float* __restrict__ big, int nyi, int nxi, int ny, int nx) {
    const int my = 2 * ny, mx = 2 * nx;
    const size_t n = (size_t)my * mx;
    const float* sb = small + (size_t)blockIdx.y * 4 * nyi * nxi;
    float* bb = big + (size_t)blockIdx.y * n;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int y = (int)(i / mx), x = (int)(i % mx);
        const int sy = y < ny ? y : y - my, sx = x < nx ? x : x - mx;             // signed offsets
        float v = 0.f;
        if (sy > -nyi && sy < nyi && sx > -nxi && sx < nxi)
            v = sb[(size_t)((sy + 2 * nyi) % (2 * nyi)) * (2 * nxi) + (sx + 2 * nxi) % (2 * nxi)];
        bb[i] = v;
    }
}
int launch_embed_psf(cudaStream_t st, const float* small, float* big, int nyi, int nxi, int ny, int nx, int nb) {
    embed_psf_kernel<<<dim3(1184, nb), 256, 0, st>>>(small, big, nyi, nxi, ny, nx);
    return (int)cudaGetLastError();
}
__global__ void patch_copy_kernel(float* __restrict__ field, int nx, float* __restrict__ patch, int nyp, int nxp, int y0, int x0, int add) {
    const size_t n = (size_t)nyp * nxp;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const size_t f = (size_t)(y0 + i / nxp) * nx + x0 + i % nxp;
        if (add) field[f] += patch[i]; else patch[i] = field[f];
    }
}
int launch_patch_copy(cudaStream_t st, float* field, int ny, int nx, float* patch, int nyp, int nxp, int y0, int x0, int add) {
    (void)ny;
    patch_copy_kernel<<<592, 256, 0, st>>>(field, nx, patch, nyp, nxp, y0, x0, add);
    return (int)cudaGetLastError();
}
__global__ void mask_outside_kernel(float* __restrict__ img, int rows, int cols, int rows_in, int cols_in) {
    float* b = img + (size_t)blockIdx.y * rows * cols;
    // the strip right of the kept block, then the rows below it: only what has to be zeroed is touched
    const size_t right = (size_t)rows_in * (cols - cols_in), below = (size_t)(rows - rows_in) * cols;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < right + below; i += (size_t)gridDim.x * blockDim.x) {
        if (i < right) b[(i / (cols - cols_in)) * cols + cols_in + i % (cols - cols_in)] = 0.f;
        else b[(size_t)rows_in * cols + (i - right)] = 0.f;
    }
}
int launch_mask_outside(cudaStream_t st, float* img, int rows, int cols, int rows_in, int cols_in, int nb) {
    if (rows_in == rows && cols_in == cols) return 0;
    mask_outside_kernel<<<dim3(592, nb), 256, 0, st>>>(img, rows, cols, rows_in, cols_in);
    return (int)cudaGetLastError();
}

}  // namespace frs
