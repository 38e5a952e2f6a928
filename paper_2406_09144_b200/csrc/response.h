// response.h -- launchers of the exact (direct-sum) response kernels, k_response.cu
#pragma once
#include <cuda_runtime.h>
namespace frs {
constexpr int kMaxResponseSide = 1024;   // nx, ny <= 1024: the phase tables of a block live in shared memory
// vis[k] = sum_pixels img[y][x] exp(-2 pi i (u_k x / (2 nx) + v_k y / (2 ny)));  uv, vis: [nvis][2] floats
int launch_exact_degrid(cudaStream_t st, const float* uv, int nvis, const float* img, int ny, int nx, float* vis);
// out = base (or 0) + sign * sum_k 2 w_k Re(vis_k exp(+2 pi i (u_k x / (2 nx) + v_k y / (2 ny))))
int launch_exact_grid(cudaStream_t st, const float* uv, const float* wgt, const float* vis, int nvis, int ny, int nx,
                      const float* base, float sign, float* out);
}  // namespace frs
