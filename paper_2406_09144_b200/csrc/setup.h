#pragma once
#include <cuda_runtime.h>
namespace frs {
int launch_weights_layout(cudaStream_t st, const float* w_half, float* wt, int ny, int nx, int nb, int* neg_flag);
// wt [nb][nx/2+1][2][ny][2] (natural orientation) -> wtT [nb][ny/2+1][2][nx][2] (transposed image orientation)
int launch_weights_transpose(cudaStream_t st, const float* wt, float* wtT, int ny, int nx, int nb);
// wt [nb][cols][nf][2]: every column into the consumption order of the DIF/DIT column pass (nf >= 256), in place
int launch_weights_permute(cudaStream_t st, float* wt, int nf, int cols, int nb);
// out[b][j][i] = in[b][i][j], in [nb][rows][cols]
int launch_transpose(cudaStream_t st, const float* in, float* out, int rows, int cols, int nb);
// Embedding of an image that is smaller than the grid (reading R19).
// big [nb][2 ny][2 nx] <- small [nb][2 nyi][2 nxi]: the PSF copied to the offsets |dy| < nyi, |dx| < nxi (wrapped), zero elsewhere
int launch_embed_psf(cudaStream_t st, const float* small, float* big, int nyi, int nxi, int ny, int nx, int nb);
// field[y0 + y][x0 + x] += patch[y][x] (add = 1)  or  patch[y][x] = field[y0 + y][x0 + x] (add = 0); patch [nyp][nxp], field [ny][nx]
int launch_patch_copy(cudaStream_t st, float* field, int ny, int nx, float* patch, int nyp, int nxp, int y0, int x0, int add);
// img [nb][rows][cols] <- 0 outside [0, rows_in) x [0, cols_in)
int launch_mask_outside(cudaStream_t st, float* img, int rows, int cols, int rows_in, int cols_in, int nb);
}
