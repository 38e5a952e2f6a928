#pragma once
#include <cuda_runtime.h>
namespace frs {
int launch_weights_layout(cudaStream_t st, const float* w_half, float* wt, int ny, int nx, int nb, int* neg_flag);
}
