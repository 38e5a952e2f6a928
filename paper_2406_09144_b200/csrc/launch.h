// launch.h -- size-dispatching launchers of the FFT passes (one translation unit per pass so the
// template instantiations compile in parallel).  Return cudaError_t as int.
#pragma once
#include <cuda_runtime.h>
#include "kernels.cuh"

namespace frs {

// valid transform lengths
inline bool valid_nf(int nf) { return nf >= 16 && nf <= 4096 && (nf & (nf - 1)) == 0; }

// rows: number of image rows (even).  nf: complex transform length (PAD: nf = nx; else nf = nx/2).
int launch_rows_fwd(cudaStream_t st, int nf, bool pad, const RowsFwdArgs& a, int nb);
// nf >= 256 runs the DIF/DIT kernel (a.tw: its tables, a.wt: weights in its permuted order), smaller nf the sorting core
int launch_conv_cols(cudaStream_t st, int nf, const ConvColsArgs& a, int nb);
inline bool conv_cols_uses_dif(int nf) { return nf >= 256; }
int launch_rows_inv(cudaStream_t st, int nf, const RowsInvArgs& a, int nb, int* grid_x);
// the inverse row pass fused with the row pass of the Hartley transform that follows (a.inv.mode: kMulS or kEnergy)
inline bool rows_inv_hart_ok(int nf) { return nf == 1024 || nf == 2048 || nf == 4096; }
int launch_rows_inv_hart(cudaStream_t st, int nf, const RowsInvHartArgs& a, int nb, int* grid_x);
int launch_hart_cols(cudaStream_t st, int nf, const HartColsArgs& a, int nb, int* grid_x = nullptr);

struct PsfColsArgs {
    const float2* t;      // row-transformed PSF, all 2 NF rows, ncols - 1 = nx bins + 1: block layout of tmap.h
    int ncols;            // columns that exist (nx + 1)
    float* wt;            // [nb][ntile][2][NF][2]
    float* stats;         // [nb][gridDim.x][3]: max |Im W|, min Re W, max Re W   (unscaled by fold)
    int ntile;
    float scale;          // 1 / (My Mx)
    float floor;          // W is stored as max(Re W, floor): 0 for a covariance kernel, -FLT_MAX for an embedded PSF
    size_t w_bstride;
    const float4* tw;
    const float2* twist;
};
int launch_psf_cols(cudaStream_t st, int nf, const PsfColsArgs& a, int nb, int* grid_x);

#define FRS_DISPATCH_NF(nf, CALL)                 \
    switch (nf) {                                 \
        case 16: { CALL(16); } break;             \
        case 32: { CALL(32); } break;             \
        case 64: { CALL(64); } break;             \
        case 128: { CALL(128); } break;           \
        case 256: { CALL(256); } break;           \
        case 512: { CALL(512); } break;           \
        case 1024: { CALL(1024); } break;         \
        case 2048: { CALL(2048); } break;         \
        case 4096: { CALL(4096); } break;         \
        default: return (int)cudaErrorInvalidValue; \
    }

template <typename K>
inline cudaError_t set_smem(K kernel, int bytes) {
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

// The shared-memory opt-in and the resident-CTA count belong to a (kernel, DEVICE) pair: cached per device,
// in a table owned by the launcher of each kernel instantiation.
constexpr int kMaxDevices = 64;
template <typename K> inline int resident_ctas(K kernel, int threads, int smem);
template <typename K>
inline int persistent_ctas(int (&cache)[kMaxDevices], K kernel, int threads, int smem, int* ctas) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
    if (dev < 0 || dev >= kMaxDevices) return (int)cudaErrorInvalidDevice;
    if (!cache[dev]) {
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return (int)e;
        const int c = resident_ctas(kernel, threads, smem);
        if (!c) return (int)cudaErrorUnknown;
        cache[dev] = c;
    }
    *ctas = cache[dev];
    return 0;
}

// resident CTAs of a persistent kernel = SMs x occupancy (0 on error)
template <typename K>
inline int resident_ctas(K kernel, int threads, int smem) {
    int dev = 0, sms = 0, occ = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem) != cudaSuccess) return 0;
    return sms * (occ > 0 ? occ : 1);
}

}  // namespace frs
