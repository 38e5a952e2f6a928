// tmap.h -- TMA tensor maps over the column-pair tile layout of the spectrum T.
// T[b][m][y][c] (complex64) is described to the TMA unit as a 4-D tensor of floats
//   d0 = 4 floats  (row y of a tile: columns 2m, 2m+1)     contiguous
//   d1 = y         stride 16 B
//   d2 = m (tile)  stride 16 rows B
//   d3 = b         stride 16 rows ntile B
// with a box of {4, 1, B, 1}: one copy moves row y of B consecutive tiles, i.e.
// 2 B consecutive bins of the half spectrum of image row y, and lands them densely in shared
// memory.  Tiles beyond ntile read as zero.  The driver entry point is fetched through the runtime, so
// the library does not link against libcuda.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

namespace frs {

// tiles per copy for rows of nf complex bins: 17 copies of nf/32 tiles cover the nf/2 + 1 tiles of a row
// and fill an exchange buffer of xbuf_len(nf) slots almost exactly
__host__ __device__ constexpr int tma_box_tiles(int nf) { return nf >= 32 ? nf / 32 : 1; }
__host__ __device__ constexpr int tma_copies(int nf) { return (nf / 2 + 1 + tma_box_tiles(nf) - 1) / tma_box_tiles(nf); }

inline int make_tile_map(CUtensorMap* out, const float2* T, int rows, int nf, int nb) {
    const int ntile = nf / 2 + 1;
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static EncodeFn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
        if (e != cudaSuccess || q != cudaDriverEntryPointSuccess || !fn) return (int)(e != cudaSuccess ? e : cudaErrorUnknown);
        encode = reinterpret_cast<EncodeFn>(fn);
    }
    const cuuint64_t dims[4] = {4, (cuuint64_t)rows, (cuuint64_t)ntile, (cuuint64_t)nb};
    const cuuint64_t strides[3] = {16, (cuuint64_t)rows * 16, (cuuint64_t)rows * 16 * ntile};   // bytes, dims 1..3
    const cuuint32_t box[4] = {4, 1, (cuuint32_t)tma_box_tiles(nf), 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = encode(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, const_cast<float2*>(T), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? 0 : (int)cudaErrorInvalidValue;
}

}  // namespace frs
