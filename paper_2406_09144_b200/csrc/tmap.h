// tmap.h -- TMA tensor maps over the spectrum T.
// T[b][m][y/2][c][y%2] (complex64): 32-byte blocks of (2 bins kx = 2m + c) x (2 image rows), so that
//   * a row pass writes / reads whole 32-byte sectors (bins 2m, 2m+1 of its row pair), and
//   * a column kx is a run of 16-byte pieces (rows 2r, 2r+1) at a stride of 32 bytes,
// both of which the TMA unit moves as boxes of a strided tensor, landing them DENSELY in shared memory:
//   row map  (4-D floats): d0 = 8 floats of a block, d1 = y/2 (32 B), d2 = m (16 rows B), d3 = b;
//             box {8, 1, B, 1} = bins [2 m0, 2 m0 + 2B) of one row pair -> 16-byte slots (Y_0[k], Y_1[k])
//   col map  (5-D floats): d0 = 4 floats of a piece, d1 = c (16 B), d2 = y/2 (32 B), d3 = m, d4 = b;
//             box {4, 1, R, 1, 1} = rows [2 r0, 2 r0 + 2R) of one column -> contiguous complex samples
// Blocks beyond the last tile read as zero.  The column pass writes its result to a second array in plain
// column-contiguous order (whole sectors, coalesced), which the inverse row pass gathers through a third map.  The driver entry point is fetched through the runtime,
// so the library does not link against libcuda.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

namespace frs {

// row map: 17 copies of nf/32 tiles cover the nf/2 + 1 tiles of a row pair and fill an exchange buffer
// of xbuf_len(nf) slots almost exactly; TMA needs 128-byte aligned boxes in shared memory
__host__ __device__ constexpr int tma_box_tiles(int nf) { return nf >= 32 ? nf / 32 : 1; }
__host__ __device__ constexpr int tma_row_copies(int nf) { return (nf / 2 + 1 + tma_box_tiles(nf) - 1) / tma_box_tiles(nf); }
__host__ __device__ constexpr bool tma_rows_ok(int nf) { return nf >= 128; }
// col map: copies of up to 256 row pairs (rows >= 32: boxes of >= 256 bytes)
__host__ __device__ constexpr int tma_box_pairs(int rows) { return rows / 2 < 256 ? rows / 2 : 256; }
__host__ __device__ constexpr int tma_col_copies(int rows) { return (rows / 2) / tma_box_pairs(rows); }

// column-contiguous spectrum T2[b][kx][y] (what conv_cols writes): 3-D floats d0 = 2 y + {re, im}, d1 = kx (8 rows B),
// d2 = b; box {4, B, 1} = bins [kx0, kx0 + B) of one row pair, 16 bytes per bin; 17 copies of B = nf/16 bins
__host__ __device__ constexpr int tma_box_bins(int nf) { return nf >= 16 ? nf / 16 : 1; }
__host__ __device__ constexpr int tma_bin_copies(int nf) { return (nf + 1 + tma_box_bins(nf) - 1) / tma_box_bins(nf); }

typedef CUresult (*TmapEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
inline TmapEncodeFn tmap_encoder() {
    static TmapEncodeFn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q);
        if (e == cudaSuccess && q == cudaDriverEntryPointSuccess) encode = reinterpret_cast<TmapEncodeFn>(fn);
    }
    return encode;
}
// T: [nb][ntile][rows/2][2][2] complex64, ntile = nf/2 + 1
inline int make_spectrum_maps(CUtensorMap* row_map, CUtensorMap* col_map, const float2* T, int rows, int nf, int nb) {
    TmapEncodeFn encode = tmap_encoder();
    if (!encode) return (int)cudaErrorUnknown;
    const cuuint64_t ntile = (cuuint64_t)nf / 2 + 1, tile_bytes = (cuuint64_t)rows * 16;
    const cuuint32_t one[5] = {1, 1, 1, 1, 1};
    {
        const cuuint64_t dims[4] = {8, (cuuint64_t)rows / 2, ntile, (cuuint64_t)nb};
        const cuuint64_t strides[3] = {32, tile_bytes, tile_bytes * ntile};
        const cuuint32_t box[4] = {8, 1, (cuuint32_t)tma_box_tiles(nf), 1};
        if (encode(row_map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, const_cast<float2*>(T), dims, strides, box, one,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) return (int)cudaErrorInvalidValue;
    }
    {
        const cuuint64_t dims[5] = {4, 2, (cuuint64_t)rows / 2, ntile, (cuuint64_t)nb};
        const cuuint64_t strides[4] = {16, 32, tile_bytes, tile_bytes * ntile};
        const cuuint32_t box[5] = {4, 1, (cuuint32_t)tma_box_pairs(rows), 1, 1};
        if (encode(col_map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, const_cast<float2*>(T), dims, strides, box, one,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) return (int)cudaErrorInvalidValue;
    }
    return 0;
}

// T2: [nb][cols][rows] complex64, bins kx = 0..nf exist
inline int make_columns_map(CUtensorMap* map, const float2* T2, int rows, int nf, int cols, int nb) {
    TmapEncodeFn encode = tmap_encoder();
    if (!encode) return (int)cudaErrorUnknown;
    const cuuint64_t dims[3] = {(cuuint64_t)rows * 2, (cuuint64_t)nf + 1, (cuuint64_t)nb};
    const cuuint64_t strides[2] = {(cuuint64_t)rows * 8, (cuuint64_t)rows * 8 * cols};
    const cuuint32_t box[3] = {4, (cuuint32_t)tma_box_bins(nf), 1};
    const cuuint32_t one[3] = {1, 1, 1};
    return encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float2*>(T2), dims, strides, box, one,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS ? 0 : (int)cudaErrorInvalidValue;
}

}  // namespace frs
