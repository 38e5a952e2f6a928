// tmap.h -- layout of the spectrum T between the row pass and the column pass, and the TMA tensor maps over it and over
// T2.
// T[b][m][y/2][c][y%2] (complex64), kx = 8 m + c: 128-byte blocks of (8 bins) x (2 image rows), so that
//   * a row pass writes whole 128-byte lines: a thread holds (X_0[k], X_1[k]) of its row pair, 8 neighbouring lanes hold
//     the 8 bins of a block (a warp store touches 4 lines; with 32-byte blocks of 2 bins it touched 16, and those
//     scattered stores were a third of the row pass's L1 data-pipe load, profiles/r2_notes.md), and
//   * a column kx is a run of 16-byte pieces (rows 2r, 2r+1) at a stride of 128 bytes inside one contiguous region of
//     64 rows bytes, which the TMA unit gathers as boxes of a strided tensor, landing them DENSELY in shared memory:
//   col map  (5-D floats): d0 = 4 floats of a piece, d1 = c (16 B), d2 = y/2 (128 B), d3 = m, d4 = b;
//             box {4, 1, R, 1, 1} = rows [2 r0, 2 r0 + 2R) of one column -> contiguous complex samples.
// The 8 columns of a block are convolved by neighbouring CTAs at about the same time, so each line leaves DRAM once.
// Blocks beyond the last bin read as zero.  The column pass writes its result to a second array T2 in plain
// column-contiguous order (coalesced), which the inverse row pass gathers through a 3-D map.  The driver entry point is
// fetched through the runtime, so the library does not link against libcuda.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

namespace frs {

// Two block widths.  The convolution's spectrum T (rows_fwd<.,PAD> -> conv_cols) uses 8 bins per block, see above.  The
// Hartley row pass and the PSF set-up (rows_fwd<.,!PAD> -> hart_cols / psf_cols) use 2: their column pass carries the
// column PAIR (2m, 2m+1) per thread, and with 2-bin blocks that pair is one CONTIGUOUS run of 16 rows bytes, fetched by a
// single bulk copy (with 8-bin blocks the same pair is 32-byte pieces at a 128-byte stride: measured 12 us slower per
// Hartley transform at 4096^2, whether read by loads or by a TMA gather).
constexpr int kBlockBins = 8;                                     // conv: bins kx per 128-byte block of T
constexpr int kPairBins = 2;                                      // Hartley / PSF set-up: bins per 32-byte block
__host__ __device__ constexpr int spec_tiles(int nf, int bins = kBlockBins) { return nf / bins + 1; }   // bins kx = 0..nf
// float2 index, inside one batch, of sample (kx, y) of the row-transformed array of `rows` image rows
__host__ __device__ constexpr size_t spec_index(int rows, int kx, int y, int bins = kBlockBins) {
    return ((((size_t)(kx / bins) * (rows / 2) + (y >> 1)) * bins + (kx % bins)) << 1) + (y & 1);
}
__host__ __device__ constexpr size_t spec_batch_stride(int rows, int nf, int bins = kBlockBins) {
    return (size_t)spec_tiles(nf, bins) * rows * bins;
}

// smaller rows: boxes below the 128-byte TMA alignment -> cp.async
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
// column map of T: [nb][spec_tiles(nf)][rows/2][8][2] complex64
inline int make_spectrum_col_map(CUtensorMap* col_map, const float2* T, int rows, int nf, int nb) {
    TmapEncodeFn encode = tmap_encoder();
    if (!encode) return (int)cudaErrorUnknown;
    const cuuint64_t ntile = (cuuint64_t)spec_tiles(nf), tile_bytes = (cuuint64_t)rows * 8 * kBlockBins;
    const cuuint32_t one[5] = {1, 1, 1, 1, 1};
    const cuuint64_t dims[5] = {4, (cuuint64_t)kBlockBins, (cuuint64_t)rows / 2, ntile, (cuuint64_t)nb};
    const cuuint64_t strides[4] = {16, 16 * kBlockBins, tile_bytes, tile_bytes * ntile};
    const cuuint32_t box[5] = {4, 1, (cuuint32_t)tma_box_pairs(rows), 1, 1};
    return encode(col_map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, const_cast<float2*>(T), dims, strides, box, one,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS ? 0 : (int)cudaErrorInvalidValue;
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
