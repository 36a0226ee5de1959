// tmap.hpp -- host-side construction of TMA tensor maps (CUtensorMap) without linking libcuda:
// cuTensorMapEncodeTiled is fetched through cudaGetDriverEntryPoint at first use.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace mesh_attn {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
            return (EncodeTiledFn) nullptr;
        return (EncodeTiledFn)p;
    }();
    return fn;
}

// bf16 tensor addressed as (d, h, row, batch) with arbitrary byte strides for h / row / batch;
// box = 64 elements of d (128 bytes, SWIZZLE_128B) x 1 head x box_rows rows x 1 batch.
inline bool make_tmap_bf16_4d(CUtensorMap* out, const void* base, uint64_t D, uint64_t H, uint64_t rows, uint64_t B,
                              uint64_t stride_h_bytes, uint64_t stride_row_bytes, uint64_t stride_b_bytes, uint32_t box_rows)
{
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    cuuint64_t dims[4] = {D, H, rows, B};
    cuuint64_t strides[3] = {stride_h_bytes, stride_row_bytes, stride_b_bytes};
    cuuint32_t box[4] = {64, 1, box_rows, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    return fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// fp32 tensor addressed as (d, h, row, batch) for the backward's dQ reduction (cp.reduce.async.bulk.tensor):
// box = all D elements of a row x 1 head x box_rows rows x 1 batch, no swizzle (the staging tile is plain row-major).
inline bool make_tmap_f32_4d(CUtensorMap* out, const void* base, uint64_t D, uint64_t H, uint64_t rows, uint64_t B,
                             uint64_t stride_h_bytes, uint64_t stride_row_bytes, uint64_t stride_b_bytes, uint32_t box_rows)
{
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    cuuint64_t dims[4] = {D, H, rows, B};
    cuuint64_t strides[3] = {stride_h_bytes, stride_row_bytes, stride_b_bytes};
    cuuint32_t box[4] = {(cuuint32_t)D, 1, box_rows, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    return fn(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace mesh_attn
