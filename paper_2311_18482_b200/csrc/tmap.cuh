// tmap.cuh — host helper: tiled TMA tensor maps for 2D row-major bf16 tensors (cuTensorMapEncodeTiled, resolved through
// the runtime at legs_create: no link-time libcuda dependency).
#pragma once
#include <cuda.h>

#include "common.cuh"

// [rows, inner] bf16 -> tensor map with a box_inner x box_rows box and the 128-byte swizzle (the UMMA K-major layout).
// Out-of-bounds box elements are zero-filled and still count towards the mbarrier's transaction bytes.
static inline int make_tmap_bf16_2d(legs_ctx* ctx, const void* base, uint64_t inner, uint64_t rows, uint32_t box_inner,
                                    uint32_t box_rows, CUtensorMap* out) {
  typedef CUresult (*EncodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  const cuuint64_t gdim[2] = {inner, rows};
  const cuuint64_t gstride[1] = {inner * 2};
  const cuuint32_t box[2] = {box_inner, box_rows};
  const cuuint32_t estride[2] = {1, 1};
  const CUresult cr = ((EncodeTiled)ctx->encode_tiled)(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), gdim,
                                                       gstride, box, estride, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                                       CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                                                       CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (cr != CUDA_SUCCESS) { ctx->last_cuda_error = (int)cr; return LEGS_ERR_CUDA; }
  return LEGS_OK;
}
