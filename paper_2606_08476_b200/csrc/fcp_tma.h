// Host helper: TMA tensor maps for token-major varlen tensors [rows, heads, D] (bf16).
// The driver entry point is resolved at run time so libfcp.so loads on machines without
// libcuda (the CPU-only build/test container).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace fcp {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn resolve_encode_tiled() {
  void* p = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) ==
          cudaSuccess &&
      q == cudaDriverEntryPointSuccess)
    return reinterpret_cast<EncodeTiledFn>(p);
  return nullptr;
}
// resolved once (thread-safe initialisation of a function-local static; the address never changes)
inline EncodeTiledFn encode_tiled_fn() {
  static const EncodeTiledFn fn = resolve_encode_tiled();
  return fn;
}

// View of base[rows][heads][D] as a 3-D tensor (D, heads, rows); box = (64 elements = 128 B,
// 1 head, box_rows rows), 128-byte swizzle, out-of-bounds rows read as zero.
inline bool make_tmap_rows(CUtensorMap* map, const void* base, int D, int heads, int64_t rows,
                           int box_rows) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return false;
  if (rows < 1) rows = 1;
  cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)heads, (cuuint64_t)rows};
  cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)heads * D * 2};   // bytes, dims 1..2
  cuuint32_t box[3] = {64, 1, (cuuint32_t)box_rows};
  cuuint32_t elem[3] = {1, 1, 1};
  return fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box,
            elem, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace fcp
