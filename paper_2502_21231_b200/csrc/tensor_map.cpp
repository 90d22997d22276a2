// tensor_map.cpp — cuTensorMapEncodeTiled through cudaGetDriverEntryPoint (no -lcuda at link).
#include <mutex>

#include "launch_utils.h"

namespace {
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*,
                                  const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;
std::once_flag g_once;
cudaError_t g_err = cudaSuccess;

void resolve() {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  g_err = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (g_err == cudaSuccess && qres == cudaDriverEntryPointSuccess) g_encode = (EncodeTiledFn)fn;
}
}  // namespace

namespace bs {

bs_status_t make_tensor_map_3d(CUtensorMap* map, const void* base, int elem_bytes, int head_dim,
                               int n_heads, int64_t rows, int64_t row_stride_elems, int box_dim,
                               int box_rows, int swizzle) {
  std::call_once(g_once, resolve);
  BS_REQUIRE(g_encode != nullptr, BS_ERR_CUDA, "cuTensorMapEncodeTiled unavailable: %s",
             cudaGetErrorString(g_err));
  BS_REQUIRE(((uintptr_t)base & 15) == 0, BS_ERR_INVALID_ARG, "tensor base not 16-byte aligned");
  BS_REQUIRE((row_stride_elems * elem_bytes) % 16 == 0, BS_ERR_INVALID_ARG,
             "row stride not a multiple of 16 bytes");
  if (rows < 1) rows = 1;  // a degenerate map is never dereferenced
  cuuint64_t dims[3] = {(cuuint64_t)head_dim, (cuuint64_t)n_heads, (cuuint64_t)rows};
  cuuint64_t strides[2] = {(cuuint64_t)head_dim * elem_bytes, (cuuint64_t)row_stride_elems * elem_bytes};
  cuuint32_t box[3] = {(cuuint32_t)box_dim, 1u, (cuuint32_t)box_rows};
  cuuint32_t estr[3] = {1u, 1u, 1u};
  CUresult r = g_encode(map, elem_bytes == 2 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16
                                              : CU_TENSOR_MAP_DATA_TYPE_FLOAT32,
                        3, const_cast<void*>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE,
                        swizzle == 128 ? CU_TENSOR_MAP_SWIZZLE_128B
                        : swizzle == 64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_NONE,
                        CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  BS_REQUIRE(r == CUDA_SUCCESS, BS_ERR_CUDA, "cuTensorMapEncodeTiled failed with CUresult %d",
             (int)r);
  return BS_OK;
}

}  // namespace bs
