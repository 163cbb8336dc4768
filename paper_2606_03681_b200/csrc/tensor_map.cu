// Host side of the TMA path: CUtensorMap descriptors over the [B,R,C,H,dh] bf16 cell tensor.
// The driver entry point is fetched through the runtime (no link-time dependency on libcuda).
#include <cuda.h>
#include <cuda_runtime.h>
#include <cudaTypedefs.h>

#include "tc_common.cuh"

namespace tabattn {

namespace {
PFN_cuTensorMapEncodeTiled_v12000 encode_fn() {
  static PFN_cuTensorMapEncodeTiled_v12000 fn = []() -> PFN_cuTensorMapEncodeTiled_v12000 {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      return nullptr;
    return reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(p);
  }();
  return fn;
}
}  // namespace

// View of one (table, column, head) sequence as a strided 2-D matrix [rows][dh] inside the cell
// tensor: dims innermost-first (dh, H, C, R, B), box (dh, 1, 1, box_rows, 1).  The shared-memory
// tile is [box_rows][dh] bf16 with the swizzle whose span equals one row (32/64/128 B for
// dh = 16/32/64), i.e. exactly the canonical UMMA K-major (and, read the other way, MN-major)
// layout.  Rows beyond R are zero-filled on load and clipped on store.
bool make_cell_tensor_map(CUtensorMap* map, const void* base, int B, int R, int C, int H, int dh, int box_rows) {
  auto fn = encode_fn();
  if (!fn) return false;
  const cuuint64_t d = (cuuint64_t)H * dh;
  cuuint64_t dims[5] = {(cuuint64_t)dh, (cuuint64_t)H, (cuuint64_t)C, (cuuint64_t)R, (cuuint64_t)B};
  cuuint64_t strides[4] = {(cuuint64_t)dh * 2, d * 2, (cuuint64_t)C * d * 2, (cuuint64_t)R * C * d * 2};
  cuuint32_t box[5] = {(cuuint32_t)dh, 1, 1, (cuuint32_t)box_rows, 1};
  cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  const CUtensorMapSwizzle sw = dh == 64   ? CU_TENSOR_MAP_SWIZZLE_128B
                                : dh == 32 ? CU_TENSOR_MAP_SWIZZLE_64B
                                           : CU_TENSOR_MAP_SWIZZLE_32B;
  CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, const_cast<void*>(base), dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, sw, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

}  // namespace tabattn
