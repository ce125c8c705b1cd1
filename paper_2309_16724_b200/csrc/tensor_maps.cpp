// Host side of the bulk-tensor (TMA) operand staging of heff_tma_kernel: encoding of the tensor maps.
//
// Every operand block is a rank-3 tensor {columns, rows, items} of FP64 elements: the columns run along the
// contiguous direction of the STORED block (row pitch ld elements, a multiple of 2 so that rows start on 16-byte
// boundaries), items are the positions of an operator family (the third index of the dense blocks),
// the Psi sectors' single item, or the batch index of a GEMM-pair microbenchmark call.  The box is what one
// bulk-tensor copy moves; the extents are the TRUE extents of the block, so that anything a box covers beyond them
// (ragged block edges, the k tail of the last pipeline stage) arrives as zeros.
//
// cuTensorMapEncodeTiled is a driver entry point; it is fetched through the runtime (cudaGetDriverEntryPoint) so
// that the library does not link against libcuda.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <tuple>

#include "su2_internal.h"

namespace su2 {

bool MapKey::operator<(const MapKey& o) const {
  return std::tie(base, rows, cols, ld, nitems, item_stride, box_c, box_r) <
         std::tie(o.base, o.rows, o.cols, o.ld, o.nitems, o.item_stride, o.box_c, o.box_r);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = []() -> EncodeTiledFn {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      return nullptr;
    return (EncodeTiledFn)p;
  }();
  return fn;
}

su2_status encode_tensor_map(void* out128, const MapKey& k) {
  static_assert(sizeof(CUtensorMap) == 128, "tensor maps are stored as 128-byte records");
  EncodeTiledFn fn = encode_fn();
  if (!fn) { set_error_text("cuTensorMapEncodeTiled is not available from this driver"); return SU2_ERR_CUDA; }
  if (((uintptr_t)k.base & 15) || (k.ld & 1) || (k.item_stride & 1) || k.box_c > 256 || k.box_r > 256 || k.cols <= 0 || k.rows <= 0 ||
      k.nitems <= 0) {
    set_error_text("operand block cannot be described by a tensor map (16-byte alignment of rows, box <= 256)");
    return SU2_ERR_INVALID_ARGUMENT;
  }
  const cuuint64_t gdim[3] = {(cuuint64_t)k.cols, (cuuint64_t)k.rows, (cuuint64_t)k.nitems};
  // strides of dimensions 1 and 2 in bytes; a single item still needs a legal (non-zero, 16-byte multiple) stride
  const cuuint64_t istride = k.item_stride > 0 ? (cuuint64_t)k.item_stride : (cuuint64_t)k.rows * (cuuint64_t)k.ld;
  const cuuint64_t gstride[2] = {(cuuint64_t)k.ld * 8u, istride * 8u};
  const cuuint32_t box[3] = {(cuuint32_t)k.box_c, (cuuint32_t)k.box_r, 1u};
  const cuuint32_t estr[3] = {1u, 1u, 1u};
  CUresult r = fn((CUtensorMap*)out128, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<void*>(k.base), gdim, gstride, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    char buf[256];
    std::snprintf(buf, sizeof(buf), "cuTensorMapEncodeTiled failed (%d): cols %d rows %d ld %d items %d box %d x %d", (int)r, k.cols,
                  k.rows, k.ld, k.nitems, k.box_c, k.box_r);
    set_error_text(buf);
    return SU2_ERR_CUDA;
  }
  return SU2_OK;
}

}  // namespace su2
