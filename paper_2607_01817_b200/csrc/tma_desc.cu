// cuTensorMapEncodeTiled through the runtime's driver-entry-point lookup, so that libhcms.so has
// no link-time dependency on libcuda (it must load on a box without a driver).
#include "hcms_internal.h"

namespace hcms {

namespace {
using EncodeFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                              const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                              CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeFn g_encode = nullptr;

cudaError_t resolve() {
  if (g_encode) return cudaSuccess;
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess) return e;
  if (qres != cudaDriverEntryPointSuccess || fn == nullptr) return cudaErrorNotSupported;
  g_encode = reinterpret_cast<EncodeFn>(fn);
  return cudaSuccess;
}
}  // namespace

cudaError_t encode_tensor_map(CUtensorMap* out, CUtensorMapDataType dt, int rank, const void* base,
                              const uint64_t* dims, const uint64_t* strides_bytes, const uint32_t* box,
                              CUtensorMapSwizzle swizzle) {
  cudaError_t e = resolve();
  if (e != cudaSuccess) return e;
  cuuint64_t gdims[5], gstrides[4];
  cuuint32_t gbox[5], estrides[5];
  for (int i = 0; i < rank; ++i) {
    gdims[i] = dims[i];
    gbox[i] = box[i];
    estrides[i] = 1;
    if (i + 1 < rank) gstrides[i] = strides_bytes[i];
  }
  CUresult r = g_encode(out, dt, static_cast<cuuint32_t>(rank), const_cast<void*>(base), gdims, gstrides, gbox,
                        estrides, CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    fail(HCMS_ERR_CUDA, "cuTensorMapEncodeTiled failed with CUresult %d (rank %d, base %p)", static_cast<int>(r),
         rank, base);
    return cudaErrorInvalidValue;
  }
  return cudaSuccess;
}

}  // namespace hcms
