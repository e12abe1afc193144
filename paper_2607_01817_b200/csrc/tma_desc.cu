// cuTensorMapEncodeTiled through the runtime's driver-entry-point lookup, so that libhcms.so has
// no link-time dependency on libcuda (it must load on a box without a driver); the per-plan
// descriptor cache ("device-level caching"); per-device one-time setup helpers.
#include <atomic>
#include <mutex>

#include "hcms_internal.h"

namespace hcms {

namespace {
using EncodeFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                              const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                              CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
std::atomic<EncodeFn> g_encode{nullptr};   // the entry point is process-wide (not per device)

cudaError_t resolve(EncodeFn* out) {
  EncodeFn f = g_encode.load(std::memory_order_acquire);
  if (!f) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess) return e;
    if (qres != cudaDriverEntryPointSuccess || fn == nullptr) return cudaErrorNotSupported;
    f = reinterpret_cast<EncodeFn>(fn);
    g_encode.store(f, std::memory_order_release);
  }
  *out = f;
  return cudaSuccess;
}

struct MapKey {          // everything cuTensorMapEncodeTiled's result depends on
  const void* base;
  uint64_t dims[5], strides[4];
  uint32_t box[5];
  int32_t dt, rank, swizzle;
};
}  // namespace

cudaError_t encode_tensor_map(TmapCache* cache, CUtensorMap* out, CUtensorMapDataType dt, int rank, const void* base,
                              const uint64_t* dims, const uint64_t* strides_bytes, const uint32_t* box,
                              CUtensorMapSwizzle swizzle) {
  std::string key;
  if (cache) {
    MapKey k;
    std::memset(&k, 0, sizeof(k));
    k.base = base;
    k.dt = static_cast<int32_t>(dt);
    k.rank = rank;
    k.swizzle = static_cast<int32_t>(swizzle);
    for (int i = 0; i < rank; ++i) {
      k.dims[i] = dims[i];
      k.box[i] = box[i];
      if (i + 1 < rank) k.strides[i] = strides_bytes[i];
    }
    key.assign(reinterpret_cast<const char*>(&k), sizeof(k));
    auto it = cache->maps.find(key);
    if (it != cache->maps.end()) {
      *out = it->second;
      cache->hits += 1;
      return cudaSuccess;
    }
  }
  EncodeFn encode = nullptr;
  cudaError_t e = resolve(&encode);
  if (e != cudaSuccess) return e;
  cuuint64_t gdims[5], gstrides[4];
  cuuint32_t gbox[5], estrides[5];
  for (int i = 0; i < rank; ++i) {
    gdims[i] = dims[i];
    gbox[i] = box[i];
    estrides[i] = 1;
    if (i + 1 < rank) gstrides[i] = strides_bytes[i];
  }
  CUresult r = encode(out, dt, static_cast<cuuint32_t>(rank), const_cast<void*>(base), gdims, gstrides, gbox,
                      estrides, CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                      CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    fail(HCMS_ERR_CUDA, "cuTensorMapEncodeTiled failed with CUresult %d (rank %d, base %p)", static_cast<int>(r),
         rank, base);
    return cudaErrorInvalidValue;
  }
  if (cache) {
    if (cache->maps.size() >= 4096) cache->maps.clear();   // a caller cycling through many tensors: start over
    cache->maps.emplace(std::move(key), *out);
    cache->encodes += 1;
  }
  return cudaSuccess;
}

static std::mutex g_device_mutex;

cudaError_t once_per_device(PerDeviceOnce* state, cudaError_t (*fn)()) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_device_mutex);
  if (!state->done[dev]) {
    state->status[dev] = fn();
    state->done[dev] = true;
  }
  return state->status[dev];
}

int device_sms(int* sms) {
  static int cached[64] = {};
  int dev = 0, n = 0;
  cudaError_t ce = cudaGetDeviceCount(&n);
  if (ce != cudaSuccess || n == 0) {
    cudaGetLastError();
    return fail(HCMS_ERR_UNSUPPORTED_DEVICE, "no CUDA device; libhcms has no CPU fallback");
  }
  HCMS_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(HCMS_ERR_UNSUPPORTED_DEVICE, "device index %d out of range", dev);
  std::lock_guard<std::mutex> lock(g_device_mutex);
  if (cached[dev] == 0) {
    int major = 0, count = 0;
    HCMS_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    HCMS_CUDA(cudaDeviceGetAttribute(&count, cudaDevAttrMultiProcessorCount, dev));
    if (major != 10) return fail(HCMS_ERR_UNSUPPORTED_DEVICE, "device %d is sm_%dx; libhcms is built for sm_100a only", dev, major);
    cached[dev] = count;
  }
  *sms = cached[dev];
  return HCMS_OK;
}

}  // namespace hcms
