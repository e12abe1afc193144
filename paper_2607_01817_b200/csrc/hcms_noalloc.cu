// hcms_attention_backward_chunk_static: the attention backward of one head chunk for callers that must not allocate
// device memory.  See include/hcms.h for the contract; this file holds the scratch array and the code that finds it.
//
// Who needs this.  hcms_attention_backward_chunk packs {lse * log2(e), dO.O} per (head, row) into a scratch buffer that
// the plan obtains with cudaMalloc on first use.  Some callers cannot do that: an operator living inside a framework
// whose caching allocator has already taken the whole card (a raw cudaMalloc from a library then fails, or is
// forbidden by the host application's policy because it bypasses the memory accounting); a serving loop with a latency
// budget, where cudaMalloc's implicit device-wide synchronisation is not acceptable after start-up; a process whose
// memory budget (a MIG slice, an MPS client limit) was committed in full at launch.  For them the scratch lives in the
// library image itself, and the entry point below makes no cudaMalloc, cudaFree or other allocating call.
//
// The array below is part of libhcms.so's device image: every GPU that loads the library keeps these
// HCMS_STATIC_SCRATCH_BYTES resident until the process exits, whether or not this entry point is ever called, which is
// why the size is modest and fixed.  In HOST code the identifier `g_static_scratch` is only a handle the runtime uses to
// look the symbol up; it is NOT a device address and must never be handed to a kernel.  The device address is asked for
// once per device with cudaGetSymbolAddress (with that device current) and cached.
#include <mutex>

#include "hcms_plan.h"

using namespace hcms;

static __device__ __align__(256) unsigned char g_static_scratch[HCMS_STATIC_SCRATCH_BYTES];

namespace {

std::mutex g_scratch_mutex;
void* g_scratch_addr[64] = {};   // per device: the device address of g_static_scratch, 0 = not asked yet

// Device address of the static scratch array on the CURRENT device.  The first call on a device asks the runtime
// (this loads the library's device image on that device if nothing has yet); later calls return the cached address.
int static_scratch_address(void** out) {
  int dev = -1;
  HCMS_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(HCMS_ERR_UNSUPPORTED_DEVICE, "device index %d out of range", dev);
  std::lock_guard<std::mutex> lock(g_scratch_mutex);
  if (!g_scratch_addr[dev]) {
    void* addr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&addr, g_static_scratch);
    if (e != cudaSuccess) return fail_cuda(e, "cudaGetSymbolAddress(static scratch)");
    if (!addr || reinterpret_cast<uintptr_t>(addr) % 256 != 0)
      return fail(HCMS_ERR_CUDA, "static scratch resolved to %p on device %d (expected a 256-byte aligned device address)",
                  addr, dev);
    g_scratch_addr[dev] = addr;
  }
  *out = g_scratch_addr[dev];
  return HCMS_OK;
}

}  // namespace

extern "C" int hcms_attention_backward_chunk_static(const void* qc, const void* kc, const void* vc, const void* oc,
                                                    const void* doc, const void* lse, void* dqc, void* dkc, void* dvc,
                                                    int64_t S, int P, int h_c, int D, float scale, void* stream) {
  if (!qc || !kc || !vc || !oc || !doc || !lse || !dqc || !dkc || !dvc) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (S <= 0 || P <= 0 || h_c <= 0) return fail(HCMS_ERR_INVALID_ARG, "S, P and h_c must be positive");
  if (D != 64 && D != 128) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "D=%d: the attention kernels take D = 64 or 128", D);
  // the size test comes before anything touches the device: heads * (S rounded up to 64) float2 entries must fit
  const int64_t s_pad = (S + 63) / 64 * 64;
  const int64_t max_entries = static_cast<int64_t>(HCMS_STATIC_SCRATCH_BYTES / sizeof(float2));
  if (s_pad > max_entries || static_cast<int64_t>(P) * h_c > max_entries / s_pad)
    return fail(HCMS_ERR_WORKSPACE_TOO_SMALL,
                "P*h_c*(S rounded up to 64)*8 = %lld*%lld*8 bytes of scratch exceed the static array's %lld bytes; use "
                "hcms_attention_backward_chunk (which allocates) or split the heads over several calls",
                static_cast<long long>(P) * h_c, static_cast<long long>(s_pad),
                static_cast<long long>(HCMS_STATIC_SCRATCH_BYTES));
  for (const void* ptr : {qc, kc, vc, oc, doc, lse, static_cast<const void*>(dqc), static_cast<const void*>(dkc),
                          static_cast<const void*>(dvc)})
    if (!aligned16(ptr)) return fail(HCMS_ERR_MISALIGNED, "pointer is not 16-byte aligned");
  int st = check_scale(scale);
  if (st) return st;
  int sms = 0;
  if ((st = device_sms(&sms)) != HCMS_OK) return st;     // a CUDA device is current and it is sm_100
  cudaError_t e = attention_bwd_init();                  // kernel attributes, once per device (no allocation)
  if (e != cudaSuccess) return fail_cuda(e, "attention_bwd_init");
  void* scratch = nullptr;
  if ((st = static_scratch_address(&scratch)) != HCMS_OK) return st;

  AttnBwdArgs a{};
  a.q = qc;
  a.k = kc;
  a.v = vc;
  a.o = oc;
  a.d_o = doc;
  a.lse = static_cast<const float*>(lse);
  a.dq = dqc;
  a.dk = dkc;
  a.dv = dvc;
  a.stats = scratch;       // the device address, never the host-side symbol
  a.S = S;
  a.D = D;
  a.P = P;
  a.h_c = h_c;
  a.scale = scale;
  a.cache = nullptr;       // no plan: the eleven TMA descriptors are encoded on the host for every call (no device work)
  // Nothing in the scratch has to start at zero: the statistics kernel rewrites every entry the two passes read,
  // including the {+inf, 0} padding rows [S, s_pad) of every head, before they run on the same stream.
  e = launch_attention_bwd(a, static_cast<cudaStream_t>(stream));
  if (e != cudaSuccess) return fail_cuda(e, "attention backward launch (static scratch)");
  return HCMS_OK;
}
