// Adaptive chunk count (PAPER.md future work L346, via Theorem 1): time the real call for every C and keep the
// fastest.  One loop serves the device-tensor and the host-buffer entry points.  See include/hcms.h.
#include "hcms_plan.h"

using namespace hcms;

namespace {

// call(plan, C) runs one forward on `plan`; returns an HCMS status
template <typename Call>
int autotune(int64_t S, int H, int D, int P, int dtype, uint32_t flags, cudaStream_t caller, int max_C, int reps,
             int* best_C, float* ms_per_call, Call call) {
  if (!best_C) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (max_C < 1 || reps < 1) return fail(HCMS_ERR_INVALID_ARG, "max_C=%d and reps=%d must be >= 1", max_C, reps);
  if (P <= 0 || H <= 0 || H % P) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "H=%d is not divisible by P=%d", H, P);
  const int Hl = H / P;
  const int top = max_C < Hl ? max_C : Hl;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  HCMS_CUDA(cudaEventCreate(&e0));
  cudaError_t ce = cudaEventCreate(&e1);
  if (ce != cudaSuccess) {
    cudaEventDestroy(e0);
    return fail_cuda(ce, "cudaEventCreate");
  }
  int status = HCMS_OK;
  float best_ms = 0.f;
  *best_C = 0;
  if (ms_per_call)
    for (int i = 0; i < max_C; ++i) ms_per_call[i] = -1.f;
  for (int C = 1; C <= top && status == HCMS_OK; ++C) {
    hcms_plan_t* plan = nullptr;
    status = hcms_plan(&plan, S, H, D, P, C, dtype, flags);
    if (status != HCMS_OK) break;
    status = call(plan, C);   // warm-up
    if (status == HCMS_OK) {
      ce = cudaEventRecord(e0, caller);
      for (int r = 0; r < reps && status == HCMS_OK && ce == cudaSuccess; ++r) status = call(plan, C);
      if (ce == cudaSuccess) ce = cudaEventRecord(e1, caller);
      if (ce == cudaSuccess) ce = cudaEventSynchronize(e1);
      float ms = 0.f;
      if (ce == cudaSuccess) ce = cudaEventElapsedTime(&ms, e0, e1);
      if (ce != cudaSuccess && status == HCMS_OK) status = fail_cuda(ce, "autotune timing");
      if (status == HCMS_OK) {
        ms /= reps;
        if (ms_per_call) ms_per_call[C - 1] = ms;
        if (*best_C == 0 || ms < best_ms) {
          best_ms = ms;
          *best_C = C;
        }
      }
    }
    plan_free(plan);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return status;
}

}  // namespace

extern "C" {

int hcms_autotune_chunks(int64_t S, int H, int D, int P, int dtype, uint32_t flags, const void* q, const void* k,
                         const void* v, void* out, float scale, void* stream, int max_C, int reps, int* best_C,
                         float* ms_per_call) {
  if (!q || !k || !v || !out) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  return autotune(S, H, D, P, dtype, flags & ~(HCMS_FLAG_SERIAL | HCMS_FLAG_PROFILE), static_cast<cudaStream_t>(stream),
                  max_C, reps, best_C, ms_per_call, [&](hcms_plan_t* plan, int C) {
                    return hcms_attention_forward(plan, q, k, v, out, S, H, D, P, C, scale, stream);
                  });
}

int hcms_autotune_chunks_host(int64_t S, int H, int D, int P, uint32_t flags, const void* q, const void* k, const void* v,
                              void* out, float scale, void* stream, int max_C, int reps, int* best_C, float* ms_per_call) {
  if (!q || !k || !v || !out) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  return autotune(S, H, D, P, HCMS_DTYPE_BF16, flags & ~(HCMS_FLAG_SERIAL | HCMS_FLAG_PROFILE | HCMS_FLAG_GRAPH),
                  static_cast<cudaStream_t>(stream), max_C, reps, best_C, ms_per_call, [&](hcms_plan_t* plan, int C) {
                    return hcms_attention_forward_host(plan, q, k, v, out, S, H, D, P, C, scale, stream);
                  });
}

}  // extern "C"
