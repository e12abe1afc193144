// Backward of the hot path (Table 15): the same chunk pipeline on the gradients.
// See include/hcms.h.
#include <cstring>

#include "hcms_plan.h"

using namespace hcms;

static int ensure_stats(hcms_plan_t* p) {
  if (!p->stats) HCMS_CUDA(cudaMalloc(&p->stats, attention_bwd_stats_bytes(p->sh.S, p->sh.H)));
  if ((p->flags & HCMS_FLAG_BWD_ONE_PASS) && p->sh.D == 128 && !p->dq_acc) {
    // two accumulators, each sized for the largest chunk: chunks alternate between the two compute streams, and the
    // kernels of one stream run one after the other
    const int heads = p->sh.P * p->chunks[0].h;      // Eq. 3: chunk 0 is a largest chunk
    HCMS_CUDA(cudaMalloc(reinterpret_cast<void**>(&p->dq_acc), 2 * attention_bwd_1pass_acc_bytes(p->sh.S, heads)));
    HCMS_CUDA(cudaMalloc(reinterpret_cast<void**>(&p->dq_turn), 2 * attention_bwd_1pass_turn_bytes(p->sh.S, heads)));
  }
  return HCMS_OK;
}

// chunk c's slice of the packed statistics: heads are laid out chunk by chunk like the lse
static void* stats_of_chunk(hcms_plan_t* p, int c) {
  const size_t per_head = attention_bwd_stats_bytes(p->sh.S, 1);
  return static_cast<char*>(p->stats) + per_head * p->sh.P * p->chunks[c].o;
}

static int do_attention_bwd(hcms_plan_t* p, const void* qc, const void* kc, const void* vc, const void* oc,
                            const void* doc, const float* lse, void* dqc, void* dkc, void* dvc, int c, float scale,
                            cudaStream_t st) {
  AttnBwdArgs a{};
  a.q = qc;
  a.k = kc;
  a.v = vc;
  a.o = oc;
  a.d_o = doc;
  a.lse = lse;
  a.dq = dqc;
  a.dk = dkc;
  a.dv = dvc;
  a.stats = stats_of_chunk(p, c);
  if (p->dq_acc) {                                   // HCMS_FLAG_BWD_ONE_PASS: the buffer pair of this chunk's compute stream
    const int heads = p->sh.P * p->chunks[0].h;
    a.dq_acc = p->dq_acc + (c & 1) * (attention_bwd_1pass_acc_bytes(p->sh.S, heads) / sizeof(float));
    a.dq_turn = p->dq_turn + (c & 1) * (attention_bwd_1pass_turn_bytes(p->sh.S, heads) / sizeof(int));
  }
  a.S = p->sh.S;
  a.D = p->sh.D;
  a.P = p->sh.P;
  a.h_c = p->chunks[c].h;
  a.scale = scale;
  a.cache = &p->tmaps;
  cudaError_t e = launch_attention_bwd(a, st);
  if (e != cudaSuccess) return fail_cuda(e, "attention backward launch");
  p->last_launches += 3;
  return HCMS_OK;
}

extern "C" {

void* hcms_plan_lse(const hcms_plan_t* plan) { return plan ? plan->lse : nullptr; }

int hcms_attention_chunk_lse(hcms_plan_t* plan, const void* qc, const void* kc, const void* vc, void* oc, void* lse,
                             int c, float scale, void* stream) {
  if (!plan || !qc || !kc || !vc || !oc || !lse) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (plan->dtype != HCMS_DTYPE_BF16) return fail(HCMS_ERR_UNSUPPORTED_DTYPE, "attention needs a bf16 plan");
  if (c < 0 || c >= plan->sh.C) return fail(HCMS_ERR_PLAN_MISMATCH, "chunk %d outside [0,%d)", c, plan->sh.C);
  if (!aligned16(qc) || !aligned16(kc) || !aligned16(vc) || !aligned16(oc) || !aligned16(lse))
    return fail(HCMS_ERR_MISALIGNED, "pointer is not 16-byte aligned");
  int st = check_scale(scale);
  if (st) return st;
  if ((st = check_plan_device(plan)) != HCMS_OK) return st;
  plan->last_launches = 0;
  return do_attention(plan, qc, kc, vc, oc, c, scale, static_cast<cudaStream_t>(stream), static_cast<float*>(lse));
}

int hcms_attention_backward_chunk(hcms_plan_t* plan, const void* qc, const void* kc, const void* vc, const void* oc,
                                  const void* doc, const void* lse, void* dqc, void* dkc, void* dvc, int c,
                                  float scale, void* stream) {
  if (!plan || !qc || !kc || !vc || !oc || !doc || !lse || !dqc || !dkc || !dvc)
    return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (plan->dtype != HCMS_DTYPE_BF16) return fail(HCMS_ERR_UNSUPPORTED_DTYPE, "attention needs a bf16 plan");
  if (c < 0 || c >= plan->sh.C) return fail(HCMS_ERR_PLAN_MISMATCH, "chunk %d outside [0,%d)", c, plan->sh.C);
  for (const void* ptr : {qc, kc, vc, oc, doc, lse, static_cast<const void*>(dqc), static_cast<const void*>(dkc),
                          static_cast<const void*>(dvc)})
    if (!aligned16(ptr)) return fail(HCMS_ERR_MISALIGNED, "pointer is not 16-byte aligned");
  int st = check_scale(scale);
  if (st) return st;
  if ((st = check_plan_device(plan)) != HCMS_OK) return st;
  st = ensure_stats(plan);
  if (st) return st;
  plan->last_launches = 0;
  return do_attention_bwd(plan, qc, kc, vc, oc, doc, static_cast<const float*>(lse), dqc, dkc, dvc, c, scale,
                          static_cast<cudaStream_t>(stream));
}

int hcms_attention_backward(hcms_plan_t* plan, const void* dout, void* dq, void* dk, void* dv, int64_t S, int H, int D,
                            int P, int C, float scale, void* stream) {
  if (!plan || !dout || !dq || !dk || !dv) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  const Shape& sh = plan->sh;
  if (S != sh.S || H != sh.H || D != sh.D || P != sh.P || C != sh.C)
    return fail(HCMS_ERR_PLAN_MISMATCH, "call shape differs from the plan's");
  if (!(plan->flags & HCMS_FLAG_TRAINING)) return fail(HCMS_ERR_INVALID_ARG, "the plan was made without HCMS_FLAG_TRAINING");
  if (!plan->forward_done || !plan->train_ws || !plan->lse || !plan->ws)
    return fail(HCMS_ERR_INVALID_ARG, "no hcms_attention_forward has run on this plan (or its workspace was replaced since)");
  int st = check_scale(scale);
  if (st) return st;
  if (std::memcmp(&scale, &plan->forward_scale, sizeof(float)) != 0)
    return fail(HCMS_ERR_INVALID_ARG, "scale=%g differs from the forward's %g: the saved lse belongs to the forward's scale",
                scale, plan->forward_scale);
  if (!aligned16(dout) || !aligned16(dq) || !aligned16(dk) || !aligned16(dv))
    return fail(HCMS_ERR_MISALIGNED, "dout, dq, dk and dv must be 16-byte aligned");
  const size_t bytes = static_cast<size_t>(S) * H * D * sh.es;
  const void* all[4] = {dout, dq, dk, dv};
  for (int i = 0; i < 4; ++i)
    for (int j = i + 1; j < 4; ++j)
      if (overlaps(all[i], bytes, all[j], bytes)) return fail(HCMS_ERR_ALIAS, "dout, dq, dk, dv must not overlap");
  if ((st = check_plan_device(plan)) != HCMS_OK) return st;
  st = ensure_stats(plan);
  if (st) return st;

  char* ws = static_cast<char*>(plan->ws);          // Q'_c, K'_c, V'_c, O'_c saved by the forward
  char* gw = static_cast<char*>(plan->train_ws);    // dO'_c at off[3], dQ'_c, dK'_c, dV'_c at off[0..2]
  plan->last_launches = 0;
  PipelineSteps steps;     // the forward's schedule on the gradients: same events, same Eq. 6-7 ordering
  steps.comm_in = [&](int c, cudaStream_t s) -> int {          // input all-to-all of the incoming gradient
    const void* src[1] = {dout};
    void* dst[1] = {gw + plan->chunks[c].off[3]};
    return do_layout(plan, 1, src, dst, c, false, s);
  };
  steps.compute = [&](int c, cudaStream_t s) -> int {          // attention backward of the chunk's heads
    const Chunk& ck = plan->chunks[c];
    const float* lse_c = plan->lse + static_cast<size_t>(sh.P) * sh.S * ck.o;
    return do_attention_bwd(plan, ws + ck.off[0], ws + ck.off[1], ws + ck.off[2], ws + ck.off[3], gw + ck.off[3], lse_c,
                            gw + ck.off[0], gw + ck.off[1], gw + ck.off[2], c, scale, s);
  };
  steps.comm_out = [&](int c, cudaStream_t s) -> int {         // output all-to-all of dQ'_c, dK'_c, dV'_c, one launch
    const Chunk& ck = plan->chunks[c];
    const void* src[3] = {gw + ck.off[0], gw + ck.off[1], gw + ck.off[2]};
    void* dst[3] = {dq, dk, dv};
    return do_layout(plan, 3, src, dst, c, true, s);
  };
  return run_pipeline(plan, static_cast<cudaStream_t>(stream), steps);
}

}  // extern "C"
