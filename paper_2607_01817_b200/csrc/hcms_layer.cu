// The attention layer around the hot path (Alg. 1 lines 2-3 and 27): QKV projection with fused
// RoPE, output projection, and the whole layer -- unfused (projection -> chunk pipeline -> projection) or with the
// all-to-alls fused into the projection GEMMs (HCMS_FLAG_FUSE_A2A).  See include/hcms.h.
#include "hcms_plan.h"

using namespace hcms;

static int run_gemm(const GemmArgs& g, cudaStream_t st, const char* what) {
  cudaError_t e = launch_gemm(g, st);
  if (e != cudaSuccess) return fail_cuda(e, what);
  return HCMS_OK;
}

// hcms_layer_forward under HCMS_FLAG_FUSE_A2A: projection epilogue -> chunk buffers -> attention per chunk -> output
// projection reading the O'_c chunk buffers.  Attention launches alternate between the two compute streams as in
// hcms_attention_forward (tail-wave backfill); the pipeline has no communication steps because no copy is left.
static int layer_forward_fused(hcms_plan_t* plan, const void* x, const void* w_qkv, const void* w_o, const void* rope_cos,
                               const void* rope_sin, void* y, int Dm, float scale, cudaStream_t caller) {
  const Shape& sh = plan->sh;
  if ((rope_cos == nullptr) != (rope_sin == nullptr)) return fail(HCMS_ERR_INVALID_ARG, "pass both RoPE tables or neither");
  if (sh.C > 16 || sh.Hl > 64)
    return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "HCMS_FLAG_FUSE_A2A needs C <= 16 and H/P <= 64 (C=%d, H/P=%d)", sh.C, sh.Hl);
  for (const void* ptr : {x, w_qkv, w_o, rope_cos, rope_sin, static_cast<const void*>(y)})
    if (!aligned16(ptr)) return fail(HCMS_ERR_MISALIGNED, "every pointer must be 16-byte aligned");
  int st = check_scale(scale);
  if (st) return st;
  if ((st = ensure_workspace(plan)) != HCMS_OK) return st;
  if ((plan->flags & HCMS_FLAG_TRAINING) && (st = ensure_training(plan)) != HCMS_OK) return st;
  char* ws = static_cast<char*>(plan->ws);
  GemmChunks ck{};
  ck.C = sh.C;
  ck.Hl = sh.Hl;
  ck.P = sh.P;
  for (int c = 0; c < sh.C; ++c) {
    ck.o[c] = plan->chunks[c].o;
    ck.h[c] = plan->chunks[c].h;
  }
  const bool profile = plan->flags & HCMS_FLAG_PROFILE;
  plan->last_launches = 0;
  if (profile) HCMS_CUDA(cudaEventRecord(plan->e_layer[0], caller));
  {  // lines 2-3 + input all-to-all
    for (int c = 0; c < sh.C; ++c)
      for (int t = 0; t < 3; ++t) ck.base[t][c] = ws + plan->chunks[c].off[t];
    GemmArgs g{};
    g.a = x;
    g.b = w_qkv;
    g.M = sh.S;
    g.N = 3 * sh.H * sh.D;
    g.K = Dm;
    g.n_per_out = sh.H * sh.D;
    g.rope_outs = rope_cos ? 2 : 0;
    g.D = sh.D;
    g.cos = static_cast<const float*>(rope_cos);
    g.sin = static_cast<const float*>(rope_sin);
    g.num_sms = plan->num_sms;
    g.fuse = 1;
    g.chunks = &ck;
    g.one_cta = plan->flags & HCMS_FLAG_GEMM_1CTA;
    g.cache = &plan->tmaps;
    st = run_gemm(g, caller, "fused QKV projection launch");
    if (st) return st;
    plan->last_launches += 1;
  }
  if (profile) HCMS_CUDA(cudaEventRecord(plan->e_layer[1], caller));
  PipelineSteps steps;            // line 15 per chunk; no comm_in / comm_out
  steps.compute = [&](int c, cudaStream_t s) -> int {
    const Chunk& k = plan->chunks[c];
    float* lse_c = plan->lse ? plan->lse + static_cast<size_t>(sh.P) * sh.S * k.o : nullptr;
    return do_attention(plan, ws + k.off[0], ws + k.off[1], ws + k.off[2], ws + k.off[3], c, scale, s, lse_c);
  };
  st = run_pipeline(plan, caller, steps);
  if (st) return st;
  if (profile) HCMS_CUDA(cudaEventRecord(plan->e_layer[2], caller));
  {  // output all-to-all + Concat + line 27
    for (int c = 0; c < sh.C; ++c) ck.base[0][c] = ws + plan->chunks[c].off[3];
    GemmArgs g{};
    g.b = w_o;
    g.out[0] = y;
    g.M = sh.S;
    g.N = Dm;
    g.K = sh.H * sh.D;
    g.n_per_out = Dm;
    g.D = sh.D;
    g.num_sms = plan->num_sms;
    g.fuse = 2;
    g.chunks = &ck;
    g.one_cta = plan->flags & HCMS_FLAG_GEMM_1CTA;
    g.cache = &plan->tmaps;
    st = run_gemm(g, caller, "fused output projection launch");
    if (st) return st;
    plan->last_launches += 1;
  }
  if (profile) {
    HCMS_CUDA(cudaEventRecord(plan->e_layer[3], caller));
    plan->layer_timed = true;
  }
  plan->forward_done = true;
  plan->forward_scale = scale;
  return HCMS_OK;
}

extern "C" {

int hcms_gemm_bf16_nt(const void* a, const void* b, void* c, int64_t M, int N, int K, void* stream) {
  if (!a || !b || !c) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (M <= 0 || N <= 0 || K <= 0) return fail(HCMS_ERR_INVALID_ARG, "M=%lld N=%d K=%d must be positive", static_cast<long long>(M), N, K);
  if (M > (1ll << 30)) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "M=%lld too large", static_cast<long long>(M));
  if (K % 8 || N % 128) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "need K %% 8 == 0 and N %% 128 == 0 (K=%d, N=%d)", K, N);
  if (!aligned16(a) || !aligned16(b) || !aligned16(c)) return fail(HCMS_ERR_MISALIGNED, "a, b and c must be 16-byte aligned");
  const size_t nc = static_cast<size_t>(M) * N * 2;
  if (overlaps(c, nc, a, static_cast<size_t>(M) * K * 2) || overlaps(c, nc, b, static_cast<size_t>(N) * K * 2))
    return fail(HCMS_ERR_ALIAS, "c overlaps an operand");
  int sms = 0;
  int st = device_sms(&sms);
  if (st) return st;
  const cudaError_t ce = gemm_init();
  if (ce != cudaSuccess) return fail_cuda(ce, "gemm_init");
  GemmArgs g{};
  g.a = a;
  g.b = b;
  g.out[0] = c;
  g.M = M;
  g.N = N;
  g.K = K;
  g.n_per_out = N;
  g.rope_outs = 0;
  g.D = 128;
  g.num_sms = sms;
  return run_gemm(g, static_cast<cudaStream_t>(stream), "gemm launch");
}

static int check_layer_shape(const hcms_plan_t* plan, int Dm) {
  if (plan->dtype != HCMS_DTYPE_BF16) return fail(HCMS_ERR_UNSUPPORTED_DTYPE, "the projections need a bf16 plan");
  if (Dm <= 0) return fail(HCMS_ERR_INVALID_ARG, "Dm=%d must be positive", Dm);
  if (Dm % 128) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "Dm=%d must be a multiple of 128", Dm);
  if ((plan->sh.H * plan->sh.D) % 128) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "H*D=%d must be a multiple of 128", plan->sh.H * plan->sh.D);
  return HCMS_OK;
}

int hcms_qkv_projection_rope(hcms_plan_t* plan, const void* x, const void* w_qkv, const void* rope_cos,
                             const void* rope_sin, void* q, void* k, void* v, int Dm, void* stream) {
  if (!plan || !x || !w_qkv || !q || !k || !v) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if ((rope_cos == nullptr) != (rope_sin == nullptr)) return fail(HCMS_ERR_INVALID_ARG, "pass both RoPE tables or neither");
  int st = check_layer_shape(plan, Dm);
  if (st) return st;
  if ((st = check_plan_device(plan)) != HCMS_OK) return st;
  for (const void* ptr : {x, w_qkv, rope_cos, rope_sin, static_cast<const void*>(q), static_cast<const void*>(k), static_cast<const void*>(v)})
    if (!aligned16(ptr)) return fail(HCMS_ERR_MISALIGNED, "every pointer must be 16-byte aligned");
  const Shape& sh = plan->sh;
  GemmArgs g{};
  g.a = x;
  g.b = w_qkv;
  g.out[0] = q;
  g.out[1] = k;
  g.out[2] = v;
  g.M = sh.S;
  g.N = 3 * sh.H * sh.D;
  g.K = Dm;
  g.n_per_out = sh.H * sh.D;
  g.rope_outs = rope_cos ? 2 : 0;
  g.D = sh.D;
  g.cos = static_cast<const float*>(rope_cos);
  g.sin = static_cast<const float*>(rope_sin);
  g.num_sms = plan->num_sms;
  g.one_cta = plan->flags & HCMS_FLAG_GEMM_1CTA;
  g.cache = &plan->tmaps;
  return run_gemm(g, static_cast<cudaStream_t>(stream), "QKV projection launch");
}

int hcms_output_projection(hcms_plan_t* plan, const void* o, const void* w_o, void* y, int Dm, void* stream) {
  if (!plan || !o || !w_o || !y) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  int st = check_layer_shape(plan, Dm);
  if (st) return st;
  if ((st = check_plan_device(plan)) != HCMS_OK) return st;
  if (!aligned16(o) || !aligned16(w_o) || !aligned16(y)) return fail(HCMS_ERR_MISALIGNED, "every pointer must be 16-byte aligned");
  const Shape& sh = plan->sh;
  GemmArgs g{};
  g.a = o;
  g.b = w_o;
  g.out[0] = y;
  g.M = sh.S;
  g.N = Dm;
  g.K = sh.H * sh.D;
  g.n_per_out = Dm;
  g.rope_outs = 0;
  g.D = sh.D;
  g.num_sms = plan->num_sms;
  g.one_cta = plan->flags & HCMS_FLAG_GEMM_1CTA;
  g.cache = &plan->tmaps;
  return run_gemm(g, static_cast<cudaStream_t>(stream), "output projection launch");
}

int hcms_layer_forward(hcms_plan_t* plan, const void* x, const void* w_qkv, const void* w_o, const void* rope_cos,
                       const void* rope_sin, void* y, int64_t S, int Dm, int H, int D, int P, int C, float scale,
                       void* stream) {
  if (!plan || !x || !w_qkv || !w_o || !y) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  const Shape& sh = plan->sh;
  if (S != sh.S || H != sh.H || D != sh.D || P != sh.P || C != sh.C)
    return fail(HCMS_ERR_PLAN_MISMATCH, "call shape differs from the plan's");
  int st = check_layer_shape(plan, Dm);
  if (st) return st;
  const size_t xy_bytes = static_cast<size_t>(S) * Dm * 2;
  if (overlaps(x, xy_bytes, y, xy_bytes)) return fail(HCMS_ERR_ALIAS, "y overlaps x");
  if ((st = check_plan_device(plan)) != HCMS_OK) return st;
  if (plan->flags & HCMS_FLAG_FUSE_A2A)
    return layer_forward_fused(plan, x, w_qkv, w_o, rope_cos, rope_sin, y, Dm, scale, static_cast<cudaStream_t>(stream));
  const size_t bytes = static_cast<size_t>(S) * H * D * sh.es;
  for (auto& b : plan->layer_buf)
    if (!b) HCMS_CUDA(cudaMalloc(&b, bytes));
  cudaStream_t caller = static_cast<cudaStream_t>(stream);
  const bool profile = plan->flags & HCMS_FLAG_PROFILE;
  if (profile) HCMS_CUDA(cudaEventRecord(plan->e_layer[0], caller));
  st = hcms_qkv_projection_rope(plan, x, w_qkv, rope_cos, rope_sin, plan->layer_buf[0], plan->layer_buf[1],
                                plan->layer_buf[2], Dm, stream);                        // lines 2-3
  if (st) return st;
  if (profile) HCMS_CUDA(cudaEventRecord(plan->e_layer[1], caller));
  st = hcms_attention_forward(plan, plan->layer_buf[0], plan->layer_buf[1], plan->layer_buf[2], plan->layer_buf[3], S, H,
                              D, P, C, scale, stream);                                  // lines 4-26
  if (st) return st;
  const int hot_launches = plan->last_launches;
  if (profile) HCMS_CUDA(cudaEventRecord(plan->e_layer[2], caller));
  st = hcms_output_projection(plan, plan->layer_buf[3], w_o, y, Dm, stream);            // line 27
  if (st) return st;
  if (profile) {
    HCMS_CUDA(cudaEventRecord(plan->e_layer[3], caller));
    plan->layer_timed = true;
  }
  plan->last_launches = hot_launches + 2;
  return HCMS_OK;
}

void* hcms_plan_layer_buffer(const hcms_plan_t* plan, int which) {
  return (plan && which >= 0 && which < 4) ? plan->layer_buf[which] : nullptr;
}

int hcms_plan_layer_timings(hcms_plan_t* plan, float* qkv_ms, float* hcms_ms, float* out_ms) {
  if (!plan) return fail(HCMS_ERR_INVALID_ARG, "plan is NULL");
  if (!(plan->flags & HCMS_FLAG_PROFILE) || !plan->layer_timed)
    return fail(HCMS_ERR_INVALID_ARG, "no hcms_layer_forward has run on this plan under HCMS_FLAG_PROFILE");
  HCMS_CUDA(cudaEventSynchronize(plan->e_layer[3]));
  float* outs[3] = {qkv_ms, hcms_ms, out_ms};
  for (int i = 0; i < 3; ++i) {
    float ms = 0.f;
    HCMS_CUDA(cudaEventElapsedTime(&ms, plan->e_layer[i], plan->e_layer[i + 1]));
    if (outs[i]) *outs[i] = ms;
  }
  return HCMS_OK;
}

}  // extern "C"
