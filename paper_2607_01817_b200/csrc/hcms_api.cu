// libhcms entry points: plan, chunk table, the dual-stream chunk scheduler (section 3.4-3.6,
// Algorithm 1), single-step hooks, host-buffer call, profile read-back.  See include/hcms.h.
// The layer (projections), the backward and the chunk-count tuners live in hcms_layer.cu, hcms_backward.cu and
// hcms_tune.cu; all of them run the ONE fork/join schedule below (run_pipeline).
#include <cmath>
#include <cstdarg>
#include <cstring>
#include <new>

#include "hcms_plan.h"

namespace hcms {

// ------------------------------------------------------------------------------------------
// errors
// ------------------------------------------------------------------------------------------
static thread_local char g_last_error[512] = "";

int fail(int status, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_last_error, sizeof(g_last_error), fmt, ap);
  va_end(ap);
  return status;
}
int fail_cuda(cudaError_t e, const char* what) {
  return fail(HCMS_ERR_CUDA, "CUDA error %d (%s: %s) in %s", static_cast<int>(e), cudaGetErrorName(e),
              cudaGetErrorString(e), what);
}

// ------------------------------------------------------------------------------------------
// host-only math
// ------------------------------------------------------------------------------------------
static int chunk_table(int Hl, int C, int* o, int* h) {
  if (Hl <= 0 || C <= 0) return fail(HCMS_ERR_INVALID_ARG, "heads_per_rank=%d and C=%d must be positive", Hl, C);
  if (C > Hl) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "C=%d exceeds heads per rank %d (every chunk needs a head)", C, Hl);
  int off = 0;
  for (int c = 0; c < C; ++c) {
    const int hc = Hl / C + (c < Hl % C ? 1 : 0);  // Eq. 3, larger chunks first (L221)
    if (o) o[c] = off;
    if (h) h[c] = hc;
    off += hc;
  }
  return HCMS_OK;
}

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ------------------------------------------------------------------------------------------
// plan helpers shared by the translation units
// ------------------------------------------------------------------------------------------
void plan_free(hcms_plan_t* p) {
  if (!p) return;
  for (cudaStream_t s : {p->s_comm, p->s_comm_out, p->s_comp, p->s_comp2, p->s_cap})
    if (s) cudaStreamSynchronize(s);
  for (auto e : p->e_comm) if (e) cudaEventDestroy(e);
  for (auto e : p->e_comp) if (e) cudaEventDestroy(e);
  if (p->e_main) cudaEventDestroy(p->e_main);
  for (auto e : p->e_fin) if (e) cudaEventDestroy(e);
  for (auto& step : p->prof)
    for (auto& side : step)
      for (auto e : side)
        if (e) cudaEventDestroy(e);
  if (p->graph_exec) cudaGraphExecDestroy(p->graph_exec);
  for (cudaStream_t s : {p->s_comm, p->s_comm_out, p->s_comp, p->s_comp2, p->s_cap})
    if (s) cudaStreamDestroy(s);
  if (p->ws_owned && p->ws) cudaFree(p->ws);
  for (auto& h : p->pinned) if (h) cudaFreeHost(h);
  for (auto& d : p->wire) if (d) cudaFree(d);
  for (auto& d : p->staging) if (d) cudaFree(d);
  for (auto& d : p->layer_buf) if (d) cudaFree(d);
  if (p->train_ws) cudaFree(p->train_ws);
  if (p->lse) cudaFree(p->lse);
  if (p->stats) cudaFree(p->stats);
  if (p->dq_acc) cudaFree(p->dq_acc);
  if (p->dq_turn) cudaFree(p->dq_turn);
  for (auto& e : p->e_layer) if (e) cudaEventDestroy(e);
  delete p;
}

int check_scale(float scale) {
  if (!std::isfinite(scale) || scale < 0.f) return fail(HCMS_ERR_INVALID_ARG, "scale=%g must be finite and >= 0", scale);
  return HCMS_OK;
}

int check_plan_device(const hcms_plan_t* p) {
  int dev = -1;
  HCMS_CUDA(cudaGetDevice(&dev));
  if (dev != p->device)
    return fail(HCMS_ERR_PLAN_MISMATCH, "the plan was made on device %d but device %d is current", p->device, dev);
  return HCMS_OK;
}

int ensure_workspace(hcms_plan_t* p) {
  if (p->ws) return HCMS_OK;
  HCMS_CUDA(cudaMalloc(&p->ws, p->ws_bytes));
  p->ws_owned = true;
  return HCMS_OK;
}

int ensure_training(hcms_plan_t* p) {
  if (!p->train_ws) HCMS_CUDA(cudaMalloc(&p->train_ws, p->ws_bytes));
  if (!p->lse) HCMS_CUDA(cudaMalloc(reinterpret_cast<void**>(&p->lse), static_cast<size_t>(p->sh.H) * p->sh.S * sizeof(float)));
  return HCMS_OK;
}

int do_layout(hcms_plan_t* p, int n, const void* const* src, void* const* dst, int c, bool gather, cudaStream_t st) {
  const Chunk& ck = p->chunks[c];
  LayoutArgs a{};
  for (int t = 0; t < n; ++t) {
    a.src[t] = src[t];
    a.dst[t] = dst[t];
  }
  a.n_tensors = n;
  a.S = p->sh.S;
  a.H = p->sh.H;
  a.D = p->sh.D;
  a.P = p->sh.P;
  a.Hl = p->sh.Hl;
  a.es = p->sh.es;
  a.o_c = ck.o;
  a.h_c = ck.h;
  a.gather = gather;
  a.cache = &p->tmaps;
  cudaError_t e = (p->flags & HCMS_FLAG_LAYOUT_TMA) ? launch_layout_tma(a, st, p->num_sms) : launch_layout_vec(a, st);
  if (e != cudaSuccess) return fail_cuda(e, gather ? "a2a gather launch" : "a2a scatter launch");
  p->last_launches += 1;
  return HCMS_OK;
}

int do_attention(hcms_plan_t* p, const void* qc, const void* kc, const void* vc, void* oc, int c, float scale,
                 cudaStream_t st, float* lse) {
  const Chunk& ck = p->chunks[c];
  AttnArgs a{qc, kc, vc, oc, p->sh.S, p->sh.D, p->sh.P, ck.h, scale};
  a.lse = lse;
  a.pair = (p->flags & HCMS_FLAG_ATTN_PAIR) != 0;
  a.cache = &p->tmaps;
  cudaError_t e = launch_attention(a, st);
  if (e != cudaSuccess) return fail_cuda(e, "attention launch");
  p->last_launches += 1;
  return HCMS_OK;
}

// ------------------------------------------------------------------------------------------
// the dual-stream chunk scheduler (Algorithm 1 lines 5-25), written once
// ------------------------------------------------------------------------------------------
constexpr int kRing = 2;     // HCMS_FLAG_RECYCLE_WS: double buffering of the chunk buffer sets

int run_pipeline(hcms_plan_t* plan, cudaStream_t caller, const PipelineSteps& steps) {
  const int C = plan->sh.C;
  const bool serial = plan->flags & HCMS_FLAG_SERIAL;
  const bool split = steps.split_out && !serial;
  // S_comp: two CUDA streams alternating by chunk parity (see HCMS_FLAG_SINGLE_COMP in hcms.h)
  const bool dual_comp = !serial && !(plan->flags & HCMS_FLAG_SINGLE_COMP) && C > 1;
  cudaStream_t s_in = serial ? caller : plan->s_comm;
  cudaStream_t s_out = serial ? caller : (split ? plan->s_comm_out : plan->s_comm);
  auto comp_stream = [&](int c) { return serial ? caller : ((dual_comp && (c & 1)) ? plan->s_comp2 : plan->s_comp); };
  auto mark = [&](int step, int c, int side, cudaStream_t s) -> cudaError_t {
    if (!steps.profile) return cudaSuccess;
    const size_t slot = static_cast<size_t>(plan->prof_calls % HCMS_PROFILE_RING) * C + c;
    return cudaEventRecord(plan->prof[step][side][slot], s);
  };
  // the streams this call forks, in the order of plan->e_fin
  cudaStream_t forked[4] = {plan->s_comm, plan->s_comp, dual_comp ? plan->s_comp2 : nullptr, split ? plan->s_comm_out : nullptr};
  bool did_fork = false;
  int st = HCMS_OK;
  auto cuda = [&](cudaError_t e, const char* what) {      // first failure wins; later steps are skipped
    if (e != cudaSuccess && st == HCMS_OK) st = fail_cuda(e, what);
    return st == HCMS_OK;
  };

  if (!serial) {
    if (cuda(cudaEventRecord(plan->e_main, caller), "record E_main")) {         // Alg. 1 line 5
      did_fork = true;
      for (cudaStream_t s : forked)                                             // lines 7, 13
        if (s) cuda(cudaStreamWaitEvent(s, plan->e_main, 0), "wait E_main");
    }
  }
  // A_c^in on S_comm (lines 8-11), then E_c^comm
  auto do_in = [&](int c) {
    if (!steps.comm_in || st != HCMS_OK) return;
    if (!cuda(mark(0, c, 0, s_in), "profile event")) return;
    const int r = steps.comm_in(c, s_in);
    if (r != HCMS_OK) { st = r; return; }
    if (!cuda(mark(0, c, 1, s_in), "profile event")) return;
    if (!serial) cuda(cudaEventRecord(plan->e_comm[c], s_in), "record E_c^comm");
  };
  // Attn_c on S_comp (lines 14-18) after wait(E_c^comm) (Eq. 6), then E_c^comp
  auto do_compute = [&](int c) {
    if (!steps.compute || st != HCMS_OK) return;
    cudaStream_t s = comp_stream(c);
    if (!serial && steps.comm_in && !(plan->flags & HCMS_FLAG_DEBUG_NO_COMM_WAIT))
      if (!cuda(cudaStreamWaitEvent(s, plan->e_comm[c], 0), "wait E_c^comm")) return;
    if (!cuda(mark(1, c, 0, s), "profile event")) return;
    const int r = steps.compute(c, s);
    if (r != HCMS_OK) { st = r; return; }
    if (!cuda(mark(1, c, 1, s), "profile event")) return;
    if (!serial) cuda(cudaEventRecord(plan->e_comp[c], s), "record E_c^comp");
  };
  // A_c^out on S_comm (lines 20-23) after wait(E_c^comp) (Eq. 7)
  auto do_out = [&](int c) {
    if (!steps.comm_out || st != HCMS_OK) return;
    if (!serial && steps.compute)
      if (!cuda(cudaStreamWaitEvent(s_out, plan->e_comp[c], 0), "wait E_c^comp")) return;
    if (!cuda(mark(2, c, 0, s_out), "profile event")) return;
    const int r = steps.comm_out(c, s_out);
    if (r != HCMS_OK) { st = r; return; }
    cuda(mark(2, c, 1, s_out), "profile event");
  };
  if (steps.ring <= 0) {
    // Alg. 1's order: the three phases one after the other (every chunk has its own buffers)
    for (int c = 0; c < C; ++c) do_in(c);
    for (int c = 0; c < C; ++c) do_compute(c);
    for (int c = 0; c < C; ++c) do_out(c);
  } else {
    // HCMS_FLAG_RECYCLE_WS: chunk c lives in buffer set c % ring, so A_c^in may only run once A_{c-ring}^out has
    // emptied that set.  S_comm's own order expresses it: ... A_{c-ring}^out, A_c^in ... (A^out waits for E^comp of a
    // computation that was enqueued in an earlier iteration, so every event is recorded before it is waited on).
    for (int c = 0; c < C + steps.ring; ++c) {
      if (c >= steps.ring) do_out(c - steps.ring);
      if (c < C) {
        do_in(c);
        do_compute(c);
      }
    }
  }
  if (steps.profile && st == HCMS_OK) plan->prof_calls += 1;
  // line 25: Synchronize(S_comm, S_comp) -- expressed as stream waits, the host is not blocked.  Also on the error
  // paths: whatever was enqueued before the failure is joined, so no side stream stays forked from the caller.
  if (did_fork) {
    const int keep = st;
    for (int i = 0; i < 4; ++i) {
      if (!forked[i]) continue;
      cudaError_t e = cudaEventRecord(plan->e_fin[i], forked[i]);
      if (e == cudaSuccess) e = cudaStreamWaitEvent(caller, plan->e_fin[i], 0);
      if (e != cudaSuccess && st == HCMS_OK) st = fail_cuda(e, "join");
    }
    if (keep != HCMS_OK) st = keep;
  }
  return st;
}

}  // namespace hcms

using namespace hcms;

static int elem_size(int dtype) {
  switch (dtype) {
    case HCMS_DTYPE_BF16:
    case HCMS_DTYPE_F16:
      return 2;
    case HCMS_DTYPE_F32:
      return 4;
    default:
      return 0;
  }
}

extern "C" {

int hcms_version(void) { return HCMS_VERSION; }

const char* hcms_status_string(int status) {
  switch (status) {
    case HCMS_OK: return "HCMS_OK";
    case HCMS_ERR_INVALID_ARG: return "HCMS_ERR_INVALID_ARG";
    case HCMS_ERR_UNSUPPORTED_SHAPE: return "HCMS_ERR_UNSUPPORTED_SHAPE";
    case HCMS_ERR_UNSUPPORTED_DTYPE: return "HCMS_ERR_UNSUPPORTED_DTYPE";
    case HCMS_ERR_UNSUPPORTED_DEVICE: return "HCMS_ERR_UNSUPPORTED_DEVICE";
    case HCMS_ERR_MISALIGNED: return "HCMS_ERR_MISALIGNED";
    case HCMS_ERR_ALIAS: return "HCMS_ERR_ALIAS";
    case HCMS_ERR_PLAN_MISMATCH: return "HCMS_ERR_PLAN_MISMATCH";
    case HCMS_ERR_WORKSPACE_TOO_SMALL: return "HCMS_ERR_WORKSPACE_TOO_SMALL";
    case HCMS_ERR_CUDA: return "HCMS_ERR_CUDA";
    default: return "HCMS_ERR_UNKNOWN";
  }
}

const char* hcms_last_error(void) { return g_last_error; }

int hcms_chunk_table_host(int heads_per_rank, int C, int* o, int* h) { return chunk_table(heads_per_rank, C, o, h); }

double hcms_model_t_hcms(int C, double t0, double t_comm, double t_attn, double beta) {
  if (C <= 0) return NAN;
  return t0 + t_comm / C + t_attn + C * beta;  // Eq. 10 (L417)
}
double hcms_model_c_star(double t_comm, double beta) {
  if (!(beta > 0) || !(t_comm >= 0)) return NAN;
  return std::sqrt(t_comm / beta);  // Theorem 1 (L156, L421)
}
double hcms_model_speedup(int C, double rho, double beta, double t_total) {
  if (C <= 0 || !(t_total > 0)) return NAN;
  return 1.0 / (1.0 - rho * (C - 1) / C + C * beta / t_total);  // Eq. 11 (L427)
}
double hcms_model_s_max(double rho) {
  if (!(rho < 1)) return NAN;
  return 1.0 / (1.0 - rho);  // Theorem 2 (L158, L429)
}
int hcms_model_choose_chunks(int heads_per_rank, double t_comm, double beta) {
  if (heads_per_rank <= 0 || std::isnan(t_comm) || std::isnan(beta)) return 0;
  if (!(t_comm > 0)) return 1;
  if (!(beta > 0)) return heads_per_rank;
  const double c_star = std::sqrt(t_comm / beta);  // Theorem 1; t_comm/C + C*beta is convex in C
  auto clamp = [&](double c) { return c < 1 ? 1 : (c > heads_per_rank ? heads_per_rank : static_cast<int>(c)); };
  const int lo = clamp(std::floor(c_star)), hi = clamp(std::ceil(c_star));
  const double f_lo = t_comm / lo + lo * beta, f_hi = t_comm / hi + hi * beta;
  return f_hi < f_lo ? hi : lo;
}

int hcms_plan(hcms_plan_t** out, int64_t S, int H, int D, int P, int C, int dtype, uint32_t flags) {
  if (!out) return fail(HCMS_ERR_INVALID_ARG, "plan output pointer is NULL");
  *out = nullptr;
  if (S <= 0 || H <= 0 || D <= 0 || P <= 0 || C <= 0)
    return fail(HCMS_ERR_INVALID_ARG, "S=%lld H=%d D=%d P=%d C=%d must all be positive", static_cast<long long>(S), H, D,
                P, C);
  const int es = elem_size(dtype);
  if (es == 0) return fail(HCMS_ERR_UNSUPPORTED_DTYPE, "unknown dtype %d", dtype);
  if (S % P) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "S=%lld is not divisible by P=%d", static_cast<long long>(S), P);
  if (H % P) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "H=%d is not divisible by P=%d", H, P);
  if (D != 64 && D != 128) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "D=%d: only head dimensions 64 and 128 are built", D);
  if (S > (1ll << 30)) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "S=%lld too large", static_cast<long long>(S));
  const int Hl = H / P;
  if (C > Hl) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "C=%d exceeds heads per rank H/P=%d", C, Hl);
  if ((flags & HCMS_FLAG_GRAPH) && (flags & HCMS_FLAG_PROFILE))
    return fail(HCMS_ERR_INVALID_ARG, "HCMS_FLAG_GRAPH and HCMS_FLAG_PROFILE exclude each other (timing events cannot be read from a graph)");
  if ((flags & HCMS_FLAG_TRAINING) && dtype != HCMS_DTYPE_BF16)
    return fail(HCMS_ERR_UNSUPPORTED_DTYPE, "HCMS_FLAG_TRAINING needs a bf16 plan");
  if ((flags & HCMS_FLAG_RECYCLE_WS) && (flags & (HCMS_FLAG_TRAINING | HCMS_FLAG_FUSE_A2A | HCMS_FLAG_SPLIT_COMM | HCMS_FLAG_DEBUG_ATTN_ONLY)))
    return fail(HCMS_ERR_INVALID_ARG, "HCMS_FLAG_RECYCLE_WS excludes TRAINING (the backward reads every chunk's saved buffers), "
                "FUSE_A2A (the projection writes all chunks at once), SPLIT_COMM and DEBUG_ATTN_ONLY");

  int dev = 0, sms = 0;
  int st = device_sms(&sms);          // also: a CUDA device exists and is sm_100
  if (st) return st;
  HCMS_CUDA(cudaGetDevice(&dev));

  hcms_plan_t* p = new (std::nothrow) hcms_plan_t();
  if (!p) return fail(HCMS_ERR_INVALID_ARG, "out of host memory");
  p->sh = Shape{S, H, D, P, C, es, Hl};
  p->dtype = dtype;
  p->flags = flags;
  p->device = dev;
  p->num_sms = sms;
  p->chunks.resize(C);
  std::vector<int> o(C), h(C);
  chunk_table(Hl, C, o.data(), h.data());
  size_t off = 0;
  // HCMS_FLAG_RECYCLE_WS: kRing buffer sets, each sized for a largest chunk (Eq. 3: chunk 0); chunk c uses set c % kRing
  p->ring = (flags & HCMS_FLAG_RECYCLE_WS) && C > kRing ? kRing : 0;
  const size_t set_stride = 4 * align_up(static_cast<size_t>(P) * S * h[0] * D * es, 1024);
  for (int c = 0; c < C; ++c) {
    Chunk& ck = p->chunks[c];
    ck.o = o[c];
    ck.h = h[c];
    ck.bytes = static_cast<size_t>(P) * S * h[c] * D * es;
    if (p->ring) off = static_cast<size_t>(c % p->ring) * set_stride;
    for (int t = 0; t < 4; ++t) {
      ck.off[t] = off;
      off += align_up(ck.bytes, 1024);
    }
  }
  p->ws_bytes = p->ring ? p->ring * set_stride : off;

  auto bail = [&](int status) {
    plan_free(p);
    return status;
  };
#define PLAN_CUDA(expr)                                              \
  do {                                                               \
    cudaError_t e__ = (expr);                                        \
    if (e__ != cudaSuccess) return bail(fail_cuda(e__, #expr));      \
  } while (0)
  int prio_lo = 0, prio_hi = 0;
  PLAN_CUDA(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
  // the communication stream outranks the compute stream so that copy CTAs are placed as soon as
  // an SM has room, instead of queueing behind the attention grid
  PLAN_CUDA(cudaStreamCreateWithPriority(&p->s_comm, cudaStreamNonBlocking, prio_hi));
  PLAN_CUDA(cudaStreamCreateWithPriority(&p->s_comm_out, cudaStreamNonBlocking, prio_hi));
  PLAN_CUDA(cudaStreamCreateWithPriority(&p->s_comp, cudaStreamNonBlocking, prio_lo));
  PLAN_CUDA(cudaStreamCreateWithPriority(&p->s_comp2, cudaStreamNonBlocking, prio_lo));
  if (flags & HCMS_FLAG_GRAPH) PLAN_CUDA(cudaStreamCreateWithFlags(&p->s_cap, cudaStreamNonBlocking));
  PLAN_CUDA(cudaEventCreateWithFlags(&p->e_main, cudaEventDisableTiming));
  for (auto& e : p->e_fin) PLAN_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  p->e_comm.assign(C, nullptr);
  p->e_comp.assign(C, nullptr);
  for (int c = 0; c < C; ++c) {
    PLAN_CUDA(cudaEventCreateWithFlags(&p->e_comm[c], cudaEventDisableTiming));
    PLAN_CUDA(cudaEventCreateWithFlags(&p->e_comp[c], cudaEventDisableTiming));
  }
  if (flags & HCMS_FLAG_PROFILE) {
    for (auto& step : p->prof)
      for (auto& side : step) {
        side.assign(static_cast<size_t>(C) * HCMS_PROFILE_RING, nullptr);
        for (auto& e : side) PLAN_CUDA(cudaEventCreate(&e));
      }
    for (auto& e : p->e_layer) PLAN_CUDA(cudaEventCreate(&e));
  }
  // kernel attributes (MaxDynamicSharedMemorySize) of every kernel the plan can launch, once per device
  if (dtype == HCMS_DTYPE_BF16) {
    PLAN_CUDA(attention_init());
    PLAN_CUDA(attention_bwd_init());
    PLAN_CUDA(gemm_init());
  }
  if (flags & (HCMS_FLAG_HOST_ROUTE_Q | HCMS_FLAG_HOST_ROUTE_K | HCMS_FLAG_HOST_ROUTE_V | HCMS_FLAG_HOST_ROUTE_O)) {
    size_t max_chunk = 0;
    for (auto& ck : p->chunks) max_chunk = ck.bytes > max_chunk ? ck.bytes : max_chunk;
    for (int t = 0; t < 4; ++t)
      if (flags & (HCMS_FLAG_HOST_ROUTE_Q << t)) {
        PLAN_CUDA(cudaMallocHost(&p->pinned[t], max_chunk));
        PLAN_CUDA(cudaMalloc(&p->wire[t], max_chunk));
      }
  }
#undef PLAN_CUDA
  // The chunk workspace (and, under HCMS_FLAG_TRAINING, the gradient workspace and lse) is allocated on first use,
  // so a caller that supplies its own through hcms_plan_set_workspace never pays for a transient second copy.
  *out = p;
  return HCMS_OK;
}

int hcms_plan_destroy(hcms_plan_t* plan) {
  plan_free(plan);
  return HCMS_OK;
}

size_t hcms_plan_workspace_bytes(const hcms_plan_t* plan) { return plan ? plan->ws_bytes : 0; }
void* hcms_plan_workspace(hcms_plan_t* plan) {
  if (!plan || ensure_workspace(plan) != HCMS_OK) return nullptr;
  return plan->ws;
}
long long hcms_plan_tensor_map_encodes(const hcms_plan_t* plan) { return plan ? plan->tmaps.encodes : 0; }

int hcms_plan_set_workspace(hcms_plan_t* plan, void* dev, size_t bytes) {
  if (!plan || !dev) return fail(HCMS_ERR_INVALID_ARG, "plan or workspace pointer is NULL");
  if (reinterpret_cast<uintptr_t>(dev) % 256) return fail(HCMS_ERR_MISALIGNED, "workspace must be 256-byte aligned");
  if (bytes < plan->ws_bytes)
    return fail(HCMS_ERR_WORKSPACE_TOO_SMALL, "workspace has %zu bytes, plan needs %zu", bytes, plan->ws_bytes);
  if (plan->ws_owned && plan->ws) {
    for (cudaStream_t s : {plan->s_comm, plan->s_comm_out, plan->s_comp, plan->s_comp2}) cudaStreamSynchronize(s);
    cudaFree(plan->ws);
  }
  plan->ws = dev;
  plan->ws_owned = false;
  // a captured graph has the previous workspace's addresses baked into every node, and the backward reads what the
  // forward saved in the workspace: both are void now
  if (plan->graph_exec) {
    cudaGraphExecDestroy(plan->graph_exec);
    plan->graph_exec = nullptr;
  }
  std::memset(plan->graph_key, 0, sizeof(plan->graph_key));
  plan->forward_done = false;
  return HCMS_OK;
}

int hcms_chunk_table(const hcms_plan_t* plan, int* o, int* h) {
  if (!plan) return fail(HCMS_ERR_INVALID_ARG, "plan is NULL");
  for (int c = 0; c < plan->sh.C; ++c) {
    if (o) o[c] = plan->chunks[c].o;
    if (h) h[c] = plan->chunks[c].h;
  }
  return HCMS_OK;
}

int hcms_chunk_layout(const hcms_plan_t* plan, int c, size_t* bytes, size_t* q_off, size_t* k_off, size_t* v_off,
                      size_t* o_off) {
  if (!plan) return fail(HCMS_ERR_INVALID_ARG, "plan is NULL");
  if (c < 0 || c >= plan->sh.C) return fail(HCMS_ERR_PLAN_MISMATCH, "chunk %d outside [0,%d)", c, plan->sh.C);
  const Chunk& ck = plan->chunks[c];
  if (bytes) *bytes = ck.bytes;
  if (q_off) *q_off = ck.off[0];
  if (k_off) *k_off = ck.off[1];
  if (v_off) *v_off = ck.off[2];
  if (o_off) *o_off = ck.off[3];
  return HCMS_OK;
}

int hcms_plan_last_launch_count(const hcms_plan_t* plan) { return plan ? plan->last_launches : 0; }

}  // extern "C"

// ------------------------------------------------------------------------------------------
// single steps
// ------------------------------------------------------------------------------------------
extern "C" {

int hcms_a2a_scatter(hcms_plan_t* plan, int n_tensors, const void* const* src, void* const* dst, int c, void* stream) {
  if (!plan || !src || !dst) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (n_tensors < 1 || n_tensors > 3) return fail(HCMS_ERR_INVALID_ARG, "n_tensors=%d must be 1..3", n_tensors);
  if (c < 0 || c >= plan->sh.C) return fail(HCMS_ERR_PLAN_MISMATCH, "chunk %d outside [0,%d)", c, plan->sh.C);
  for (int t = 0; t < n_tensors; ++t) {
    if (!src[t] || !dst[t]) return fail(HCMS_ERR_INVALID_ARG, "tensor %d pointer is NULL", t);
    if (!aligned16(src[t]) || !aligned16(dst[t])) return fail(HCMS_ERR_MISALIGNED, "tensor %d is not 16-byte aligned", t);
  }
  int st = check_plan_device(plan);
  if (st) return st;
  plan->last_launches = 0;
  return do_layout(plan, n_tensors, src, dst, c, false, static_cast<cudaStream_t>(stream));
}

int hcms_a2a_gather(hcms_plan_t* plan, const void* src, void* dst, int c, void* stream) {
  if (!plan || !src || !dst) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (c < 0 || c >= plan->sh.C) return fail(HCMS_ERR_PLAN_MISMATCH, "chunk %d outside [0,%d)", c, plan->sh.C);
  if (!aligned16(src) || !aligned16(dst)) return fail(HCMS_ERR_MISALIGNED, "pointer is not 16-byte aligned");
  int st = check_plan_device(plan);
  if (st) return st;
  const void* s[1] = {src};
  void* d[1] = {dst};
  plan->last_launches = 0;
  return do_layout(plan, 1, s, d, c, true, static_cast<cudaStream_t>(stream));
}

int hcms_attention_chunk(hcms_plan_t* plan, const void* qc, const void* kc, const void* vc, void* oc, int c, float scale,
                         void* stream) {
  if (!plan || !qc || !kc || !vc || !oc) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (plan->dtype != HCMS_DTYPE_BF16) return fail(HCMS_ERR_UNSUPPORTED_DTYPE, "attention needs a bf16 plan");
  if (c < 0 || c >= plan->sh.C) return fail(HCMS_ERR_PLAN_MISMATCH, "chunk %d outside [0,%d)", c, plan->sh.C);
  if (!aligned16(qc) || !aligned16(kc) || !aligned16(vc) || !aligned16(oc))
    return fail(HCMS_ERR_MISALIGNED, "pointer is not 16-byte aligned");
  int st = check_scale(scale);
  if (st) return st;
  if ((st = check_plan_device(plan)) != HCMS_OK) return st;
  plan->last_launches = 0;
  return do_attention(plan, qc, kc, vc, oc, c, scale, static_cast<cudaStream_t>(stream));
}

}  // extern "C"

// ------------------------------------------------------------------------------------------
// hcms_attention_forward: Algorithm 1 lines 4-25 on device tensors
// ------------------------------------------------------------------------------------------
// Enqueue Alg. 1 lines 4-25 for validated arguments: kernels, copies, event records and waits; no host synchronisation.
static int enqueue_forward(hcms_plan_t* plan, const void* q, const void* k, const void* v, void* out, float scale,
                           cudaStream_t caller) {
  char* ws = static_cast<char*>(plan->ws);
  plan->last_launches = 0;
  // The emulated wire of BASELINE.json configs[4]: a routed tensor's chunk is produced into the plan's
  // device send buffer, crosses to pinned host memory and comes back into the buffer its consumer reads
  // (scatter -> wire -> D2H -> H2D -> Q'_c/K'_c/V'_c;  O'_c -> D2H -> H2D -> wire -> gather).  Same bits.
  auto routed = [&](int t) { return (plan->flags & (HCMS_FLAG_HOST_ROUTE_Q << t)) != 0; };
  auto host_hop = [&](int t, const void* from, void* to, size_t bytes, cudaStream_t s) -> int {
    HCMS_CUDA(cudaMemcpyAsync(plan->pinned[t], from, bytes, cudaMemcpyDeviceToHost, s));
    HCMS_CUDA(cudaMemcpyAsync(to, plan->pinned[t], bytes, cudaMemcpyHostToDevice, s));
    plan->last_launches += 2;
    return HCMS_OK;
  };
  const bool attn_only = plan->flags & HCMS_FLAG_DEBUG_ATTN_ONLY;
  PipelineSteps steps;
  steps.split_out = plan->flags & HCMS_FLAG_SPLIT_COMM;
  steps.profile = plan->flags & HCMS_FLAG_PROFILE;
  steps.ring = plan->ring;
  steps.comm_in = [&](int c, cudaStream_t s) -> int {           // line 8: AllToAll(Q_c, K_c, V_c), one launch
    if (attn_only) return HCMS_OK;
    const Chunk& ck = plan->chunks[c];
    const void* src[3] = {q, k, v};
    void* dst[3];
    for (int t = 0; t < 3; ++t) dst[t] = routed(t) ? plan->wire[t] : static_cast<void*>(ws + ck.off[t]);
    int st = do_layout(plan, 3, src, dst, c, false, s);
    for (int t = 0; t < 3 && st == HCMS_OK; ++t)
      if (routed(t)) st = host_hop(t, plan->wire[t], ws + ck.off[t], ck.bytes, s);
    return st;
  };
  steps.compute = [&](int c, cudaStream_t s) -> int {           // line 15
    const Chunk& ck = plan->chunks[c];
    float* lse_c = plan->lse ? plan->lse + static_cast<size_t>(plan->sh.P) * plan->sh.S * ck.o : nullptr;   // [P*h_c][S]
    return do_attention(plan, ws + ck.off[0], ws + ck.off[1], ws + ck.off[2], ws + ck.off[3], c, scale, s, lse_c);
  };
  steps.comm_out = [&](int c, cudaStream_t s) -> int {          // line 21 + Concat (line 26)
    if (attn_only) return HCMS_OK;
    const Chunk& ck = plan->chunks[c];
    if (routed(3)) {
      const int st = host_hop(3, ws + ck.off[3], plan->wire[3], ck.bytes, s);
      if (st) return st;
    }
    const void* src[1] = {routed(3) ? plan->wire[3] : static_cast<const void*>(ws + ck.off[3])};
    void* dst[1] = {out};
    return do_layout(plan, 1, src, dst, c, true, s);
  };
  const int st = run_pipeline(plan, caller, steps);
  if (st == HCMS_OK) {
    plan->forward_done = true;
    plan->forward_scale = scale;
  }
  return st;
}

// HCMS_FLAG_GRAPH: the whole chunk pipeline (kernels on S_comm / S_comp, the event forks and joins of Eq. 6-7) is
// captured once into a CUDA graph on a plan-owned stream and replayed with one launch per call; a call with other
// tensors or another scale captures again, and so does the first call after hcms_plan_set_workspace.  The capture
// runs on the plan's own stream because the caller's may be the legacy default stream, which cannot be captured.
static int forward_graph(hcms_plan_t* plan, const void* q, const void* k, const void* v, void* out, float scale,
                         cudaStream_t caller) {
  const void* key[4] = {q, k, v, out};
  const bool hit = plan->graph_exec && std::memcmp(key, plan->graph_key, sizeof(key)) == 0 &&
                   std::memcmp(&scale, &plan->graph_scale, sizeof(float)) == 0;
  if (!hit) {
    if (plan->graph_exec) {
      HCMS_CUDA(cudaGraphExecDestroy(plan->graph_exec));
      plan->graph_exec = nullptr;
    }
    HCMS_CUDA(cudaStreamBeginCapture(plan->s_cap, cudaStreamCaptureModeRelaxed));
    const int st = enqueue_forward(plan, q, k, v, out, scale, plan->s_cap);
    cudaGraph_t graph = nullptr;
    const cudaError_t ce = cudaStreamEndCapture(plan->s_cap, &graph);   // always ends the capture, also after a failure
    if (st != HCMS_OK) {
      if (graph) cudaGraphDestroy(graph);
      cudaGetLastError();
      return st;
    }
    if (ce != cudaSuccess) return fail_cuda(ce, "cudaStreamEndCapture");
    const cudaError_t ci = cudaGraphInstantiate(&plan->graph_exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ci != cudaSuccess) {
      plan->graph_exec = nullptr;
      return fail_cuda(ci, "cudaGraphInstantiate");
    }
    std::memcpy(plan->graph_key, key, sizeof(key));
    plan->graph_scale = scale;
    plan->graph_launches = plan->last_launches;
    plan->graph_captures += 1;
  }
  HCMS_CUDA(cudaGraphLaunch(plan->graph_exec, caller));
  plan->last_launches = plan->graph_launches;
  plan->forward_done = true;
  plan->forward_scale = scale;
  return HCMS_OK;
}

extern "C" {

int hcms_attention_forward(hcms_plan_t* plan, const void* q, const void* k, const void* v, void* out, int64_t S, int H,
                           int D, int P, int C, float scale, void* stream) {
  if (!plan || !q || !k || !v || !out) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  const Shape& sh = plan->sh;
  if (S != sh.S || H != sh.H || D != sh.D || P != sh.P || C != sh.C)
    return fail(HCMS_ERR_PLAN_MISMATCH, "call (S=%lld,H=%d,D=%d,P=%d,C=%d) != plan (S=%lld,H=%d,D=%d,P=%d,C=%d)",
                static_cast<long long>(S), H, D, P, C, static_cast<long long>(sh.S), sh.H, sh.D, sh.P, sh.C);
  if (plan->dtype != HCMS_DTYPE_BF16) return fail(HCMS_ERR_UNSUPPORTED_DTYPE, "attention needs a bf16 plan");
  int st = check_scale(scale);
  if (st) return st;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(out))
    return fail(HCMS_ERR_MISALIGNED, "q, k, v and out must be 16-byte aligned");
  const size_t bytes = static_cast<size_t>(S) * H * D * sh.es;
  for (const void* in : {q, k, v})
    if (overlaps(out, bytes, in, bytes)) return fail(HCMS_ERR_ALIAS, "out overlaps an input tensor");
  if ((st = check_plan_device(plan)) != HCMS_OK) return st;
  if ((st = ensure_workspace(plan)) != HCMS_OK) return st;
  if ((plan->flags & HCMS_FLAG_TRAINING) && (st = ensure_training(plan)) != HCMS_OK) return st;
  cudaStream_t caller = static_cast<cudaStream_t>(stream);
  if (plan->flags & HCMS_FLAG_GRAPH) return forward_graph(plan, q, k, v, out, scale, caller);
  return enqueue_forward(plan, q, k, v, out, scale, caller);
}

int hcms_attention_forward_host(hcms_plan_t* plan, const void* q, const void* k, const void* v, void* out, int64_t S,
                                int H, int D, int P, int C, float scale, void* stream) {
  if (!plan || !q || !k || !v || !out) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  const Shape& sh = plan->sh;
  if (S != sh.S || H != sh.H || D != sh.D || P != sh.P || C != sh.C)
    return fail(HCMS_ERR_PLAN_MISMATCH, "call shape differs from the plan's");
  const size_t bytes = static_cast<size_t>(S) * H * D * sh.es;
  cudaStream_t caller = static_cast<cudaStream_t>(stream);
  int st = check_plan_device(plan);
  if (st) return st;
  if (!(plan->flags & (HCMS_FLAG_HOST_STAGED | HCMS_FLAG_SERIAL | HCMS_FLAG_GRAPH)) && plan->dtype == HCMS_DTYPE_BF16) {
    // The host link is the wire: strided copies on the copy engines perform the all-to-all layout change themselves.
    // Chunk c of rank p's heads is a 2-D region of the host tensor (S rows of h_c*D elements, pitch H*D) and lands as
    // the dense [S][h_c][D] slab of Q'_c / K'_c / V'_c; the output all-to-all is the reverse copy from O'_c into
    // `out`.  H2D copies run on S_comm, D2H copies on the second communication stream (separate copy engines), the
    // attention of chunk c on S_comp between them, ordered by the same events as Alg. 1: no scatter / gather
    // kernels, no staging tensors, and the transfer of chunk c+1 overlaps the attention of chunk c.
    if ((st = check_scale(scale)) != HCMS_OK) return st;
    if ((st = ensure_workspace(plan)) != HCMS_OK) return st;
    if ((plan->flags & HCMS_FLAG_TRAINING) && (st = ensure_training(plan)) != HCMS_OK) return st;
    char* ws = static_cast<char*>(plan->ws);
    const size_t row = static_cast<size_t>(H) * D * sh.es;       // host pitch
    const void* host_in[3] = {q, k, v};
    plan->last_launches = 0;
    PipelineSteps steps;
    steps.split_out = plan->ring == 0;   // HCMS_FLAG_RECYCLE_WS: D2H of chunk c - ring before H2D of chunk c, on ONE stream
    steps.ring = plan->ring;
    steps.profile = plan->flags & HCMS_FLAG_PROFILE;   // same event ring as the device path: 0 = H2D, 1 = attention, 2 = D2H
    steps.comm_in = [&](int c, cudaStream_t s) -> int {
      const Chunk& ck = plan->chunks[c];
      const size_t width = static_cast<size_t>(ck.h) * D * sh.es, slab = width * S;
      for (int t = 0; t < 3; ++t)
        for (int p = 0; p < sh.P; ++p) {
          const char* src = static_cast<const char*>(host_in[t]) + (static_cast<size_t>(p) * sh.Hl + ck.o) * D * sh.es;
          HCMS_CUDA(cudaMemcpy2DAsync(ws + ck.off[t] + p * slab, width, src, row, width, S, cudaMemcpyHostToDevice, s));
          plan->last_launches += 1;
        }
      return HCMS_OK;
    };
    steps.compute = [&](int c, cudaStream_t s) -> int {
      const Chunk& ck = plan->chunks[c];
      float* lse_c = plan->lse ? plan->lse + static_cast<size_t>(sh.P) * sh.S * ck.o : nullptr;
      return do_attention(plan, ws + ck.off[0], ws + ck.off[1], ws + ck.off[2], ws + ck.off[3], c, scale, s, lse_c);
    };
    steps.comm_out = [&](int c, cudaStream_t s) -> int {
      const Chunk& ck = plan->chunks[c];
      const size_t width = static_cast<size_t>(ck.h) * D * sh.es, slab = width * S;
      for (int p = 0; p < sh.P; ++p) {
        char* dst = static_cast<char*>(out) + (static_cast<size_t>(p) * sh.Hl + ck.o) * D * sh.es;
        HCMS_CUDA(cudaMemcpy2DAsync(dst, row, ws + ck.off[3] + p * slab, width, width, S, cudaMemcpyDeviceToHost, s));
        plan->last_launches += 1;
      }
      return HCMS_OK;
    };
    st = run_pipeline(plan, caller, steps);
    const cudaError_t ce = cudaStreamSynchronize(caller);      // also after a failure: the caller's buffers are host memory
    if (st) return st;
    if (ce != cudaSuccess) return fail_cuda(ce, "cudaStreamSynchronize");
    plan->forward_done = true;
    plan->forward_scale = scale;
    return HCMS_OK;
  }
  for (int t = 0; t < 4; ++t)
    if (!plan->staging[t]) HCMS_CUDA(cudaMalloc(&plan->staging[t], bytes));
  const void* host_in[3] = {q, k, v};
  for (int t = 0; t < 3; ++t)
    HCMS_CUDA(cudaMemcpyAsync(plan->staging[t], host_in[t], bytes, cudaMemcpyHostToDevice, caller));
  st = hcms_attention_forward(plan, plan->staging[0], plan->staging[1], plan->staging[2], plan->staging[3], S, H, D,
                              P, C, scale, stream);
  if (st) {
    cudaStreamSynchronize(caller);
    return st;
  }
  HCMS_CUDA(cudaMemcpyAsync(out, plan->staging[3], bytes, cudaMemcpyDeviceToHost, caller));
  HCMS_CUDA(cudaStreamSynchronize(caller));
  return HCMS_OK;
}

int hcms_plan_graph_captures(const hcms_plan_t* plan) { return plan ? static_cast<int>(plan->graph_captures) : 0; }

int hcms_plan_timings(hcms_plan_t* plan, int calls_back, float* scatter_ms, float* attn_ms, float* gather_ms) {
  if (!plan) return fail(HCMS_ERR_INVALID_ARG, "plan is NULL");
  if (!(plan->flags & HCMS_FLAG_PROFILE)) return fail(HCMS_ERR_INVALID_ARG, "plan was made without HCMS_FLAG_PROFILE");
  if (calls_back < 0 || calls_back >= HCMS_PROFILE_RING || calls_back >= plan->prof_calls)
    return fail(HCMS_ERR_INVALID_ARG, "calls_back=%d: %lld profiled calls so far, ring keeps %d", calls_back,
                plan->prof_calls, HCMS_PROFILE_RING);
  const size_t base = static_cast<size_t>((plan->prof_calls - 1 - calls_back) % HCMS_PROFILE_RING) * plan->sh.C;
  float* outs[3] = {scatter_ms, attn_ms, gather_ms};
  for (int step = 0; step < 3; ++step)
    for (int c = 0; c < plan->sh.C; ++c) {
      HCMS_CUDA(cudaEventSynchronize(plan->prof[step][1][base + c]));
      float ms = 0.f;
      HCMS_CUDA(cudaEventElapsedTime(&ms, plan->prof[step][0][base + c], plan->prof[step][1][base + c]));
      if (outs[step]) outs[step][c] = ms;
    }
  return HCMS_OK;
}

int hcms_plan_step_span(hcms_plan_t* plan, int calls_back, int step, float* span_ms) {
  if (!plan || !span_ms) return fail(HCMS_ERR_INVALID_ARG, "plan or span_ms is NULL");
  if (!(plan->flags & HCMS_FLAG_PROFILE)) return fail(HCMS_ERR_INVALID_ARG, "plan was made without HCMS_FLAG_PROFILE");
  if (step < 0 || step > 2) return fail(HCMS_ERR_INVALID_ARG, "step=%d must be 0 (scatter), 1 (attention) or 2 (gather)", step);
  if (calls_back < 0 || calls_back >= HCMS_PROFILE_RING || calls_back >= plan->prof_calls)
    return fail(HCMS_ERR_INVALID_ARG, "calls_back=%d: %lld profiled calls so far, ring keeps %d", calls_back,
                plan->prof_calls, HCMS_PROFILE_RING);
  const size_t base = static_cast<size_t>((plan->prof_calls - 1 - calls_back) % HCMS_PROFILE_RING) * plan->sh.C;
  // chunk 0 begins first and chunk C-1 ends last on every stream arrangement (in-order streams, Eq. 6-7 waits)
  for (int c = 0; c < plan->sh.C; ++c) HCMS_CUDA(cudaEventSynchronize(plan->prof[step][1][base + c]));
  float best = 0.f;
  for (int c = 0; c < plan->sh.C; ++c) {
    float ms = 0.f;
    HCMS_CUDA(cudaEventElapsedTime(&ms, plan->prof[step][0][base], plan->prof[step][1][base + c]));
    best = ms > best ? ms : best;
  }
  *span_ms = best;
  return HCMS_OK;
}

int hcms_plan_timeline(hcms_plan_t* plan, int calls_back, float* begin_ms, float* end_ms) {
  if (!plan || !begin_ms || !end_ms) return fail(HCMS_ERR_INVALID_ARG, "plan, begin_ms or end_ms is NULL");
  if (!(plan->flags & HCMS_FLAG_PROFILE)) return fail(HCMS_ERR_INVALID_ARG, "plan was made without HCMS_FLAG_PROFILE");
  if (calls_back < 0 || calls_back >= HCMS_PROFILE_RING || calls_back >= plan->prof_calls)
    return fail(HCMS_ERR_INVALID_ARG, "calls_back=%d: %lld profiled calls so far, ring keeps %d", calls_back,
                plan->prof_calls, HCMS_PROFILE_RING);
  const int C = plan->sh.C;
  const size_t base = static_cast<size_t>((plan->prof_calls - 1 - calls_back) % HCMS_PROFILE_RING) * C;
  for (int step = 0; step < 3; ++step)
    for (int c = 0; c < C; ++c) HCMS_CUDA(cudaEventSynchronize(plan->prof[step][1][base + c]));
  cudaEvent_t origin = plan->prof[0][0][base];  // chunk 0's scatter begins first (Alg. 1 order on S_comm)
  for (int step = 0; step < 3; ++step)
    for (int c = 0; c < C; ++c) {
      HCMS_CUDA(cudaEventElapsedTime(&begin_ms[step * C + c], origin, plan->prof[step][0][base + c]));
      HCMS_CUDA(cudaEventElapsedTime(&end_ms[step * C + c], origin, plan->prof[step][1][base + c]));
    }
  return HCMS_OK;
}

}  // extern "C"
