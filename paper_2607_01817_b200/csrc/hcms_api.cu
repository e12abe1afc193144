// libhcms entry points: plan, chunk table, dual-stream chunk scheduler (section 3.4-3.6,
// Algorithm 1), single-step hooks, host-buffer convenience call.  See include/hcms.h.
#include <cmath>
#include <cstdarg>
#include <cstring>
#include <new>

#include "hcms_internal.h"

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

}  // namespace hcms

using namespace hcms;

// ------------------------------------------------------------------------------------------
// plan
// ------------------------------------------------------------------------------------------
struct hcms_plan {
  Shape sh{};
  int dtype = 0;
  uint32_t flags = 0;
  int device = 0;
  int num_sms = 0;
  std::vector<Chunk> chunks;
  size_t ws_bytes = 0;
  void* ws = nullptr;
  bool ws_owned = false;
  cudaStream_t s_comm = nullptr, s_comm_out = nullptr, s_comp = nullptr, s_comp2 = nullptr;
  cudaEvent_t e_main = nullptr, e_fin_comm = nullptr, e_fin_comp = nullptr, e_fin_comp2 = nullptr, e_fin_in = nullptr;
  std::vector<cudaEvent_t> e_comm, e_comp;
  // host route (config 5): per routed tensor one pinned host buffer and one device "send/receive" buffer,
  // each as large as the largest chunk tensor
  void* pinned[4] = {nullptr, nullptr, nullptr, nullptr};
  void* wire[4] = {nullptr, nullptr, nullptr, nullptr};
  // host-buffer entry point staging
  void* staging[4] = {nullptr, nullptr, nullptr, nullptr};
  int last_launches = 0;
  // hcms_layer_forward: q,k,v,o [S,H,D] (allocated on first use) and, under HCMS_FLAG_PROFILE, 4 events
  void* layer_buf[4] = {nullptr, nullptr, nullptr, nullptr};
  cudaEvent_t e_layer[4] = {nullptr, nullptr, nullptr, nullptr};
  bool layer_timed = false;
  // HCMS_FLAG_TRAINING: gradient chunk buffers dO'_c, dQ'_c, dK'_c, dV'_c (same offsets as the forward's), lse [H][S]
  void* train_ws = nullptr;
  float* lse = nullptr;
  void* stats = nullptr;      // packed {lse*log2e, delta}: [H][s_pad] float2 (lazily allocated)
  bool forward_done = false;
  // HCMS_FLAG_GRAPH: the captured chunk pipeline of the last (q, k, v, out, scale) and the stream it was captured on
  cudaStream_t s_cap = nullptr;
  cudaGraphExec_t graph_exec = nullptr;
  const void* graph_key[4] = {nullptr, nullptr, nullptr, nullptr};
  float graph_scale = 0.f;
  int graph_launches = 0;
  long long graph_captures = 0;
  // HCMS_FLAG_PROFILE: [step 0=scatter,1=attention,2=gather][begin,end][ring slot * C + chunk]
  std::vector<cudaEvent_t> prof[3][2];
  long long prof_calls = 0;   // forward calls that recorded a full set of events
};

static void plan_free(hcms_plan_t* p) {
  if (!p) return;
  if (p->s_comm) cudaStreamSynchronize(p->s_comm);
  if (p->s_comm_out) cudaStreamSynchronize(p->s_comm_out);
  if (p->s_comp) cudaStreamSynchronize(p->s_comp);
  if (p->s_comp2) cudaStreamSynchronize(p->s_comp2);
  for (auto e : p->e_comm) cudaEventDestroy(e);
  for (auto e : p->e_comp) cudaEventDestroy(e);
  if (p->e_main) cudaEventDestroy(p->e_main);
  if (p->e_fin_comm) cudaEventDestroy(p->e_fin_comm);
  if (p->e_fin_comp) cudaEventDestroy(p->e_fin_comp);
  if (p->e_fin_comp2) cudaEventDestroy(p->e_fin_comp2);
  if (p->e_fin_in) cudaEventDestroy(p->e_fin_in);
  for (auto& step : p->prof)
    for (auto& side : step)
      for (auto e : side)
        if (e) cudaEventDestroy(e);
  if (p->s_comm) cudaStreamDestroy(p->s_comm);
  if (p->s_comm_out) cudaStreamDestroy(p->s_comm_out);
  if (p->s_comp) cudaStreamDestroy(p->s_comp);
  if (p->s_comp2) cudaStreamDestroy(p->s_comp2);
  if (p->ws_owned && p->ws) cudaFree(p->ws);
  for (auto& h : p->pinned)
    if (h) cudaFreeHost(h);
  for (auto& d : p->wire)
    if (d) cudaFree(d);
  for (auto& d : p->staging)
    if (d) cudaFree(d);
  for (auto& d : p->layer_buf)
    if (d) cudaFree(d);
  if (p->graph_exec) cudaGraphExecDestroy(p->graph_exec);
  if (p->s_cap) cudaStreamDestroy(p->s_cap);
  if (p->train_ws) cudaFree(p->train_ws);
  if (p->lse) cudaFree(p->lse);
  if (p->stats) cudaFree(p->stats);
  for (auto& e : p->e_layer)
    if (e) cudaEventDestroy(e);
  delete p;
}

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

  int dev = 0, n = 0;
  cudaError_t ce = cudaGetDeviceCount(&n);
  if (ce != cudaSuccess || n == 0) {
    cudaGetLastError();
    return fail(HCMS_ERR_UNSUPPORTED_DEVICE, "no CUDA device (%s); libhcms has no CPU fallback",
                ce == cudaSuccess ? "count is 0" : cudaGetErrorString(ce));
  }
  HCMS_CUDA(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  HCMS_CUDA(cudaGetDeviceProperties(&prop, dev));
  if (prop.major != 10)
    return fail(HCMS_ERR_UNSUPPORTED_DEVICE, "device %d is sm_%d%d; libhcms is built for sm_100a only", dev, prop.major,
                prop.minor);

  hcms_plan_t* p = new (std::nothrow) hcms_plan_t();
  if (!p) return fail(HCMS_ERR_INVALID_ARG, "out of host memory");
  p->sh = Shape{S, H, D, P, C, es, Hl};
  p->dtype = dtype;
  p->flags = flags;
  p->device = dev;
  p->num_sms = prop.multiProcessorCount;
  p->chunks.resize(C);
  std::vector<int> o(C), h(C);
  chunk_table(Hl, C, o.data(), h.data());
  size_t off = 0;
  for (int c = 0; c < C; ++c) {
    Chunk& ck = p->chunks[c];
    ck.o = o[c];
    ck.h = h[c];
    ck.bytes = static_cast<size_t>(P) * S * h[c] * D * es;
    for (int t = 0; t < 4; ++t) {
      ck.off[t] = off;
      off += align_up(ck.bytes, 1024);
    }
  }
  p->ws_bytes = off;

  auto bail = [&](int st) {
    plan_free(p);
    return st;
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
  PLAN_CUDA(cudaEventCreateWithFlags(&p->e_fin_comm, cudaEventDisableTiming));
  PLAN_CUDA(cudaEventCreateWithFlags(&p->e_fin_comp, cudaEventDisableTiming));
  PLAN_CUDA(cudaEventCreateWithFlags(&p->e_fin_comp2, cudaEventDisableTiming));
  PLAN_CUDA(cudaEventCreateWithFlags(&p->e_fin_in, cudaEventDisableTiming));
  p->e_comm.assign(C, nullptr);
  p->e_comp.assign(C, nullptr);
  for (int c = 0; c < C; ++c) {
    PLAN_CUDA(cudaEventCreateWithFlags(&p->e_comm[c], cudaEventDisableTiming));
    PLAN_CUDA(cudaEventCreateWithFlags(&p->e_comp[c], cudaEventDisableTiming));
  }
  if (flags & HCMS_FLAG_PROFILE)
    for (auto& step : p->prof)
      for (auto& side : step) {
        side.assign(static_cast<size_t>(C) * HCMS_PROFILE_RING, nullptr);
        for (auto& e : side) PLAN_CUDA(cudaEventCreate(&e));
      }
  if (flags & HCMS_FLAG_PROFILE)
    for (auto& e : p->e_layer) PLAN_CUDA(cudaEventCreate(&e));
  PLAN_CUDA(cudaMalloc(&p->ws, p->ws_bytes));
  p->ws_owned = true;
  if (dtype == HCMS_DTYPE_BF16) PLAN_CUDA(attention_init());
  if (dtype == HCMS_DTYPE_BF16) PLAN_CUDA(attention_bwd_init());
  if (flags & HCMS_FLAG_TRAINING) {
    if (dtype != HCMS_DTYPE_BF16) return bail(fail(HCMS_ERR_UNSUPPORTED_DTYPE, "HCMS_FLAG_TRAINING needs a bf16 plan"));
    PLAN_CUDA(cudaMalloc(&p->train_ws, p->ws_bytes));
    PLAN_CUDA(cudaMalloc(reinterpret_cast<void**>(&p->lse), static_cast<size_t>(H) * S * sizeof(float)));
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
  *out = p;
  return HCMS_OK;
}

int hcms_plan_destroy(hcms_plan_t* plan) {
  plan_free(plan);
  return HCMS_OK;
}

size_t hcms_plan_workspace_bytes(const hcms_plan_t* plan) { return plan ? plan->ws_bytes : 0; }
void* hcms_plan_workspace(const hcms_plan_t* plan) { return plan ? plan->ws : nullptr; }

int hcms_plan_set_workspace(hcms_plan_t* plan, void* dev, size_t bytes) {
  if (!plan || !dev) return fail(HCMS_ERR_INVALID_ARG, "plan or workspace pointer is NULL");
  if (reinterpret_cast<uintptr_t>(dev) % 256) return fail(HCMS_ERR_MISALIGNED, "workspace must be 256-byte aligned");
  if (bytes < plan->ws_bytes)
    return fail(HCMS_ERR_WORKSPACE_TOO_SMALL, "workspace has %zu bytes, plan needs %zu", bytes, plan->ws_bytes);
  if (plan->ws_owned && plan->ws) {
    cudaStreamSynchronize(plan->s_comm);
    cudaStreamSynchronize(plan->s_comm_out);
    cudaStreamSynchronize(plan->s_comp);
    cudaStreamSynchronize(plan->s_comp2);
    cudaFree(plan->ws);
  }
  plan->ws = dev;
  plan->ws_owned = false;
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
static bool aligned16(const void* p) { return reinterpret_cast<uintptr_t>(p) % 16 == 0; }

static int do_layout(hcms_plan_t* p, int n, const void* const* src, void* const* dst, int c, bool gather,
                     cudaStream_t st) {
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
  cudaError_t e = (p->flags & HCMS_FLAG_LAYOUT_TMA) ? launch_layout_tma(a, st, p->num_sms) : launch_layout_vec(a, st);
  if (e != cudaSuccess) return fail_cuda(e, gather ? "a2a gather launch" : "a2a scatter launch");
  p->last_launches += 1;
  return HCMS_OK;
}

static int do_attention(hcms_plan_t* p, const void* qc, const void* kc, const void* vc, void* oc, int c, float scale,
                        cudaStream_t st, float* lse = nullptr) {
  const Chunk& ck = p->chunks[c];
  AttnArgs a{qc, kc, vc, oc, p->sh.S, p->sh.D, p->sh.P, ck.h, scale};
  a.lse = lse;
  a.pair = (p->flags & HCMS_FLAG_ATTN_PAIR) != 0;
  cudaError_t e = launch_attention(a, st);
  if (e != cudaSuccess) return fail_cuda(e, "attention launch");
  p->last_launches += 1;
  return HCMS_OK;
}

static int check_scale(float scale) {
  if (!std::isfinite(scale) || scale < 0.f) return fail(HCMS_ERR_INVALID_ARG, "scale=%g must be finite and >= 0", scale);
  return HCMS_OK;
}

extern "C" {

int hcms_a2a_scatter(hcms_plan_t* plan, int n_tensors, const void* const* src, void* const* dst, int c, void* stream) {
  if (!plan || !src || !dst) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (n_tensors < 1 || n_tensors > 3) return fail(HCMS_ERR_INVALID_ARG, "n_tensors=%d must be 1..3", n_tensors);
  if (c < 0 || c >= plan->sh.C) return fail(HCMS_ERR_PLAN_MISMATCH, "chunk %d outside [0,%d)", c, plan->sh.C);
  for (int t = 0; t < n_tensors; ++t) {
    if (!src[t] || !dst[t]) return fail(HCMS_ERR_INVALID_ARG, "tensor %d pointer is NULL", t);
    if (!aligned16(src[t]) || !aligned16(dst[t])) return fail(HCMS_ERR_MISALIGNED, "tensor %d is not 16-byte aligned", t);
  }
  plan->last_launches = 0;
  return do_layout(plan, n_tensors, src, dst, c, false, static_cast<cudaStream_t>(stream));
}

int hcms_a2a_gather(hcms_plan_t* plan, const void* src, void* dst, int c, void* stream) {
  if (!plan || !src || !dst) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (c < 0 || c >= plan->sh.C) return fail(HCMS_ERR_PLAN_MISMATCH, "chunk %d outside [0,%d)", c, plan->sh.C);
  if (!aligned16(src) || !aligned16(dst)) return fail(HCMS_ERR_MISALIGNED, "pointer is not 16-byte aligned");
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
  plan->last_launches = 0;
  return do_attention(plan, qc, kc, vc, oc, c, scale, static_cast<cudaStream_t>(stream));
}

// ------------------------------------------------------------------------------------------
// the dual-stream chunk scheduler (Algorithm 1 lines 4-25)
// ------------------------------------------------------------------------------------------
}  // extern "C"
static int enqueue_forward(hcms_plan_t* plan, const void* q, const void* k, const void* v, void* out, float scale,
                           cudaStream_t caller);
static int forward_graph(hcms_plan_t* plan, const void* q, const void* k, const void* v, void* out, float scale,
                         cudaStream_t caller);
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
  const char* ob = static_cast<const char*>(out);
  for (const void* in : {q, k, v}) {
    const char* ib = static_cast<const char*>(in);
    if (ob < ib + bytes && ib < ob + bytes) return fail(HCMS_ERR_ALIAS, "out overlaps an input tensor");
  }
  if (!plan->ws) return fail(HCMS_ERR_WORKSPACE_TOO_SMALL, "plan has no workspace");
  cudaStream_t caller = static_cast<cudaStream_t>(stream);
  if (plan->flags & HCMS_FLAG_GRAPH) return forward_graph(plan, q, k, v, out, scale, caller);
  return enqueue_forward(plan, q, k, v, out, scale, caller);
}

}  // extern "C"

// Enqueue Alg. 1 lines 4-25 for validated arguments: kernels, copies, event records and waits; no host synchronisation.
static int enqueue_forward(hcms_plan_t* plan, const void* q, const void* k, const void* v, void* out, float scale,
                           cudaStream_t caller) {
  const Shape& sh = plan->sh;
  int st = HCMS_OK;
  const bool serial = plan->flags & HCMS_FLAG_SERIAL;
  const bool split = (plan->flags & HCMS_FLAG_SPLIT_COMM) && !serial;
  cudaStream_t s_in = serial ? caller : plan->s_comm;
  cudaStream_t s_out = serial ? caller : (split ? plan->s_comm_out : plan->s_comm);
  // S_comp: two CUDA streams alternating by chunk parity (see HCMS_FLAG_SINGLE_COMP in hcms.h)
  const bool dual_comp = !serial && !(plan->flags & HCMS_FLAG_SINGLE_COMP) && sh.C > 1;
  auto comp_stream = [&](int c) { return serial ? caller : ((dual_comp && (c & 1)) ? plan->s_comp2 : plan->s_comp); };
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

  const bool profile = plan->flags & HCMS_FLAG_PROFILE;
  auto mark = [&](int step, int c, int side, cudaStream_t s) -> cudaError_t {
    const size_t slot = static_cast<size_t>(plan->prof_calls % HCMS_PROFILE_RING) * sh.C + c;
    return profile ? cudaEventRecord(plan->prof[step][side][slot], s) : cudaSuccess;
  };

  if (!serial) {
    HCMS_CUDA(cudaEventRecord(plan->e_main, caller));            // Alg. 1 line 5
    HCMS_CUDA(cudaStreamWaitEvent(s_in, plan->e_main, 0));       // line 7
    HCMS_CUDA(cudaStreamWaitEvent(plan->s_comp, plan->e_main, 0));     // line 13
    if (dual_comp) HCMS_CUDA(cudaStreamWaitEvent(plan->s_comp2, plan->e_main, 0));
    if (split) HCMS_CUDA(cudaStreamWaitEvent(s_out, plan->e_main, 0));
  }
  // Phase 1 -- input all-to-all of every chunk on S_comm (lines 8-11)
  for (int c = 0; c < sh.C; ++c) {
    const Chunk& ck = plan->chunks[c];
    const void* src[3] = {q, k, v};
    void* dst[3];
    for (int t = 0; t < 3; ++t) dst[t] = routed(t) ? plan->wire[t] : static_cast<void*>(ws + ck.off[t]);
    HCMS_CUDA(mark(0, c, 0, s_in));
    st = do_layout(plan, 3, src, dst, c, false, s_in);
    if (st) return st;
    for (int t = 0; t < 3; ++t) {
      if (!routed(t)) continue;
      st = host_hop(t, plan->wire[t], ws + ck.off[t], ck.bytes, s_in);
      if (st) return st;
    }
    HCMS_CUDA(mark(0, c, 1, s_in));
    if (!serial) HCMS_CUDA(cudaEventRecord(plan->e_comm[c], s_in));  // E_c^comm
  }
  // Phase 2 -- attention per chunk on S_comp (lines 14-18); Attn_c <- wait(E_c^comm)  (Eq. 6)
  for (int c = 0; c < sh.C; ++c) {
    const Chunk& ck = plan->chunks[c];
    cudaStream_t s_comp = comp_stream(c);
    if (!serial && !(plan->flags & HCMS_FLAG_DEBUG_NO_COMM_WAIT))
      HCMS_CUDA(cudaStreamWaitEvent(s_comp, plan->e_comm[c], 0));
    HCMS_CUDA(mark(1, c, 0, s_comp));
    float* lse_c = plan->lse ? plan->lse + static_cast<size_t>(sh.P) * sh.S * ck.o : nullptr;   // chunk c: [P*h_c][S]
    st = do_attention(plan, ws + ck.off[0], ws + ck.off[1], ws + ck.off[2], ws + ck.off[3], c, scale, s_comp, lse_c);
    if (st) return st;
    HCMS_CUDA(mark(1, c, 1, s_comp));
    if (!serial) HCMS_CUDA(cudaEventRecord(plan->e_comp[c], s_comp));  // E_c^comp
  }
  // Phase 3 -- output all-to-all per chunk on S_comm (lines 20-23); A_c^out <- wait(E_c^comp)  (Eq. 7)
  for (int c = 0; c < sh.C; ++c) {
    const Chunk& ck = plan->chunks[c];
    if (!serial) HCMS_CUDA(cudaStreamWaitEvent(s_out, plan->e_comp[c], 0));
    HCMS_CUDA(mark(2, c, 0, s_out));
    if (routed(3)) {
      st = host_hop(3, ws + ck.off[3], plan->wire[3], ck.bytes, s_out);
      if (st) return st;
    }
    const void* src[1] = {routed(3) ? plan->wire[3] : static_cast<const void*>(ws + ck.off[3])};
    void* dst[1] = {out};
    st = do_layout(plan, 1, src, dst, c, true, s_out);
    if (st) return st;
    HCMS_CUDA(mark(2, c, 1, s_out));
  }
  if (profile) plan->prof_calls += 1;
  plan->forward_done = true;
  if (!serial) {
    // line 25: Synchronize(S_comm, S_comp) -- expressed as stream waits, the host is not blocked
    HCMS_CUDA(cudaEventRecord(plan->e_fin_comm, s_out));
    HCMS_CUDA(cudaEventRecord(plan->e_fin_comp, plan->s_comp));
    HCMS_CUDA(cudaStreamWaitEvent(caller, plan->e_fin_comm, 0));
    HCMS_CUDA(cudaStreamWaitEvent(caller, plan->e_fin_comp, 0));
    if (dual_comp) {
      HCMS_CUDA(cudaEventRecord(plan->e_fin_comp2, plan->s_comp2));
      HCMS_CUDA(cudaStreamWaitEvent(caller, plan->e_fin_comp2, 0));
    }
    if (split) {
      HCMS_CUDA(cudaEventRecord(plan->e_fin_in, s_in));
      HCMS_CUDA(cudaStreamWaitEvent(caller, plan->e_fin_in, 0));
    }
  }
  return HCMS_OK;
}

// HCMS_FLAG_GRAPH: the whole chunk pipeline (kernels on S_comm / S_comp, the event forks and joins of Eq. 6-7) is
// captured once into a CUDA graph on a plan-owned stream and replayed with one launch per call; a call with other
// tensors or another scale captures again.  The capture runs on the plan's own stream because the caller's may be
// the legacy default stream, which cannot be captured.
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
  return HCMS_OK;
}

extern "C" {

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

int hcms_autotune_chunks(int64_t S, int H, int D, int P, int dtype, uint32_t flags, const void* q, const void* k,
                         const void* v, void* out, float scale, void* stream, int max_C, int reps, int* best_C,
                         float* ms_per_call) {
  if (!q || !k || !v || !out || !best_C) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (max_C < 1 || reps < 1) return fail(HCMS_ERR_INVALID_ARG, "max_C=%d and reps=%d must be >= 1", max_C, reps);
  if (P <= 0 || H <= 0 || H % P) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "H=%d is not divisible by P=%d", H, P);
  const int Hl = H / P;
  const int top = max_C < Hl ? max_C : Hl;
  cudaStream_t caller = static_cast<cudaStream_t>(stream);
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
    status = hcms_plan(&plan, S, H, D, P, C, dtype, flags & ~(HCMS_FLAG_SERIAL | HCMS_FLAG_PROFILE));
    if (status != HCMS_OK) break;
    status = hcms_attention_forward(plan, q, k, v, out, S, H, D, P, C, scale, stream);  // warm-up
    if (status == HCMS_OK) {
      ce = cudaEventRecord(e0, caller);
      for (int r = 0; r < reps && status == HCMS_OK && ce == cudaSuccess; ++r)
        status = hcms_attention_forward(plan, q, k, v, out, S, H, D, P, C, scale, stream);
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

int hcms_autotune_chunks_host(int64_t S, int H, int D, int P, uint32_t flags, const void* q, const void* k, const void* v,
                              void* out, float scale, void* stream, int max_C, int reps, int* best_C, float* ms_per_call) {
  if (!q || !k || !v || !out || !best_C) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (max_C < 1 || reps < 1) return fail(HCMS_ERR_INVALID_ARG, "max_C=%d and reps=%d must be >= 1", max_C, reps);
  if (P <= 0 || H <= 0 || H % P) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "H=%d is not divisible by P=%d", H, P);
  const int Hl = H / P;
  const int top = max_C < Hl ? max_C : Hl;
  cudaStream_t caller = static_cast<cudaStream_t>(stream);
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
    status = hcms_plan(&plan, S, H, D, P, C, HCMS_DTYPE_BF16, flags & ~(HCMS_FLAG_SERIAL | HCMS_FLAG_PROFILE | HCMS_FLAG_GRAPH));
    if (status != HCMS_OK) break;
    status = hcms_attention_forward_host(plan, q, k, v, out, S, H, D, P, C, scale, stream);   // warm-up
    if (status == HCMS_OK) {
      ce = cudaEventRecord(e0, caller);
      for (int r = 0; r < reps && status == HCMS_OK && ce == cudaSuccess; ++r)
        status = hcms_attention_forward_host(plan, q, k, v, out, S, H, D, P, C, scale, stream);
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

int hcms_attention_forward_host(hcms_plan_t* plan, const void* q, const void* k, const void* v, void* out, int64_t S,
                                int H, int D, int P, int C, float scale, void* stream) {
  if (!plan || !q || !k || !v || !out) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  const Shape& sh = plan->sh;
  if (S != sh.S || H != sh.H || D != sh.D || P != sh.P || C != sh.C)
    return fail(HCMS_ERR_PLAN_MISMATCH, "call shape differs from the plan's");
  const size_t bytes = static_cast<size_t>(S) * H * D * sh.es;
  cudaStream_t caller = static_cast<cudaStream_t>(stream);
  if (!(plan->flags & (HCMS_FLAG_HOST_STAGED | HCMS_FLAG_SERIAL | HCMS_FLAG_GRAPH)) && plan->dtype == HCMS_DTYPE_BF16) {
    // The host link is the wire: strided copies on the copy engines perform the all-to-all layout change themselves.
    // Chunk c of rank p's heads is a 2-D region of the host tensor (S rows of h_c*D elements, pitch H*D) and lands as
    // the dense [S][h_c][D] slab of Q'_c / K'_c / V'_c; the output all-to-all is the reverse copy from O'_c into
    // `out`.  H2D copies run on S_comm, D2H copies on the second communication stream (separate copy engines), the
    // attention of chunk c on S_comp between them, ordered by the same events as Alg. 1: no scatter / gather
    // kernels, no staging tensors, and the transfer of chunk c+1 overlaps the attention of chunk c.
    int st = check_scale(scale);
    if (st) return st;
    if (!plan->ws) return fail(HCMS_ERR_WORKSPACE_TOO_SMALL, "plan has no workspace");
    char* ws = static_cast<char*>(plan->ws);
    const size_t row = static_cast<size_t>(H) * D * sh.es;       // host pitch
    const bool dual_comp = !(plan->flags & HCMS_FLAG_SINGLE_COMP) && sh.C > 1;
    plan->last_launches = 0;
    HCMS_CUDA(cudaEventRecord(plan->e_main, caller));
    for (cudaStream_t s : {plan->s_comm, plan->s_comm_out, plan->s_comp, plan->s_comp2}) HCMS_CUDA(cudaStreamWaitEvent(s, plan->e_main, 0));
    const void* host_in[3] = {q, k, v};
    const bool profile = plan->flags & HCMS_FLAG_PROFILE;   // same event ring as the device path: 0 = H2D, 1 = attention, 2 = D2H
    auto mark = [&](int step, int c, int side, cudaStream_t s) -> cudaError_t {
      const size_t slot = static_cast<size_t>(plan->prof_calls % HCMS_PROFILE_RING) * sh.C + c;
      return profile ? cudaEventRecord(plan->prof[step][side][slot], s) : cudaSuccess;
    };
    for (int c = 0; c < sh.C; ++c) {
      const Chunk& ck = plan->chunks[c];
      const size_t width = static_cast<size_t>(ck.h) * D * sh.es, slab = width * S;
      HCMS_CUDA(mark(0, c, 0, plan->s_comm));
      for (int t = 0; t < 3; ++t)
        for (int p = 0; p < sh.P; ++p) {
          const char* src = static_cast<const char*>(host_in[t]) + (static_cast<size_t>(p) * sh.Hl + ck.o) * D * sh.es;
          HCMS_CUDA(cudaMemcpy2DAsync(ws + ck.off[t] + p * slab, width, src, row, width, S, cudaMemcpyHostToDevice, plan->s_comm));
          plan->last_launches += 1;
        }
      HCMS_CUDA(mark(0, c, 1, plan->s_comm));
      HCMS_CUDA(cudaEventRecord(plan->e_comm[c], plan->s_comm));
    }
    for (int c = 0; c < sh.C; ++c) {
      const Chunk& ck = plan->chunks[c];
      cudaStream_t s_comp = (dual_comp && (c & 1)) ? plan->s_comp2 : plan->s_comp;
      HCMS_CUDA(cudaStreamWaitEvent(s_comp, plan->e_comm[c], 0));
      float* lse_c = plan->lse ? plan->lse + static_cast<size_t>(sh.P) * sh.S * ck.o : nullptr;
      HCMS_CUDA(mark(1, c, 0, s_comp));
      st = do_attention(plan, ws + ck.off[0], ws + ck.off[1], ws + ck.off[2], ws + ck.off[3], c, scale, s_comp, lse_c);
      if (st) return st;
      HCMS_CUDA(mark(1, c, 1, s_comp));
      HCMS_CUDA(cudaEventRecord(plan->e_comp[c], s_comp));
    }
    for (int c = 0; c < sh.C; ++c) {
      const Chunk& ck = plan->chunks[c];
      const size_t width = static_cast<size_t>(ck.h) * D * sh.es, slab = width * S;
      HCMS_CUDA(cudaStreamWaitEvent(plan->s_comm_out, plan->e_comp[c], 0));
      HCMS_CUDA(mark(2, c, 0, plan->s_comm_out));
      for (int p = 0; p < sh.P; ++p) {
        char* dst = static_cast<char*>(out) + (static_cast<size_t>(p) * sh.Hl + ck.o) * D * sh.es;
        HCMS_CUDA(cudaMemcpy2DAsync(dst, row, ws + ck.off[3] + p * slab, width, width, S, cudaMemcpyDeviceToHost, plan->s_comm_out));
        plan->last_launches += 1;
      }
      HCMS_CUDA(mark(2, c, 1, plan->s_comm_out));
    }
    if (profile) plan->prof_calls += 1;
    HCMS_CUDA(cudaEventRecord(plan->e_fin_comm, plan->s_comm_out));
    HCMS_CUDA(cudaEventRecord(plan->e_fin_in, plan->s_comm));
    HCMS_CUDA(cudaEventRecord(plan->e_fin_comp, plan->s_comp));
    HCMS_CUDA(cudaEventRecord(plan->e_fin_comp2, plan->s_comp2));
    for (cudaEvent_t e : {plan->e_fin_comm, plan->e_fin_in, plan->e_fin_comp, plan->e_fin_comp2}) HCMS_CUDA(cudaStreamWaitEvent(caller, e, 0));
    plan->forward_done = true;
    HCMS_CUDA(cudaStreamSynchronize(caller));
    return HCMS_OK;
  }
  for (int t = 0; t < 4; ++t)
    if (!plan->staging[t]) HCMS_CUDA(cudaMalloc(&plan->staging[t], bytes));
  const void* host_in[3] = {q, k, v};
  for (int t = 0; t < 3; ++t)
    HCMS_CUDA(cudaMemcpyAsync(plan->staging[t], host_in[t], bytes, cudaMemcpyHostToDevice, caller));
  int st = hcms_attention_forward(plan, plan->staging[0], plan->staging[1], plan->staging[2], plan->staging[3], S, H, D,
                                  P, C, scale, stream);
  if (st) return st;
  HCMS_CUDA(cudaMemcpyAsync(out, plan->staging[3], bytes, cudaMemcpyDeviceToHost, caller));
  HCMS_CUDA(cudaStreamSynchronize(caller));
  return HCMS_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------
// the attention layer around the hot path (Alg. 1 lines 2-3 and 27)
// ------------------------------------------------------------------------------------------
static bool overlaps(const void* a, size_t na, const void* b, size_t nb) {
  const char* x = static_cast<const char*>(a);
  const char* y = static_cast<const char*>(b);
  return x < y + nb && y < x + na;
}

static int device_sms(int* sms) {
  static int cached = 0;
  if (cached == 0) {
    int dev = 0, n = 0;
    cudaError_t ce = cudaGetDeviceCount(&n);
    if (ce != cudaSuccess || n == 0) {
      cudaGetLastError();
      return fail(HCMS_ERR_UNSUPPORTED_DEVICE, "no CUDA device; libhcms has no CPU fallback");
    }
    HCMS_CUDA(cudaGetDevice(&dev));
    int major = 0, count = 0;
    HCMS_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    HCMS_CUDA(cudaDeviceGetAttribute(&count, cudaDevAttrMultiProcessorCount, dev));
    if (major != 10) return fail(HCMS_ERR_UNSUPPORTED_DEVICE, "device %d is sm_%dx; libhcms is built for sm_100a only", dev, major);
    cached = count;
  }
  *sms = cached;
  return HCMS_OK;
}

static int run_gemm(const GemmArgs& g, cudaStream_t st, const char* what) {
  cudaError_t e = launch_gemm(g, st);
  if (e != cudaSuccess) return fail_cuda(e, what);
  return HCMS_OK;
}

// hcms_layer_forward under HCMS_FLAG_FUSE_A2A: projection epilogue -> chunk buffers -> attention per chunk -> output
// projection reading the O'_c chunk buffers.  Attention launches alternate between the two compute streams as in
// hcms_attention_forward (tail-wave backfill); there is no communication stream because no copy is left.
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
  if (!plan->ws) return fail(HCMS_ERR_WORKSPACE_TOO_SMALL, "plan has no workspace");
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
  const bool serial = plan->flags & HCMS_FLAG_SERIAL;
  const bool dual_comp = !serial && !(plan->flags & HCMS_FLAG_SINGLE_COMP) && sh.C > 1;
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
    st = run_gemm(g, caller, "fused QKV projection launch");
    if (st) return st;
    plan->last_launches += 1;
  }
  if (profile) HCMS_CUDA(cudaEventRecord(plan->e_layer[1], caller));
  if (!serial) {
    HCMS_CUDA(cudaEventRecord(plan->e_main, caller));
    HCMS_CUDA(cudaStreamWaitEvent(plan->s_comp, plan->e_main, 0));
    if (dual_comp) HCMS_CUDA(cudaStreamWaitEvent(plan->s_comp2, plan->e_main, 0));
  }
  for (int c = 0; c < sh.C; ++c) {   // line 15 per chunk
    const Chunk& k = plan->chunks[c];
    cudaStream_t s_comp = serial ? caller : ((dual_comp && (c & 1)) ? plan->s_comp2 : plan->s_comp);
    float* lse_c = plan->lse ? plan->lse + static_cast<size_t>(sh.P) * sh.S * k.o : nullptr;
    st = do_attention(plan, ws + k.off[0], ws + k.off[1], ws + k.off[2], ws + k.off[3], c, scale, s_comp, lse_c);
    if (st) return st;
  }
  if (!serial) {
    HCMS_CUDA(cudaEventRecord(plan->e_fin_comp, plan->s_comp));
    HCMS_CUDA(cudaStreamWaitEvent(caller, plan->e_fin_comp, 0));
    if (dual_comp) {
      HCMS_CUDA(cudaEventRecord(plan->e_fin_comp2, plan->s_comp2));
      HCMS_CUDA(cudaStreamWaitEvent(caller, plan->e_fin_comp2, 0));
    }
  }
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
    st = run_gemm(g, caller, "fused output projection launch");
    if (st) return st;
    plan->last_launches += 1;
  }
  if (profile) {
    HCMS_CUDA(cudaEventRecord(plan->e_layer[3], caller));
    plan->layer_timed = true;
  }
  plan->forward_done = true;
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
  return run_gemm(g, static_cast<cudaStream_t>(stream), "QKV projection launch");
}

int hcms_output_projection(hcms_plan_t* plan, const void* o, const void* w_o, void* y, int Dm, void* stream) {
  if (!plan || !o || !w_o || !y) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  int st = check_layer_shape(plan, Dm);
  if (st) return st;
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

// ------------------------------------------------------------------------------------------
// backward of the hot path: the same chunk pipeline on the gradients
// ------------------------------------------------------------------------------------------
static int ensure_stats(hcms_plan_t* p) {
  if (!p->stats) HCMS_CUDA(cudaMalloc(&p->stats, attention_bwd_stats_bytes(p->sh.S, p->sh.H)));
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
  a.S = p->sh.S;
  a.D = p->sh.D;
  a.P = p->sh.P;
  a.h_c = p->chunks[c].h;
  a.scale = scale;
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
  if (!(plan->flags & HCMS_FLAG_TRAINING) || !plan->train_ws || !plan->lse)
    return fail(HCMS_ERR_INVALID_ARG, "the plan was made without HCMS_FLAG_TRAINING");
  if (!plan->forward_done) return fail(HCMS_ERR_INVALID_ARG, "no hcms_attention_forward has run on this plan");
  int st = check_scale(scale);
  if (st) return st;
  if (!aligned16(dout) || !aligned16(dq) || !aligned16(dk) || !aligned16(dv))
    return fail(HCMS_ERR_MISALIGNED, "dout, dq, dk and dv must be 16-byte aligned");
  const size_t bytes = static_cast<size_t>(S) * H * D * sh.es;
  const void* all[4] = {dout, dq, dk, dv};
  for (int i = 0; i < 4; ++i)
    for (int j = i + 1; j < 4; ++j)
      if (overlaps(all[i], bytes, all[j], bytes)) return fail(HCMS_ERR_ALIAS, "dout, dq, dk, dv must not overlap");
  if (!plan->ws) return fail(HCMS_ERR_WORKSPACE_TOO_SMALL, "plan has no workspace");
  st = ensure_stats(plan);
  if (st) return st;

  cudaStream_t caller = static_cast<cudaStream_t>(stream);
  const bool serial = plan->flags & HCMS_FLAG_SERIAL;
  cudaStream_t s_comm = serial ? caller : plan->s_comm;
  const bool dual_comp = !serial && !(plan->flags & HCMS_FLAG_SINGLE_COMP) && sh.C > 1;
  auto comp_stream = [&](int c) { return serial ? caller : ((dual_comp && (c & 1)) ? plan->s_comp2 : plan->s_comp); };
  char* ws = static_cast<char*>(plan->ws);          // Q'_c, K'_c, V'_c, O'_c saved by the forward
  char* gw = static_cast<char*>(plan->train_ws);    // dO'_c at off[3], dQ'_c, dK'_c, dV'_c at off[0..2]
  plan->last_launches = 0;
  if (!serial) {
    HCMS_CUDA(cudaEventRecord(plan->e_main, caller));
    HCMS_CUDA(cudaStreamWaitEvent(s_comm, plan->e_main, 0));
    HCMS_CUDA(cudaStreamWaitEvent(plan->s_comp, plan->e_main, 0));
    if (dual_comp) HCMS_CUDA(cudaStreamWaitEvent(plan->s_comp2, plan->e_main, 0));
  }
  // input all-to-all of the incoming gradient, every chunk, on S_comm
  for (int c = 0; c < sh.C; ++c) {
    const Chunk& ck = plan->chunks[c];
    const void* src[1] = {dout};
    void* dst[1] = {gw + ck.off[3]};
    st = do_layout(plan, 1, src, dst, c, false, s_comm);
    if (st) return st;
    if (!serial) HCMS_CUDA(cudaEventRecord(plan->e_comm[c], s_comm));
  }
  // attention backward per chunk on S_comp
  for (int c = 0; c < sh.C; ++c) {
    const Chunk& ck = plan->chunks[c];
    cudaStream_t s_comp = comp_stream(c);
    if (!serial) HCMS_CUDA(cudaStreamWaitEvent(s_comp, plan->e_comm[c], 0));
    const float* lse_c = plan->lse + static_cast<size_t>(sh.P) * sh.S * ck.o;
    st = do_attention_bwd(plan, ws + ck.off[0], ws + ck.off[1], ws + ck.off[2], ws + ck.off[3], gw + ck.off[3], lse_c,
                          gw + ck.off[0], gw + ck.off[1], gw + ck.off[2], c, scale, s_comp);
    if (st) return st;
    if (!serial) HCMS_CUDA(cudaEventRecord(plan->e_comp[c], s_comp));
  }
  // output all-to-all of dQ'_c, dK'_c, dV'_c (one launch for the three) on S_comm
  for (int c = 0; c < sh.C; ++c) {
    const Chunk& ck = plan->chunks[c];
    if (!serial) HCMS_CUDA(cudaStreamWaitEvent(s_comm, plan->e_comp[c], 0));
    const void* src[3] = {gw + ck.off[0], gw + ck.off[1], gw + ck.off[2]};
    void* dst[3] = {dq, dk, dv};
    st = do_layout(plan, 3, src, dst, c, true, s_comm);
    if (st) return st;
  }
  if (!serial) {
    HCMS_CUDA(cudaEventRecord(plan->e_fin_comm, s_comm));
    HCMS_CUDA(cudaEventRecord(plan->e_fin_comp, plan->s_comp));
    HCMS_CUDA(cudaStreamWaitEvent(caller, plan->e_fin_comm, 0));
    HCMS_CUDA(cudaStreamWaitEvent(caller, plan->e_fin_comp, 0));
    if (dual_comp) {
      HCMS_CUDA(cudaEventRecord(plan->e_fin_comp2, plan->s_comp2));
      HCMS_CUDA(cudaStreamWaitEvent(caller, plan->e_fin_comp2, 0));
    }
  }
  return HCMS_OK;
}

}  // extern "C"
