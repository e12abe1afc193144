// The plan object and the ONE fork/join chunk schedule every entry point of libhcms uses
// (section 3.4-3.6, Algorithm 1).  Internal; not installed.
#pragma once

#include <functional>

#include "hcms_internal.h"

struct hcms_plan {
  hcms::Shape sh{};
  int dtype = 0;
  uint32_t flags = 0;
  int device = 0;
  int num_sms = 0;
  std::vector<hcms::Chunk> chunks;
  size_t ws_bytes = 0;
  void* ws = nullptr;          // chunk workspace; plan-owned memory is allocated on first use
  bool ws_owned = false;
  int ring = 0;               // HCMS_FLAG_RECYCLE_WS: number of chunk buffer sets (0 = one per chunk)
  cudaStream_t s_comm = nullptr, s_comm_out = nullptr, s_comp = nullptr, s_comp2 = nullptr;
  cudaEvent_t e_main = nullptr, e_fin[4] = {nullptr, nullptr, nullptr, nullptr};
  std::vector<cudaEvent_t> e_comm, e_comp;
  hcms::TmapCache tmaps;       // every TMA descriptor this plan has encoded ("device-level caching", L221)
  // host route (config 5): per routed tensor one pinned host buffer and one device "send/receive" buffer,
  // each as large as the largest chunk tensor
  void* pinned[4] = {nullptr, nullptr, nullptr, nullptr};
  void* wire[4] = {nullptr, nullptr, nullptr, nullptr};
  // host-buffer entry point staging (HCMS_FLAG_HOST_STAGED)
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
  float* dq_acc = nullptr;    // HCMS_FLAG_BWD_ONE_PASS: fp32 dQ accumulator of the largest chunk, and its turn counters
  int* dq_turn = nullptr;
  bool forward_done = false;
  float forward_scale = 0.f;  // the scale the saved lse belongs to
  // HCMS_FLAG_GRAPH: the captured chunk pipeline of the last (q, k, v, out, scale) and the stream it was captured on
  cudaStream_t s_cap = nullptr;
  cudaGraphExec_t graph_exec = nullptr;
  const void* graph_key[4] = {nullptr, nullptr, nullptr, nullptr};
  float graph_scale = 0.f;
  int graph_launches = 0;
  long long graph_captures = 0;
  // HCMS_FLAG_PROFILE: [step 0=scatter,1=attention,2=gather][begin,end][ring slot * C + chunk]
  std::vector<cudaEvent_t> prof[3][2];
  long long prof_calls = 0;   // pipeline runs that recorded a full set of events
};

namespace hcms {

void plan_free(hcms_plan_t* p);
int check_scale(float scale);
int check_plan_device(const hcms_plan_t* p);          // the plan's device must be current
int ensure_workspace(hcms_plan_t* p);                 // allocates the plan-owned workspace on first use
int ensure_training(hcms_plan_t* p);                  // gradient workspace + lse (HCMS_FLAG_TRAINING plans)
inline bool aligned16(const void* p) { return reinterpret_cast<uintptr_t>(p) % 16 == 0; }
inline bool overlaps(const void* a, size_t na, const void* b, size_t nb) {
  const char* x = static_cast<const char*>(a);
  const char* y = static_cast<const char*>(b);
  return x < y + nb && y < x + na;
}

int do_layout(hcms_plan_t* p, int n, const void* const* src, void* const* dst, int c, bool gather, cudaStream_t st);
int do_attention(hcms_plan_t* p, const void* qc, const void* kc, const void* vc, void* oc, int c, float scale,
                 cudaStream_t st, float* lse = nullptr);

// The three per-chunk steps of Alg. 1; each enqueues chunk c's work on the stream it is given and returns an HCMS
// status.  An empty std::function means the step does not exist for this entry point (e.g. the fused layer has no
// all-to-all kernels).
struct PipelineSteps {
  std::function<int(int c, cudaStream_t s)> comm_in;    // line 8   A_c^in   (S_comm)
  std::function<int(int c, cudaStream_t s)> compute;    // line 15  Attn_c   (S_comp), after wait(E_c^comm)  (Eq. 6)
  std::function<int(int c, cudaStream_t s)> comm_out;   // line 21  A_c^out  (S_comm), after wait(E_c^comp)  (Eq. 7)
  bool split_out = false;    // output all-to-all on the second communication stream (Eq. 8; HCMS_FLAG_SPLIT_COMM)
  bool profile = false;      // record the HCMS_FLAG_PROFILE event ring around every step
  int ring = 0;              // > 0: chunk c shares its buffers with chunk c - ring (HCMS_FLAG_RECYCLE_WS): A_c^in follows A_{c-ring}^out
};

// Algorithm 1 lines 5-25: record E_main on `caller`, fork S_comm / S_comp (/ their second streams), enqueue the three
// phases with E_c^comm and E_c^comp, and make `caller` wait for every forked stream (line 25) -- on every path, also
// when a step fails (the side streams are never left forked).  HCMS_FLAG_SERIAL: the three phases back to back on
// `caller` (Eq. 1).  No host synchronisation.  Returns the first failing status.
int run_pipeline(hcms_plan_t* plan, cudaStream_t caller, const PipelineSteps& steps);

}  // namespace hcms
