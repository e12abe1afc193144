// HCMS between P REAL ranks (Algorithm 1 lines 8 and 21, Table 1): one rank per
// process / GPU, each holding its sequence shard [S/P, H, D].  The all-to-alls are not library collectives: the
// scatter kernel of rank r STORES its [S/P, h_c, D] slices straight into every peer's chunk buffers Q'_c, K'_c, V'_c
// (push), and the gather kernel LOADS this rank's rows of every peer's O'_c (pull), through CUDA-IPC / peer mappings
// of the ranks' exchange blocks (NVLink 5 / NVSwitch on a real node; the same mapping works between processes that
// share one GPU, which is how the tests run it).  The per-chunk events E_c^comm / E_c^comp of Eq. 6-7 become
// device-side epoch flags in the consumer's memory: the producer's stream writes them after its kernel (a one-warp
// signal kernel with system-scope release stores), the consumer's stream waits on them with cuStreamWaitValue32 --
// no kernel ever spins on another rank, no host synchronisation, no NCCL on the data path.
//
//   S_comm of rank r : wait E_main; for c: push_c (q,k,v -> all peers), signal arrived[c][r] on all peers;
//                      then for c: wait ready[c][p] for all p, pull_c (all peers' O'_c -> out)
//   S_comp of rank r : wait E_main; for c: wait arrived[c][p] for all p, attention_c on the local heads,
//                      signal ready[c][r] on all peers
//
// Buffer reuse across calls needs no extra flags: rank r's push of call e+1 follows its pull of call e on S_comm, and
// that pull waited for every peer's attention_c of call e (ready), so the peers' Q'_c/K'_c/V'_c are free; rank r's
// attention_c of call e+1 overwrites O'_c only after arrived[c][p] = e+1 for all p, i.e. after every peer's S_comm
// has passed its pulls of call e.
#include <cstring>
#include <new>

#include "hcms_plan.h"

using namespace hcms;

namespace {

using WaitValueFn = CUresult (*)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
WaitValueFn g_wait_value = nullptr;

// cuStreamBatchMemOp: the P flag waits of one chunk as ONE stream operation (P = 8, C = 4: 8 operations per call on each
// stream instead of 64).  Optional: without it the waits are enqueued one by one.
using BatchMemOpFn = CUresult (*)(CUstream, unsigned int, CUstreamBatchMemOpParams*, unsigned int);
BatchMemOpFn g_batch_mem_op = nullptr;

int resolve_wait_value() {
  if (g_wait_value) return HCMS_OK;
  {
    void* bfn = nullptr;
    cudaDriverEntryPointQueryResult bres;
    if (cudaGetDriverEntryPoint("cuStreamBatchMemOp", &bfn, cudaEnableDefault, &bres) == cudaSuccess &&
        bres == cudaDriverEntryPointSuccess && bfn)
      g_batch_mem_op = reinterpret_cast<BatchMemOpFn>(bfn);
    else
      cudaGetLastError();
  }
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuStreamWaitValue32", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess) return fail_cuda(e, "cudaGetDriverEntryPoint(cuStreamWaitValue32)");
  if (qres != cudaDriverEntryPointSuccess || !fn) return fail(HCMS_ERR_UNSUPPORTED_DEVICE, "cuStreamWaitValue32 is not available");
  g_wait_value = reinterpret_cast<WaitValueFn>(fn);
  return HCMS_OK;
}

// One warp: lane p publishes `value` at flags[p] (an address in rank p's exchange block).  The kernels that produced
// the data ran earlier on the same stream; the system-scope fence + release store order their (peer) writes before
// the flag for an observer on another GPU or in another process.
struct SignalTargets {
  uint32_t* flag[kMaxPeers];
};
__global__ void hcms_dist_signal_kernel(const __grid_constant__ SignalTargets t, int n, uint32_t value) {
  const int p = threadIdx.x;
  if (p < n) {
    __threadfence_system();
    asm volatile("st.release.sys.global.u32 [%0], %1;" ::"l"(t.flag[p]), "r"(value) : "memory");
  }
}

struct ExportHandle {            // what hcms_dist_export writes (HCMS_DIST_HANDLE_BYTES)
  cudaIpcMemHandle_t mem;        // 64 bytes
  uint64_t bytes;
  uint64_t magic;
  int32_t rank, P, C, device;
  int64_t S;
  int32_t H, D;
  uint8_t pad[HCMS_DIST_HANDLE_BYTES - 64 - 8 - 8 - 16 - 8 - 8];
};
static_assert(sizeof(ExportHandle) == HCMS_DIST_HANDLE_BYTES, "handle layout");
constexpr uint64_t kMagic = 0x48434d5344495354ull;   // "HCMSDIST"

}  // namespace

struct hcms_dist_plan {
  Shape sh{};                    // global shape; sh.P = number of real ranks
  int rank = 0;
  uint32_t flags = 0;
  int device = 0;
  int64_t Sl = 0;                // tokens per rank
  std::vector<Chunk> chunks;     // bytes / off: this rank's buffers [S][h_c][D] inside the exchange block
  size_t out_off = 0;            // HCMS_FLAG_DIST_FUSE_OUT: this rank's output [Sl][H][D], written by every rank's attention epilogue
  size_t out_bytes = 0;
  size_t out_pad = 0;            // pad rows in front of it
  size_t flag_off = 0;           // arrived[C][P] then ready[C][P], uint32
  size_t block_bytes = 0;
  char* block = nullptr;         // this rank's exchange block (cudaMalloc, exported through CUDA IPC)
  std::vector<char*> peer;       // base of every rank's exchange block in THIS process' address space
  std::vector<bool> peer_ipc;    // opened with cudaIpcOpenMemHandle (to be closed)
  bool attached = false;
  bool local = false;            // attached with hcms_dist_attach_local: driven by the group call only
  bool poisoned = false;         // a forward call failed after its epoch was taken: this rank's flags no longer line up with the peers'
  uint32_t epoch = 0;
  cudaStream_t s_comm = nullptr, s_comp = nullptr;
  cudaEvent_t e_main = nullptr, e_fin[2] = {nullptr, nullptr};
  TmapCache tmaps;
  int last_launches = 0;
  int num_sms = 0;
  void* staging[4] = {nullptr, nullptr, nullptr, nullptr};   // hcms_dist_attention_forward_host: device copies of q, k, v, out shards
};

static void dist_free(hcms_dist_plan_t* p) {
  if (!p) return;
  if (p->s_comm) cudaStreamSynchronize(p->s_comm);
  if (p->s_comp) cudaStreamSynchronize(p->s_comp);
  for (size_t i = 0; i < p->peer.size(); ++i)
    if (p->peer_ipc[i] && p->peer[i]) cudaIpcCloseMemHandle(p->peer[i]);
  if (p->e_main) cudaEventDestroy(p->e_main);
  for (auto e : p->e_fin) if (e) cudaEventDestroy(e);
  if (p->s_comm) cudaStreamDestroy(p->s_comm);
  if (p->s_comp) cudaStreamDestroy(p->s_comp);
  if (p->block) cudaFree(p->block);
  for (void* b : p->staging) if (b) cudaFree(b);
  delete p;
}

static uint32_t* flag_ptr(const hcms_dist_plan_t* p, char* base, int which /*0 arrived, 1 ready*/, int c, int r) {
  return reinterpret_cast<uint32_t*>(base + p->flag_off) + (static_cast<size_t>(which) * p->sh.C + c) * p->sh.P + r;
}

extern "C" {

int hcms_dist_plan(hcms_dist_plan_t** out, int64_t S, int H, int D, int P, int C, int dtype, uint32_t flags, int rank) {
  if (!out) return fail(HCMS_ERR_INVALID_ARG, "plan output pointer is NULL");
  *out = nullptr;
  if (S <= 0 || H <= 0 || D <= 0 || P <= 0 || C <= 0)
    return fail(HCMS_ERR_INVALID_ARG, "S=%lld H=%d D=%d P=%d C=%d must all be positive", static_cast<long long>(S), H, D, P, C);
  if (rank < 0 || rank >= P) return fail(HCMS_ERR_INVALID_ARG, "rank=%d outside [0,%d)", rank, P);
  if (dtype != HCMS_DTYPE_BF16) return fail(HCMS_ERR_UNSUPPORTED_DTYPE, "the distributed path is bf16 only");
  if (flags & ~static_cast<uint32_t>(HCMS_FLAG_ATTN_PAIR | HCMS_FLAG_DIST_FUSE_OUT | HCMS_FLAG_DEBUG_DIST_FAIL))
    return fail(HCMS_ERR_INVALID_ARG, "hcms_dist_plan accepts HCMS_FLAG_ATTN_PAIR, HCMS_FLAG_DIST_FUSE_OUT and the test-only "
                "HCMS_FLAG_DEBUG_DIST_FAIL (flags=0x%x)", flags);
  if (S % P) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "S=%lld is not divisible by P=%d", static_cast<long long>(S), P);
  if (H % P) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "H=%d is not divisible by P=%d", H, P);
  if (D != 64 && D != 128) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "D=%d: only head dimensions 64 and 128 are built", D);
  if (P > kMaxPeers) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "P=%d exceeds the %d ranks the peer table holds", P, kMaxPeers);
  const int Hl = H / P;
  if (C > Hl) return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "C=%d exceeds heads per rank H/P=%d", C, Hl);
  int sms = 0, dev = 0;
  int st = device_sms(&sms);
  if (st) return st;
  if ((st = resolve_wait_value()) != HCMS_OK) return st;
  HCMS_CUDA(cudaGetDevice(&dev));

  hcms_dist_plan_t* p = new (std::nothrow) hcms_dist_plan_t();
  if (!p) return fail(HCMS_ERR_INVALID_ARG, "out of host memory");
  p->sh = Shape{S, H, D, P, C, 2, Hl};
  p->rank = rank;
  p->flags = flags;
  p->device = dev;
  p->num_sms = sms;
  p->Sl = S / P;
  p->chunks.resize(C);
  std::vector<int> o(C), h(C);
  hcms_chunk_table_host(Hl, C, o.data(), h.data());
  size_t off = 0;
  for (int c = 0; c < C; ++c) {
    Chunk& ck = p->chunks[c];
    ck.o = o[c];
    ck.h = h[c];
    ck.bytes = static_cast<size_t>(S) * h[c] * D * 2;            // this rank's heads only: [S][h_c][D]
    for (int t = 0; t < 4; ++t) {
      ck.off[t] = off;
      off += (ck.bytes + 1023) / 1024 * 1024;
    }
  }
  if (flags & HCMS_FLAG_DIST_FUSE_OUT) {
    p->out_pad = static_cast<size_t>(kAttnPushPadRows) * H * D * 2;      // spill rows of tiles that straddle two ranks
    p->out_off = off;
    p->out_bytes = static_cast<size_t>(S / P) * H * D * 2;
    off += (p->out_pad + p->out_bytes + 1023) / 1024 * 1024;
  }
  p->flag_off = off;
  p->block_bytes = off + (static_cast<size_t>(2) * C * P * sizeof(uint32_t) + 1023) / 1024 * 1024;
  auto bail = [&](int status) {
    dist_free(p);
    return status;
  };
#define DIST_CUDA(expr)                                             \
  do {                                                              \
    cudaError_t e__ = (expr);                                       \
    if (e__ != cudaSuccess) return bail(fail_cuda(e__, #expr));     \
  } while (0)
  DIST_CUDA(cudaMalloc(reinterpret_cast<void**>(&p->block), p->block_bytes));
  DIST_CUDA(cudaMemset(p->block + p->flag_off, 0, p->block_bytes - p->flag_off));   // epoch 0 everywhere
  DIST_CUDA(cudaDeviceSynchronize());
  int prio_lo = 0, prio_hi = 0;
  DIST_CUDA(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
  DIST_CUDA(cudaStreamCreateWithPriority(&p->s_comm, cudaStreamNonBlocking, prio_hi));
  DIST_CUDA(cudaStreamCreateWithPriority(&p->s_comp, cudaStreamNonBlocking, prio_lo));
  DIST_CUDA(cudaEventCreateWithFlags(&p->e_main, cudaEventDisableTiming));
  for (auto& e : p->e_fin) DIST_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
  DIST_CUDA(attention_init());
#undef DIST_CUDA
  p->peer.assign(P, nullptr);
  p->peer_ipc.assign(P, false);
  p->peer[rank] = p->block;
  *out = p;
  return HCMS_OK;
}

int hcms_dist_plan_destroy(hcms_dist_plan_t* plan) {
  dist_free(plan);
  return HCMS_OK;
}

size_t hcms_dist_block_bytes(const hcms_dist_plan_t* plan) { return plan ? plan->block_bytes : 0; }
int hcms_dist_last_launch_count(const hcms_dist_plan_t* plan) { return plan ? plan->last_launches : 0; }

int hcms_dist_export(hcms_dist_plan_t* plan, void* handle) {
  if (!plan || !handle) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  ExportHandle h;
  std::memset(&h, 0, sizeof(h));
  HCMS_CUDA(cudaIpcGetMemHandle(&h.mem, plan->block));
  h.bytes = plan->block_bytes;
  h.magic = kMagic;
  h.rank = plan->rank;
  h.P = plan->sh.P;
  h.C = plan->sh.C;
  h.device = plan->device;
  h.S = plan->sh.S;
  h.H = plan->sh.H;
  h.D = plan->sh.D;
  std::memcpy(handle, &h, sizeof(h));
  return HCMS_OK;
}

static int check_peer_shape(const hcms_dist_plan_t* plan, int r, int64_t S, int H, int D, int P, int C, int rank, uint64_t bytes) {
  const Shape& sh = plan->sh;
  if (rank != r || P != sh.P || C != sh.C || S != sh.S || H != sh.H || D != sh.D || bytes != plan->block_bytes)
    return fail(HCMS_ERR_PLAN_MISMATCH, "entry %d describes rank %d of (S=%lld,H=%d,D=%d,P=%d,C=%d), this plan is rank %d of "
                "(S=%lld,H=%d,D=%d,P=%d,C=%d)", r, rank, static_cast<long long>(S), H, D, P, C, plan->rank,
                static_cast<long long>(sh.S), sh.H, sh.D, sh.P, sh.C);
  return HCMS_OK;
}

int hcms_dist_attach(hcms_dist_plan_t* plan, const void* handles, int n) {
  if (!plan || !handles) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (n != plan->sh.P) return fail(HCMS_ERR_PLAN_MISMATCH, "%d handles for P=%d ranks", n, plan->sh.P);
  if (plan->attached) return fail(HCMS_ERR_INVALID_ARG, "the plan is attached already");
  int dev = -1;
  HCMS_CUDA(cudaGetDevice(&dev));
  if (dev != plan->device) return fail(HCMS_ERR_PLAN_MISMATCH, "the plan was made on device %d but device %d is current", plan->device, dev);
  const ExportHandle* hs = static_cast<const ExportHandle*>(handles);
  for (int r = 0; r < n; ++r) {
    ExportHandle h;
    std::memcpy(&h, hs + r, sizeof(h));
    if (h.magic != kMagic) return fail(HCMS_ERR_INVALID_ARG, "entry %d is not a handle written by hcms_dist_export", r);
    int st = check_peer_shape(plan, r, h.S, h.H, h.D, h.P, h.C, h.rank, h.bytes);
    if (st) return st;
  }
  for (int r = 0; r < n; ++r) {
    if (r == plan->rank) continue;
    ExportHandle h;
    std::memcpy(&h, hs + r, sizeof(h));
    void* base = nullptr;
    HCMS_CUDA(cudaIpcOpenMemHandle(&base, h.mem, cudaIpcMemLazyEnablePeerAccess));
    plan->peer[r] = static_cast<char*>(base);
    plan->peer_ipc[r] = true;
  }
  plan->attached = true;
  return HCMS_OK;
}

int hcms_dist_attach_local(hcms_dist_plan_t* plan, hcms_dist_plan_t* const* peers, int n) {
  if (!plan || !peers) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (n != plan->sh.P) return fail(HCMS_ERR_PLAN_MISMATCH, "%d peers for P=%d ranks", n, plan->sh.P);
  if (plan->attached) return fail(HCMS_ERR_INVALID_ARG, "the plan is attached already");
  for (int r = 0; r < n; ++r) {
    if (!peers[r]) return fail(HCMS_ERR_INVALID_ARG, "peer %d is NULL", r);
    const Shape& s = peers[r]->sh;
    int st = check_peer_shape(plan, r, s.S, s.H, s.D, s.P, s.C, peers[r]->rank, peers[r]->block_bytes);
    if (st) return st;
  }
  if (peers[plan->rank] != plan) return fail(HCMS_ERR_INVALID_ARG, "peers[%d] must be this plan", plan->rank);
  int dev = -1;
  HCMS_CUDA(cudaGetDevice(&dev));
  if (dev != plan->device) return fail(HCMS_ERR_PLAN_MISMATCH, "the plan was made on device %d but device %d is current", plan->device, dev);
  for (int r = 0; r < n; ++r) {
    if (peers[r]->device != plan->device) {       // same process, another GPU: plain peer access
      cudaError_t e = cudaDeviceEnablePeerAccess(peers[r]->device, 0);
      if (e == cudaErrorPeerAccessAlreadyEnabled) cudaGetLastError();
      else if (e != cudaSuccess) return fail_cuda(e, "cudaDeviceEnablePeerAccess");
    }
    plan->peer[r] = peers[r]->block;
  }
  plan->attached = true;
  plan->local = true;
  return HCMS_OK;
}

// (the forward entry points follow the phase helper below)
}  // extern "C"

namespace {

struct RankCall {           // one rank's arguments of a forward call
  hcms_dist_plan_t* plan;
  const void *q, *k, *v;
  void* out;
  cudaStream_t caller;
  uint32_t epoch;
  // hcms_dist_layer_forward: the input all-to-all is the QKV projection's epilogue, the output projection reads the
  // assembled output from the exchange block (q, k, v, out above are unused)
  const void *x = nullptr, *w_qkv = nullptr, *w_o = nullptr, *rope_cos = nullptr, *rope_sin = nullptr;
  void* y = nullptr;
  int Dm = 0;
};

// Everything that can be refused without touching a stream is refused HERE, before the caller takes the next epoch: a
// call that returns an error from these checks has enqueued nothing and leaves the rank in step with its peers.
// `group`: the call switches to each plan's device itself, so only the switch is tried; otherwise the plan's device
// must be current.
int check_plan_state(hcms_dist_plan_t* plan, bool group) {
  if (!plan->attached) return fail(HCMS_ERR_INVALID_ARG, "the plan has not been attached to its peers");
  if (plan->poisoned)
    return fail(HCMS_ERR_INVALID_ARG, "an earlier forward call on this plan failed after part of its work had been enqueued; its epoch "
                "flags no longer agree with the peers': destroy the plans of all ranks and make new ones");
  if (group) {
    HCMS_CUDA(cudaSetDevice(plan->device));
    return HCMS_OK;
  }
  int dev = -1;
  HCMS_CUDA(cudaGetDevice(&dev));
  if (dev != plan->device)
    return fail(HCMS_ERR_PLAN_MISMATCH, "the plan was made on device %d but device %d is current", plan->device, dev);
  return HCMS_OK;
}

int check_call(const RankCall& rc, float scale, bool group) {
  hcms_dist_plan_t* plan = rc.plan;
  if (!plan || !rc.q || !rc.k || !rc.v || !rc.out) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (int ps = check_plan_state(plan, group)) return ps;
  int st = check_scale(scale);
  if (st) return st;
  if (!aligned16(rc.q) || !aligned16(rc.k) || !aligned16(rc.v) || !aligned16(rc.out))
    return fail(HCMS_ERR_MISALIGNED, "q, k, v and out must be 16-byte aligned");
  const Shape& sh = plan->sh;
  const size_t bytes = static_cast<size_t>(plan->Sl) * sh.H * sh.D * sh.es;
  for (const void* in : {rc.q, rc.k, rc.v})
    if (overlaps(rc.out, bytes, in, bytes)) return fail(HCMS_ERR_ALIAS, "out overlaps an input tensor");
  return HCMS_OK;
}

// phase 0 = fork + pushes (Alg. 1 lines 5-11), 1 = attention (lines 13-18), 2 = pulls + join (lines 19-25),
// 3 = the join alone (line 25): what a failed call still runs, so that the caller's stream is never left waiting on a
// flag that nobody will publish any more
int enqueue_phase(const RankCall& rc, int phase, float scale) {
  hcms_dist_plan_t* plan = rc.plan;
  const Shape& sh = plan->sh;
  const int P = sh.P, C = sh.C, r = plan->rank;
  const uint32_t epoch = rc.epoch;
  int status = HCMS_OK;
  auto cuda = [&](cudaError_t e, const char* what) {
    if (e != cudaSuccess && status == HCMS_OK) status = fail_cuda(e, what);
    return status == HCMS_OK;
  };
  int dev = -1;
  if (!cuda(cudaGetDevice(&dev), "cudaGetDevice")) return status;
  if (dev != plan->device) return fail(HCMS_ERR_PLAN_MISMATCH, "the plan was made on device %d but device %d is current", plan->device, dev);
  auto signal = [&](int which, int c, cudaStream_t s) {          // publish flag[which][c][r] = epoch on every rank
    SignalTargets t{};
    for (int p = 0; p < P; ++p) t.flag[p] = flag_ptr(plan, plan->peer[p], which, c, r);
    hcms_dist_signal_kernel<<<1, 32, 0, s>>>(t, P, epoch);
    plan->last_launches += 1;
    return cuda(cudaGetLastError(), "signal launch");
  };
  auto wait_all = [&](int which, int c, cudaStream_t s) {        // until flag[which][c][p] >= epoch for every p (local memory)
    if (g_batch_mem_op && P > 1) {
      CUstreamBatchMemOpParams ops[kMaxPeers];
      std::memset(ops, 0, sizeof(ops));
      for (int p = 0; p < P; ++p) {
        ops[p].waitValue.operation = CU_STREAM_MEM_OP_WAIT_VALUE_32;
        ops[p].waitValue.address = reinterpret_cast<CUdeviceptr>(flag_ptr(plan, plan->block, which, c, p));
        ops[p].waitValue.value = epoch;
        ops[p].waitValue.flags = CU_STREAM_WAIT_VALUE_GEQ;
      }
      const CUresult cr = g_batch_mem_op(reinterpret_cast<CUstream>(s), static_cast<unsigned>(P), ops, 0);
      if (cr != CUDA_SUCCESS) status = fail(HCMS_ERR_CUDA, "cuStreamBatchMemOp failed with CUresult %d", static_cast<int>(cr));
      return status == HCMS_OK;
    }
    for (int p = 0; p < P && status == HCMS_OK; ++p) {
      const CUresult cr = g_wait_value(reinterpret_cast<CUstream>(s),
                                       reinterpret_cast<CUdeviceptr>(flag_ptr(plan, plan->block, which, c, p)), epoch,
                                       CU_STREAM_WAIT_VALUE_GEQ);
      if (cr != CUDA_SUCCESS) status = fail(HCMS_ERR_CUDA, "cuStreamWaitValue32 failed with CUresult %d", static_cast<int>(cr));
    }
    return status == HCMS_OK;
  };
  auto layout = [&](int c, bool gather, int n, const void* const* local, cudaStream_t s) {
    const Chunk& ck = plan->chunks[c];
    LayoutArgs a{};
    std::vector<void*> tab[3];
    for (int t = 0; t < n; ++t) {
      // dense side: rows [r*Sl, (r+1)*Sl) of rank p's buffer (push: tensor t of Q'_c,K'_c,V'_c; pull: O'_c)
      tab[t].resize(P);
      for (int p = 0; p < P; ++p)
        tab[t][p] = plan->peer[p] + ck.off[gather ? 3 : t] + static_cast<size_t>(r) * plan->Sl * ck.h * sh.D * sh.es;
      a.peer[t] = tab[t].data();
      if (gather) a.dst[t] = const_cast<void*>(local[t]); else a.src[t] = local[t];
    }
    a.n_tensors = n;
    a.S = plan->Sl;
    a.H = sh.H;
    a.D = sh.D;
    a.P = P;
    a.Hl = sh.Hl;
    a.es = sh.es;
    a.o_c = ck.o;
    a.h_c = ck.h;
    a.gather = gather;
    plan->last_launches += 1;
    return cuda(launch_layout_vec(a, s), gather ? "pull gather launch" : "push scatter launch");
  };

  if (phase == 0) {
    plan->last_launches = 0;
    if (!cuda(cudaEventRecord(plan->e_main, rc.caller), "record E_main")) return status;       // Alg. 1 line 5
    cuda(cudaStreamWaitEvent(plan->s_comm, plan->e_main, 0), "wait E_main");
    cuda(cudaStreamWaitEvent(plan->s_comp, plan->e_main, 0), "wait E_main");
    // lines 8-11: input all-to-all of every chunk = stores into the peers' chunk buffers, then E_c^comm as a flag
    if (rc.x) {
      // Alg. 1 lines 2-3 and 8 in ONE kernel: the projection GEMM's epilogue (RoPE, bf16) TMA-stores every 128 x 64 panel
      // of q, k, v into the chunk buffer of the rank that owns its head -- peer memory; then E_c^comm for every chunk
      std::vector<void*> peers(static_cast<size_t>(3) * C * P);
      GemmChunks ck{};
      ck.C = C;
      ck.Hl = sh.Hl;
      ck.P = P;
      for (int c = 0; c < C; ++c) {
        ck.o[c] = plan->chunks[c].o;
        ck.h[c] = plan->chunks[c].h;
        for (int t = 0; t < 3; ++t)
          for (int p = 0; p < P; ++p)
            peers[(static_cast<size_t>(t) * C + c) * P + p] =
                plan->peer[p] + plan->chunks[c].off[t] + static_cast<size_t>(r) * plan->Sl * ck.h[c] * sh.D * sh.es;
      }
      ck.peer = peers.data();
      GemmArgs g{};
      g.a = rc.x;
      g.b = rc.w_qkv;
      g.M = plan->Sl;
      g.N = 3 * sh.H * sh.D;
      g.K = rc.Dm;
      g.n_per_out = sh.H * sh.D;
      g.rope_outs = rc.rope_cos ? 2 : 0;
      g.D = sh.D;
      g.cos = static_cast<const float*>(rc.rope_cos);
      g.sin = static_cast<const float*>(rc.rope_sin);
      g.num_sms = plan->num_sms;
      g.fuse = 1;
      g.chunks = &ck;
      g.cache = &plan->tmaps;
      plan->last_launches += 1;
      if (cuda(launch_gemm(g, plan->s_comm), "QKV projection with the fused push"))
        for (int c = 0; c < C && status == HCMS_OK; ++c) signal(0, c, plan->s_comm);
    } else {
      for (int c = 0; c < C && status == HCMS_OK; ++c) {
        const void* src[3] = {rc.q, rc.k, rc.v};
        if (layout(c, false, 3, src, plan->s_comm)) signal(0, c, plan->s_comm);
      }
    }
  } else if (phase == 1) {
    // lines 14-18: attention of this rank's heads of chunk c once every rank's slice has arrived (Eq. 6)
    for (int c = 0; c < C && status == HCMS_OK; ++c) {
      const Chunk& ck = plan->chunks[c];
      if (!wait_all(0, c, plan->s_comp)) break;
      if (plan->flags & HCMS_FLAG_DEBUG_DIST_FAIL)      // TEST ONLY: a launch failure after the pushes and the first wait
        return fail(HCMS_ERR_CUDA, "injected failure (HCMS_FLAG_DEBUG_DIST_FAIL) before the attention launch of chunk %d", c);
      AttnArgs a{plan->block + ck.off[0], plan->block + ck.off[1], plan->block + ck.off[2], plan->block + ck.off[3],
                 sh.S, sh.D, 1, ck.h, scale};
      a.pair = (plan->flags & HCMS_FLAG_ATTN_PAIR) != 0;
      a.cache = &plan->tmaps;
      void* push[kMaxPeers];
      if (plan->out_bytes) {          // output all-to-all in the attention epilogue: TMA stores into every rank's output
        for (int p = 0; p < P; ++p) push[p] = plan->peer[p] + plan->out_off;
        a.o_push = push;
        a.n_push = P;
        a.push_rows = plan->Sl;
        a.push_heads = sh.H;
        a.push_head0 = r * sh.Hl + ck.o;
      }
      plan->last_launches += 1;
      if (cuda(launch_attention(a, plan->s_comp), "attention launch")) signal(1, c, plan->s_comp);   // E_c^comp as a flag
    }
  } else if (phase == 2) {
    // lines 20-23, 26: output all-to-all = loads of this rank's rows from every peer's O'_c (Eq. 7), written into `out`
    for (int c = 0; c < C && status == HCMS_OK; ++c) {
      if (!wait_all(1, c, plan->s_comm)) break;
      if (plan->out_bytes) continue;        // fused: the peers' attention kernels have already delivered chunk c's heads
      const void* dst[1] = {rc.out};
      layout(c, true, 1, dst, plan->s_comm);
    }
    if (plan->out_bytes && status == HCMS_OK && !rc.x)   // Concat (line 26): the assembled output leaves the exchange block
      cuda(cudaMemcpyAsync(rc.out, plan->block + plan->out_off + plan->out_pad, plan->out_bytes, cudaMemcpyDeviceToDevice, plan->s_comm),
           "copy of the assembled output");
    if (rc.x && status == HCMS_OK) {                     // line 27: y = o W_o^T on the assembled [Sl, H*D] output, in place
      GemmArgs g{};
      g.a = plan->block + plan->out_off + plan->out_pad;
      g.b = rc.w_o;
      g.out[0] = rc.y;
      g.M = plan->Sl;
      g.N = rc.Dm;
      g.K = sh.H * sh.D;
      g.n_per_out = rc.Dm;
      g.D = sh.D;
      g.num_sms = plan->num_sms;
      g.cache = &plan->tmaps;
      plan->last_launches += 1;
      cuda(launch_gemm(g, plan->s_comm), "output projection");
    }
  }
  if (phase >= 2) {
    // line 25, on every path
    cudaStream_t forked[2] = {plan->s_comm, plan->s_comp};
    const int keep = status;
    for (int i = 0; i < 2; ++i) {
      cudaError_t e = cudaEventRecord(plan->e_fin[i], forked[i]);
      if (e == cudaSuccess) e = cudaStreamWaitEvent(rc.caller, plan->e_fin[i], 0);
      if (e != cudaSuccess && status == HCMS_OK) status = fail_cuda(e, "join");
    }
    if (keep != HCMS_OK) status = keep;
  }
  return status;
}

struct DeviceRestore {       // group calls switch devices; put the caller's back on every return path
  int dev;
  ~DeviceRestore() {
    if (dev >= 0) cudaSetDevice(dev);
  }
};

// The forward of n validated ranks (n = 1: one process per rank; n = P: the group call).  The epochs are taken HERE, after
// every check that can refuse the call.  Phase by phase over ALL ranks: every flag a stream waits on is produced by work
// already enqueued, so no stream ever blocks a hardware queue ahead of its producer.  On the first failure nothing more of
// the data path is enqueued -- in particular none of phase 2's waits on ready[c][p], whose producers (the attention
// kernels) may never have been launched -- every rank only joins its side streams back into its caller's stream, and the
// plans are poisoned: their epochs were consumed, so a later call could not line up with the peers' flags.
int run_ranks(RankCall* rc, int n, float scale, bool group) {
  for (int r = 0; r < n; ++r) rc[r].epoch = ++rc[r].plan->epoch;
  int st = HCMS_OK;
  for (int phase = 0; phase < 3 && st == HCMS_OK; ++phase)
    for (int r = 0; r < n && st == HCMS_OK; ++r) {
      if (group) cudaSetDevice(rc[r].plan->device);
      st = enqueue_phase(rc[r], phase, scale);
    }
  if (st != HCMS_OK) {
    const std::string text = hcms_last_error();     // the join below must not replace the first failure's text
    for (int r = 0; r < n; ++r) {
      rc[r].plan->poisoned = true;
      if (group) cudaSetDevice(rc[r].plan->device);
      enqueue_phase(rc[r], 3, scale);
    }
    fail(st, "%s", text.c_str());
  }
  return st;
}

}  // namespace

extern "C" {

int hcms_dist_attention_forward(hcms_dist_plan_t* plan, const void* q, const void* k, const void* v, void* out, float scale,
                                void* stream) {
  RankCall rc{plan, q, k, v, out, static_cast<cudaStream_t>(stream), 0};
  int st = check_call(rc, scale, false);
  if (st) return st;
  if (plan->local)
    return fail(HCMS_ERR_INVALID_ARG, "ranks attached with hcms_dist_attach_local are driven by hcms_dist_attention_forward_group "
                "(a rank-by-rank enqueue from one process can deadlock on shared hardware queues)");
  return run_ranks(&rc, 1, scale, false);
}

int hcms_dist_attention_forward_host(hcms_dist_plan_t* plan, const void* q, const void* k, const void* v, void* out, float scale,
                                     void* stream) {
  if (!plan || !q || !k || !v || !out) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  const Shape& sh = plan->sh;
  const size_t bytes = static_cast<size_t>(plan->Sl) * sh.H * sh.D * sh.es;
  for (const void* in : {q, k, v})
    if (overlaps(out, bytes, in, bytes)) return fail(HCMS_ERR_ALIAS, "out overlaps an input tensor");
  if (int ps = check_plan_state(plan, false)) return ps;      // before the staging is touched: attached, healthy, right device
  for (void*& b : plan->staging)
    if (!b) HCMS_CUDA(cudaMalloc(&b, bytes));
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const void* host_in[3] = {q, k, v};
  for (int t = 0; t < 3; ++t) HCMS_CUDA(cudaMemcpyAsync(plan->staging[t], host_in[t], bytes, cudaMemcpyHostToDevice, st));
  const int status = hcms_dist_attention_forward(plan, plan->staging[0], plan->staging[1], plan->staging[2], plan->staging[3], scale, stream);
  if (status != HCMS_OK) return status;                       // the failed call has joined its streams; nothing to copy back
  HCMS_CUDA(cudaMemcpyAsync(out, plan->staging[3], bytes, cudaMemcpyDeviceToHost, st));
  HCMS_CUDA(cudaStreamSynchronize(st));
  return HCMS_OK;
}

int hcms_dist_attention_forward_group(hcms_dist_plan_t* const* plans, int n, const void* const* q, const void* const* k,
                                      const void* const* v, void* const* out, float scale, void* const* streams) {
  if (!plans || !q || !k || !v || !out || !streams) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (n < 1 || n > kMaxPeers) return fail(HCMS_ERR_INVALID_ARG, "n=%d outside [1,%d]", n, kMaxPeers);
  RankCall rc[kMaxPeers];
  int prev = -1;
  cudaGetDevice(&prev);
  DeviceRestore restore{prev};     // the checks and the phases switch to each plan's device
  for (int r = 0; r < n; ++r) {
    rc[r] = RankCall{plans[r], q[r], k[r], v[r], out[r], static_cast<cudaStream_t>(streams[r]), 0};
    int st = check_call(rc[r], scale, true);
    if (st) return st;
    if (plans[r]->sh.P != n || plans[r]->rank != r)
      return fail(HCMS_ERR_PLAN_MISMATCH, "plans[%d] is rank %d of %d: pass all P plans in rank order", r, plans[r]->rank, plans[r]->sh.P);
    for (int o = 0; o < r; ++o)
      if (rc[o].caller == rc[r].caller) return fail(HCMS_ERR_INVALID_ARG, "ranks %d and %d share a caller stream", o, r);
  }
  return run_ranks(rc, n, scale, true);
}

// ---- the whole layer between real ranks: both all-to-alls inside compute kernels -------------------------------
static int check_layer_call(const RankCall& rc, float scale, bool group) {
  hcms_dist_plan_t* plan = rc.plan;
  if (!plan || !rc.x || !rc.w_qkv || !rc.w_o || !rc.y) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (int ps = check_plan_state(plan, group)) return ps;
  if (!plan->out_bytes) return fail(HCMS_ERR_INVALID_ARG, "hcms_dist_layer_forward needs a plan made with HCMS_FLAG_DIST_FUSE_OUT");
  if ((rc.rope_cos == nullptr) != (rc.rope_sin == nullptr)) return fail(HCMS_ERR_INVALID_ARG, "pass both RoPE tables or neither");
  int st = check_scale(scale);
  if (st) return st;
  const Shape& sh = plan->sh;
  if (rc.Dm <= 0 || rc.Dm % 128 || (sh.H * sh.D) % 128)
    return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "Dm=%d and H*D=%d must be multiples of 128", rc.Dm, sh.H * sh.D);
  if (3 * sh.C * sh.P > 96 || sh.Hl > 64)
    return fail(HCMS_ERR_UNSUPPORTED_SHAPE, "the fused push holds 96 tensor maps: 3*C*P = %d (C=%d, P=%d); H/P=%d must be <= 64",
                3 * sh.C * sh.P, sh.C, sh.P, sh.Hl);
  for (const void* ptr : {rc.x, rc.w_qkv, rc.w_o, rc.rope_cos, rc.rope_sin, static_cast<const void*>(rc.y)})
    if (!aligned16(ptr)) return fail(HCMS_ERR_MISALIGNED, "every pointer must be 16-byte aligned");
  return HCMS_OK;
}

int hcms_dist_layer_forward(hcms_dist_plan_t* plan, const void* x, const void* w_qkv, const void* w_o, const void* rope_cos,
                            const void* rope_sin, void* y, int Dm, float scale, void* stream) {
  RankCall rc{plan, nullptr, nullptr, nullptr, nullptr, static_cast<cudaStream_t>(stream), 0};
  rc.x = x; rc.w_qkv = w_qkv; rc.w_o = w_o; rc.rope_cos = rope_cos; rc.rope_sin = rope_sin; rc.y = y; rc.Dm = Dm;
  int st = check_layer_call(rc, scale, false);
  if (st) return st;
  if (plan->local)
    return fail(HCMS_ERR_INVALID_ARG, "ranks attached with hcms_dist_attach_local are driven by hcms_dist_layer_forward_group");
  return run_ranks(&rc, 1, scale, false);
}

int hcms_dist_layer_forward_group(hcms_dist_plan_t* const* plans, int n, const void* const* x, const void* w_qkv, const void* w_o,
                                  const void* const* rope_cos, const void* const* rope_sin, void* const* y, int Dm, float scale,
                                  void* const* streams) {
  if (!plans || !x || !y || !streams) return fail(HCMS_ERR_INVALID_ARG, "NULL argument");
  if (n < 1 || n > kMaxPeers) return fail(HCMS_ERR_INVALID_ARG, "n=%d outside [1,%d]", n, kMaxPeers);
  RankCall rc[kMaxPeers];
  int prev = -1;
  cudaGetDevice(&prev);
  DeviceRestore restore{prev};
  for (int r = 0; r < n; ++r) {
    rc[r] = RankCall{plans[r], nullptr, nullptr, nullptr, nullptr, static_cast<cudaStream_t>(streams[r]), 0};
    rc[r].x = x[r]; rc[r].w_qkv = w_qkv; rc[r].w_o = w_o; rc[r].y = y[r]; rc[r].Dm = Dm;
    rc[r].rope_cos = rope_cos ? rope_cos[r] : nullptr;
    rc[r].rope_sin = rope_sin ? rope_sin[r] : nullptr;
    int st = check_layer_call(rc[r], scale, true);
    if (st) return st;
    if (plans[r]->sh.P != n || plans[r]->rank != r)
      return fail(HCMS_ERR_PLAN_MISMATCH, "plans[%d] is rank %d of %d: pass all P plans in rank order", r, plans[r]->rank, plans[r]->sh.P);
    for (int o = 0; o < r; ++o)
      if (rc[o].caller == rc[r].caller) return fail(HCMS_ERR_INVALID_ARG, "ranks %d and %d share a caller stream", o, r);
  }
  return run_ranks(rc, n, scale, true);
}

}  // extern "C"
