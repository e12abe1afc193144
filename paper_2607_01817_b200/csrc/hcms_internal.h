// Internal declarations shared by the translation units of libhcms (not installed).
#pragma once

#include <cuda.h>  // CUtensorMap and enums only; libcuda is reached through cudaGetDriverEntryPoint
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <string>
#include <unordered_map>
#include <vector>

#include "hcms.h"

namespace hcms {

// ---- error plumbing ---------------------------------------------------------------------
int fail(int status, const char* fmt, ...);  // records thread-local text, returns status
int fail_cuda(cudaError_t e, const char* what);

#define HCMS_CUDA(expr)                                        \
  do {                                                         \
    cudaError_t e__ = (expr);                                  \
    if (e__ != cudaSuccess) return ::hcms::fail_cuda(e__, #expr); \
  } while (0)

// ---- chunk geometry (Eq. 3 L83-84 on Hl = H/P; Table 8) ------------------------
struct Chunk {
  int o;             // first local head
  int h;             // number of local heads
  size_t bytes;      // P*S*h*D*es
  size_t off[4];     // workspace byte offsets of Q'_c, K'_c, V'_c, O'_c
};

struct Shape {
  int64_t S;
  int H, D, P, C;
  int es;            // element size in bytes
  int Hl;            // heads per logical rank
};

// ---- tensor maps (tma_desc.cu) ----------------------------------------------------------------
// "Device-level caching" for TMA descriptors: a plan owns one TmapCache, every launch helper looks its
// descriptors up by (base, dims, strides, box, type, swizzle) and encodes only on a miss, so a steady-state call
// encodes nothing.  Workspace-side maps are hit from the second call on; caller tensors are hit as long as the caller
// passes the same addresses.  Not thread-safe: a plan serves one host thread / caller stream at a time (hcms.h).
struct TmapCache {
  std::unordered_map<std::string, CUtensorMap> maps;
  long long encodes = 0;   // misses = calls of cuTensorMapEncodeTiled
  long long hits = 0;
};
// dims/strides innermost first; strides[0] is implied (element size).  `cache` may be NULL (always encodes).
cudaError_t encode_tensor_map(TmapCache* cache, CUtensorMap* out, CUtensorMapDataType dt, int rank, const void* base,
                              const uint64_t* dims, const uint64_t* strides_bytes, const uint32_t* box,
                              CUtensorMapSwizzle swizzle);

// ---- per-device one-time setup ------------------------------------------------------------------
// Kernel attributes (MaxDynamicSharedMemorySize) are per device: `fn` runs once for every device that becomes
// current when the helper is called (mutex-guarded; 64 devices at most).
struct PerDeviceOnce {
  bool done[64] = {};
  cudaError_t status[64] = {};
};
cudaError_t once_per_device(PerDeviceOnce* state, cudaError_t (*fn)());
// SM count of the current device (cached per device); HCMS status, fails on a non-sm_100 device
int device_sms(int* sms);

// ---- layout kernels (layout_kernels.cu) -------------------------------------------------
constexpr int kMaxPeers = 16;   // ranks a peer table of the distributed layout kernels holds
struct LayoutArgs {
  const void* src[3];
  void* dst[3];
  int n_tensors;
  int64_t S;
  int H, D, P, Hl, es;
  int o_c, h_c;
  bool gather;       // false: [S,H,D] -> [P][S][h_c][D];  true: the inverse
  TmapCache* cache = nullptr;
  // Distributed form (hcms_dist.cu): the strided tensor is this rank's shard [S_local][H][D] (S = S_local) and the
  // dense block of logical rank p is NOT src/dst + p*S*h_c*D but the explicit address peer[t][p] (a region of rank
  // p's chunk buffer, local or mapped peer memory).  NULL = the single-device emulation.
  void* const* peer[3] = {nullptr, nullptr, nullptr};
};
cudaError_t launch_layout_vec(const LayoutArgs& a, cudaStream_t stream);
cudaError_t launch_layout_tma(const LayoutArgs& a, cudaStream_t stream, int num_sms);

// ---- attention kernel (attention_fwd.cu) ------------------------------------------------
constexpr int kAttnPushPadRows = 128;
struct AttnArgs {
  const void* q;     // [P][S][h_c][D] bf16
  const void* k;
  const void* v;
  void* o;
  int64_t S;
  int D, P, h_c;
  float scale;
  float* lse = nullptr;   // optional [P*h_c][S] fp32: log sum_k exp(scale q.k) per row (saved for the backward)
  bool pair = false;      // CTA-pair kernel (HCMS_FLAG_ATTN_PAIR; D = 128 only, ignored otherwise)
  TmapCache* cache = nullptr;
  // Output all-to-all fused into the epilogue (hcms_dist, HCMS_FLAG_DIST_FUSE_OUT; needs P == 1): instead of o, the 128-row
  // output tiles are TMA-stored straight into the sequence-sharded [push_rows][push_heads][D] tensors of n_push ranks --
  // row s of local head j goes to o_push[s / push_rows] at row s % push_rows, head push_head0 + j.  o_push[r] must point at
  // kAttnPushPadRows pad rows in FRONT of rank r's row 0 (tiles that straddle two ranks spill there).  NULL = plain o.
  void* const* o_push = nullptr;
  int n_push = 0;
  int64_t push_rows = 0;
  int push_heads = 0, push_head0 = 0;
};
cudaError_t launch_attention(const AttnArgs& a, cudaStream_t stream);
cudaError_t attention_init();  // sets kernel attributes once per device

// ---- attention backward (attention_bwd.cu) -------------------------------------------------
struct AttnBwdArgs {
  const void* q;       // [P][S][h_c][D] bf16, the chunk buffers the forward read
  const void* k;
  const void* v;
  const void* o;       // the forward's output chunk
  const void* d_o;     // dL/dO', same layout
  const float* lse;    // [P*h_c][S] fp32, natural log, as the forward wrote it
  void* dq;            // outputs, same layout as q
  void* dk;
  void* dv;
  void* stats;         // scratch, attention_bwd_stats_bytes(S, P*h_c) bytes
  float* dq_acc = nullptr;   // single-pass kernel (D = 128): fp32 dQ accumulator, attention_bwd_1pass_acc_bytes(S, P*h_c)
  int* dq_turn = nullptr;    // and its turn counters, attention_bwd_1pass_turn_bytes(S, P*h_c); both NULL = two passes
  int64_t S;
  int D, P, h_c;
  float scale;
  TmapCache* cache = nullptr;
};
cudaError_t launch_attention_bwd(const AttnBwdArgs& a, cudaStream_t stream);   // 3 launches
cudaError_t attention_bwd_init();
size_t attention_bwd_stats_bytes(int64_t S, int heads);
// attention_bwd_1pass.cu: after the statistics kernel; a memset, the kernel and the dQ conversion on `stream`
cudaError_t launch_attention_bwd_1pass(const AttnBwdArgs& a, const void* stats, int s_pad, cudaStream_t stream);
cudaError_t attention_bwd_1pass_init();
size_t attention_bwd_1pass_acc_bytes(int64_t S, int heads);
size_t attention_bwd_1pass_turn_bytes(int64_t S, int heads);

// ---- projection GEMMs (gemm_bf16.cu): C[M,N] = A[M,K] * B[N,K]^T, bf16 -> fp32 -> bf16 -------
// chunk buffers of a plan, for the fused all-to-all modes of the projection GEMMs
struct GemmChunks {
  int C, Hl, P;
  int o[16], h[16];        // Eq. 3 chunk table
  void* base[3][16];       // [tensor][chunk] -> [P][S][h_c][D] bf16 (fuse = 1: Q'_c, K'_c, V'_c; fuse = 2: base[0] = O'_c)
  void* const* peer = nullptr;   // fuse = 1 between real ranks: [(t * C + c) * P + p] -> rank p's [M][h_c][D] rows for this rank's tokens
                                 // (3 * C * P <= 96 pointers); base is then unused
};
struct GemmArgs {
  const void* a;       // [M, K] bf16, row-major
  const void* b;       // [N, K] bf16, row-major (torch.nn.Linear weight)
  void* out[3];        // N / n_per_out output tensors, each [M, n_per_out] bf16 row-major
  int64_t M;
  int N, K;
  int n_per_out;       // multiple of 128; N for a plain GEMM, H*D for the QKV projection
  int rope_outs;       // RoPE on the first rope_outs outputs (0 = none)
  int D;               // head dimension (RoPE only): 64 or 128
  const float* cos;    // [M, D/2] fp32 (RoPE only)
  const float* sin;
  int num_sms;
  int fuse = 0;                       // 0: plain; 1: outputs stored into the chunk buffers (`out` unused);
                                      // 2: A loaded from the O'_c chunk buffers (`a` unused)
  const GemmChunks* chunks = nullptr;
  bool one_cta = false;               // HCMS_FLAG_GEMM_1CTA: the single-CTA kernel also where the CTA-pair kernel applies
  TmapCache* cache = nullptr;
};
cudaError_t launch_gemm(const GemmArgs& a, cudaStream_t stream);
cudaError_t gemm_init();

}  // namespace hcms
