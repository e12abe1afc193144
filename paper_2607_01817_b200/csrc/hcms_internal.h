// Internal declarations shared by the translation units of libhcms (not installed).
#pragma once

#include <cuda.h>  // CUtensorMap and enums only; libcuda is reached through cudaGetDriverEntryPoint
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>
#include <cstdio>
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

// ---- layout kernels (layout_kernels.cu) -------------------------------------------------
struct LayoutArgs {
  const void* src[3];
  void* dst[3];
  int n_tensors;
  int64_t S;
  int H, D, P, Hl, es;
  int o_c, h_c;
  bool gather;       // false: [S,H,D] -> [P][S][h_c][D];  true: the inverse
};
cudaError_t launch_layout_vec(const LayoutArgs& a, cudaStream_t stream);
cudaError_t launch_layout_tma(const LayoutArgs& a, cudaStream_t stream, int num_sms);

// ---- attention kernel (attention_fwd.cu) ------------------------------------------------
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
};
cudaError_t launch_attention(const AttnArgs& a, cudaStream_t stream);
cudaError_t attention_init();  // sets kernel attributes once; resolves cuTensorMapEncodeTiled

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
  int64_t S;
  int D, P, h_c;
  float scale;
};
cudaError_t launch_attention_bwd(const AttnBwdArgs& a, cudaStream_t stream);   // 3 launches
cudaError_t attention_bwd_init();
size_t attention_bwd_stats_bytes(int64_t S, int heads);

// ---- projection GEMMs (gemm_bf16.cu): C[M,N] = A[M,K] * B[N,K]^T, bf16 -> fp32 -> bf16 -------
// chunk buffers of a plan, for the fused all-to-all modes of the projection GEMMs
struct GemmChunks {
  int C, Hl, P;
  int o[16], h[16];        // Eq. 3 chunk table
  void* base[3][16];       // [tensor][chunk] -> [P][S][h_c][D] bf16 (fuse = 1: Q'_c, K'_c, V'_c; fuse = 2: base[0] = O'_c)
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
};
cudaError_t launch_gemm(const GemmArgs& a, cudaStream_t stream);
cudaError_t gemm_init();

// ---- driver entry point for tensor maps (tma_desc.cu) ------------------------------------
// dims/strides innermost first; strides[0] is implied (element size). Returns cudaSuccess or an error.
cudaError_t encode_tensor_map(CUtensorMap* out, CUtensorMapDataType dt, int rank, const void* base,
                              const uint64_t* dims, const uint64_t* strides_bytes, const uint32_t* box,
                              CUtensorMapSwizzle swizzle);

}  // namespace hcms
