/*
 * hcms.h -- C ABI of libhcms: the HCMS (Head-Chunked Multi-Stream) attention hot path,
 * emulated on ONE NVIDIA B200 (sm_100a).
 *
 * Source of the method: arxiv/paper_2607_01817 (PAPER.md; "L<n>" = PAPER.md line).
 *   - Ulysses all-to-all sequence parallelism: the input all-to-all turns "sequence-sharded,
 *     heads-complete" activations into "sequence-complete, heads-sharded" ones, attention runs,
 *     the output all-to-all inverts the layout (L45, L59).
 *   - HCMS splits the heads of every rank into C chunks (Eq. 3; Table 8),
 *     runs all all-to-alls on a communication stream and all attention calls on a compute
 *     stream, ordered by CUDA events (section 3.4-3.5; Algorithm 1).
 *
 * Emulation: the P ranks are logical.  The concatenation, in rank order, of the P ranks'
 * shards [S/P, H, D] is the global tensor [S, H, D]; rank p owns global heads
 * [p*Hl, (p+1)*Hl), Hl = H/P; chunk c is local heads [o_c, o_c+h_c) on every rank with
 * h_c = floor(Hl/C) + 1[c < Hl mod C], o_c = sum_{c'<c} h_c'.  The all-to-all is a device
 * layout kernel writing the head-sharded chunk buffer
 *
 *        X'_c [P][S][h_c][D]   with   X'_c[p][s][j][d] = X[s][p*Hl + o_c + j][d]
 *
 * (row-major, densely packed); this layout is part of the contract.
 *
 * Conventions
 *   - every function is extern "C", returns an int status (HCMS_OK == 0, errors < 0) unless it
 *     returns a size or a string, never throws, never exits, never synchronises the host
 *     unless stated;
 *   - "device pointer" = CUDA device memory owned by the caller; "host pointer" = ordinary host
 *     memory owned by the caller; the library never frees caller memory;
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream);
 *   - there is NO CPU fallback: without a compute-capability-10.x device every call that needs
 *     the GPU returns HCMS_ERR_UNSUPPORTED_DEVICE or HCMS_ERR_CUDA.
 */
#ifndef HCMS_H_
#define HCMS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HCMS_VERSION 600 /* major*10000 + minor*100 + patch */

/* ---- status codes ------------------------------------------------------------------- */
enum {
  HCMS_OK = 0,
  HCMS_ERR_INVALID_ARG = -1,         /* NULL pointer, non-positive size, non-finite or negative scale */
  HCMS_ERR_UNSUPPORTED_SHAPE = -2,   /* S%P, H%P, C>H/P, D not in {64,128}, D*es%16 */
  HCMS_ERR_UNSUPPORTED_DTYPE = -3,   /* attention needs bf16; layout kernels take 2- or 4-byte elements */
  HCMS_ERR_UNSUPPORTED_DEVICE = -4,  /* no CUDA device of compute capability 10.x */
  HCMS_ERR_MISALIGNED = -5,          /* a device pointer is not 16-byte aligned */
  HCMS_ERR_ALIAS = -6,               /* `out` overlaps q, k or v */
  HCMS_ERR_PLAN_MISMATCH = -7,       /* S,H,D,P,C differ from the plan's, or chunk index out of range */
  HCMS_ERR_WORKSPACE_TOO_SMALL = -8,
  HCMS_ERR_CUDA = -9                 /* a CUDA call failed; hcms_last_error() carries its text */
};

/* ---- element types ------------------------------------------------------------------ */
enum {
  HCMS_DTYPE_BF16 = 0, /* 2 bytes; the only type hcms_attention_* accepts */
  HCMS_DTYPE_F32 = 1,  /* 4 bytes; layout kernels only (BASELINE.json config 1's permutation check) */
  HCMS_DTYPE_F16 = 2   /* 2 bytes; layout kernels only */
};

/* ---- plan flags ----------------------------------------------------------------------- */
#define HCMS_FLAG_SERIAL 0x1u          /* Ulysses baseline order (Eq. 1): all scatters, all
                                          attention, all gathers, on the caller's stream, no overlap */
#define HCMS_FLAG_LAYOUT_TMA 0x2u      /* layout kernels use the TMA bulk-tensor variant instead of the
                                          128-bit ld/st variant (same bits out) */
#define HCMS_FLAG_SPLIT_COMM 0x4u      /* separate streams for input and output all-to-all (Eq. 8
                                          "all three in parallel"); default is Alg. 1's single S_comm */
#define HCMS_FLAG_HOST_ROUTE_Q 0x10u   /* config 5: this tensor's chunk crosses an emulated wire through pinned  */
#define HCMS_FLAG_HOST_ROUTE_K 0x20u   /* host memory: scatter -> device send buffer -> D2H -> H2D -> Q'_c/K'_c/ */
#define HCMS_FLAG_HOST_ROUTE_V 0x40u   /* V'_c, and O'_c -> D2H -> H2D -> device receive buffer -> gather, to    */
#define HCMS_FLAG_HOST_ROUTE_O 0x80u   /* raise the communication ratio rho (section 3.7).  Same bits.     */
#define HCMS_FLAG_DEBUG_NO_COMM_WAIT 0x100u /* TEST ONLY: drop the compute stream's wait on E_c^comm
                                          (Eq. 6) so a negative test can observe the race */

#define HCMS_FLAG_PROFILE 0x200u       /* record timing-enabled CUDA events around every scatter, attention
                                          and gather of hcms_attention_forward, each on the stream it runs on;
                                          read them with hcms_plan_timings */

#define HCMS_FLAG_SINGLE_COMP 0x400u   /* issue every attention launch on ONE compute stream, literally as
                                          Alg. 1 does.  Default: S_comp is realised as two CUDA streams that
                                          alternate by chunk parity, so that chunk c+1's thread blocks fill
                                          the SMs vacated by the last (partial) wave of chunk c; the event
                                          dependencies of Eq. 6-7 are unchanged and so are the bits. */

#define HCMS_FLAG_TRAINING 0x800u      /* the plan also serves the backward pass (L304, Table 15): its
                                          workspace doubles (dO'_c, dQ'_c, dK'_c, dV'_c per chunk), and
                                          hcms_attention_forward saves the row statistic lse_i = log sum_k
                                          exp(scale q_i.k_k) of every head (H*S floats) and keeps Q'_c, K'_c,
                                          V'_c, O'_c for hcms_attention_backward */

#define HCMS_FLAG_FUSE_A2A 0x1000u     /* hcms_layer_forward only: the QKV-projection epilogue stores q, k, v
                                          straight into the head-sharded chunk buffers Q'_c, K'_c, V'_c (the input
                                          all-to-all is the epilogue's TMA store; on P real GPUs it would be a store to
                                          peer memory) and the output projection loads its A operand straight from the
                                          O'_c chunk buffers (output all-to-all + Concat in the producer's TMA load):
                                          2 + C launches per layer, no scatter / gather kernels, no [S,H,D]
                                          intermediates.  Same bits as the unfused layer.  Needs C <= 16, H/P <= 64. */

#define HCMS_FLAG_GRAPH 0x2000u        /* hcms_attention_forward captures the whole chunk pipeline (every kernel and copy
                                          on S_comm / S_comp with the event forks and joins of Eq. 6-7) into a CUDA
                                          graph on first use and replays it with ONE launch per call; other tensor
                                          addresses or another scale capture again.  For launch-bound shapes
                                          (BASELINE.json configs 1-2).  Same bits.  Excludes HCMS_FLAG_PROFILE. */

#define HCMS_FLAG_ATTN_PAIR 0x4000u    /* D = 128 only: the attention forward runs on CTA pairs (thread-block clusters of 2,
                                          tcgen05 cta_group::2): the two CTAs share every K_j / V_j tile (each loads
                                          half) and the leader CTA issues M = 256 MMAs over both CTAs' query tiles.
                                          Same bits as the single-CTA kernel.  Measured on B200 (cfg 3): -13 % power at
                                          equal clocks, +0.5 % throughput under the power cap; off by default. */

#define HCMS_FLAG_HOST_STAGED 0x8000u   /* hcms_attention_forward_host copies whole tensors to device staging first and runs
                                          the device path on them (the first implementation).  Default: the host link
                                          is the wire -- strided cudaMemcpy2DAsync copies carry chunk c of rank p's
                                          heads straight between the host tensors and the chunk buffers (they ARE the
                                          all-to-all), chunk c+1's transfer overlapping chunk c's attention. */

#define HCMS_FLAG_GEMM_1CTA 0x10000u    /* projections (hcms_qkv_projection_rope, hcms_output_projection, hcms_layer_forward):
                                          use the single-CTA tcgen05 GEMM (128 x 256 tiles) also where the default
                                          CTA-pair kernel (cta_group::2, 256 x 256 tiles) applies.  Same bits. */

#define HCMS_FLAG_DEBUG_ATTN_ONLY 0x20000u /* MEASUREMENT ONLY: hcms_attention_forward skips the scatter and gather
                                          kernels (events, streams and attention launches unchanged), so that the
                                          compute side of the pipeline can be timed in the same stream arrangement
                                          without copies; the chunk buffers must hold an earlier call's data */

#define HCMS_FLAG_BWD_ONE_PASS 0x40000u  /* D = 128: hcms_attention_backward (HCMS_FLAG_TRAINING plans) and hcms_attention_backward_chunk
                                          (any bf16 plan) form S = QK^T and dP = dO V^T once per (key tile, query tile) instead
                                          of once per pass (5 executed contractions instead of 7): one kernel keeps dK_j, dV_j in
                                          tensor memory and adds its dQ partials to an fp32 accumulator in a fixed key-tile
                                          order (deterministic; gradients still independent of P and C).  Scratch, allocated on
                                          first use: TWO accumulators (one per compute stream, chunks alternate) of
                                          P*h_max*(S rounded up to 64)*D*4 bytes each, h_max = the largest chunk, plus
                                          2*P*h_max*(S/64 + 1) 4-byte counters -- 2 x 201 MB at BASELINE.json config 3.
                                          A CTA of this kernel waits for the CTAs of the lower key tiles of its head; each CTA
                                          draws its key tile from a per-head ticket counter as it starts, so it only ever waits
                                          for CTAs that are already running (no reliance on blockIdx dispatch order).
                                          Measured slower than the two-pass default.  Ignored at D = 64. */

#define HCMS_FLAG_RECYCLE_WS 0x80000u    /* chunk c shares its buffers Q'_c, K'_c, V'_c, O'_c with chunk c - 2: the workspace is 2 buffer
                                          sets sized for a largest chunk instead of one set per chunk (2/C of it for even
                                          chunks; the paper reports 8.7 % lower peak memory for HCMS, Table 16),
                                          and the communication stream runs A_{c-2}^out before A_c^in instead of all
                                          inputs first (same Eq. 6-7 waits).  Same bits.  No effect for C <= 2.  Excludes
                                          TRAINING, FUSE_A2A, SPLIT_COMM, DEBUG_ATTN_ONLY.  hcms_chunk_layout reports the
                                          shared offsets. */

#define HCMS_FLAG_DIST_FUSE_OUT 0x100000u /* hcms_dist_plan only: the output all-to-all (Alg. 1 line 21) happens in the attention
                                          kernel's epilogue -- every 128-row output tile is TMA-stored straight into the
                                          destination rank's sequence-sharded output inside that rank's exchange block
                                          (peer memory), instead of O'_c followed by a pull-gather kernel: one kernel does
                                          the compute and its collective.  The exchange block grows by S/P*H*D*2 bytes; the
                                          call ends with one local copy into `out`.  Same bits. */

#define HCMS_FLAG_DEBUG_DIST_FAIL 0x200000u /* TEST ONLY, hcms_dist_plan: every forward call on the plan fails with HCMS_ERR_CUDA
                                          in the attention phase, after its pushes and the first flag wait were enqueued, so
                                          that a test can check the error path (join, poisoned plan) */

typedef struct hcms_plan hcms_plan_t;

/* ---- introspection (host only, no GPU needed) ---------------------------------------- */
int hcms_version(void);
const char* hcms_status_string(int status); /* static string, never NULL */
const char* hcms_last_error(void);          /* thread-local text of the last failure ("" if none) */

/*
 * Chunk table, Eq. 3 (L83-84) applied to the per-rank head count (Table 8,
 * "more-first-less-later" L221).  Host only.  o[c], h[c] for c < C; either array may be NULL.
 * Errors: INVALID_ARG (heads_per_rank <= 0, C <= 0), UNSUPPORTED_SHAPE (C > heads_per_rank).
 */
int hcms_chunk_table_host(int heads_per_rank, int C, int* o, int* h);

/*
 * Time model of section 3.7 / Appendix A (host only, doubles in any one time unit).
 *   hcms_model_t_hcms : Eq. 10  T_0 + T_comm/C + T_attn + C*beta
 *   hcms_model_c_star : Theorem 1  sqrt(T_comm/beta)
 *   hcms_model_speedup: Eq. 11  1/(1 - rho*(C-1)/C + C*beta/T_total)
 *   hcms_model_s_max  : Theorem 2  1/(1-rho)
 * Arguments out of domain (C<=0, beta<=0 for c_star, rho>=1) yield NaN.
 */
double hcms_model_t_hcms(int C, double t0, double t_comm, double t_attn, double beta);
double hcms_model_c_star(double t_comm, double beta);
double hcms_model_speedup(int C, double rho, double beta, double t_total);
double hcms_model_s_max(double rho);
/*
 * Integer chunk count from the model (adaptive C, the paper's future work L346, via Theorem 1):
 * the C in [1, heads_per_rank] that minimises Eq. 10's C-dependent part  t_comm/C + C*beta.  That
 * function is convex in C, so the minimiser is floor(C*) or ceil(C*), C* = sqrt(t_comm/beta), clamped
 * to the range; ties go to the smaller C (fewer launches).  beta <= 0 (no per-chunk overhead) returns
 * heads_per_rank; t_comm <= 0 returns 1.  Returns 0 if heads_per_rank <= 0 or an argument is NaN.
 * Worked pin: Table 12 row 1 (L440): t_comm = 0.396*73.3 ms, beta = 1.41 ms, 5 heads per rank -> 5.
 */
int hcms_model_choose_chunks(int heads_per_rank, double t_comm, double beta);

/* ---- plan ------------------------------------------------------------------------------ */
/*
 * Create a plan for global tensors [S,H,D], P logical ranks, C head chunks (Alg. 1's
 * `num_chunks`) on the CURRENT device.  Validates the shape, builds the chunk table, creates the
 * communication and compute streams (device-level stream caching, L221) and 5+2C timing-disabled
 * events, and sets the kernel attributes once per device.  The chunk workspace (4*S*H*D*es bytes +
 * alignment; twice that plus H*S floats under HCMS_FLAG_TRAINING) is allocated on the first call
 * that needs it, unless hcms_plan_set_workspace supplied caller memory before.  Every TMA
 * descriptor a call needs is encoded once and cached in the plan, keyed by address and shape
 * (hcms_plan_tensor_map_encodes counts the encodes).  `*plan` is owned by the library; free it
 * with hcms_plan_destroy.
 *
 * Concurrency: a plan owns ONE set of streams, events and chunk buffers, so it serves one host
 * thread and one caller stream at a time; calls on the same plan from two caller streams must be
 * ordered by the caller (or use two plans).  Every call on a plan must be made with the plan's
 * device current (PLAN_MISMATCH otherwise).
 * Errors: INVALID_ARG, UNSUPPORTED_SHAPE, UNSUPPORTED_DTYPE, UNSUPPORTED_DEVICE, CUDA.
 */
int hcms_plan(hcms_plan_t** plan, int64_t S, int H, int D, int P, int C, int dtype, uint32_t flags);
int hcms_plan_destroy(hcms_plan_t* plan); /* synchronises the plan's streams; NULL is a no-op */

/* Bytes of device workspace the plan needs (0 for a NULL plan). */
size_t hcms_plan_workspace_bytes(const hcms_plan_t* plan);
/*
 * Use caller memory (device pointer, 256-byte aligned, >= hcms_plan_workspace_bytes) as the
 * workspace; the plan's own allocation, if any, is released (after synchronising the plan's
 * streams).  The caller keeps ownership.  A captured graph (HCMS_FLAG_GRAPH) and the forward
 * state saved for hcms_attention_backward are discarded: the next forward captures again.
 * Errors: INVALID_ARG, MISALIGNED, WORKSPACE_TOO_SMALL.
 */
int hcms_plan_set_workspace(hcms_plan_t* plan, void* dev, size_t bytes);

/* Copy the plan's chunk table to o[C], h[C] (either may be NULL). */
int hcms_chunk_table(const hcms_plan_t* plan, int* o, int* h);
/*
 * Layout of chunk c inside the workspace: `bytes` = size of one chunk tensor
 * (P*S*h_c*D*es); q_off,k_off,v_off,o_off = byte offsets of Q'_c, K'_c, V'_c, O'_c from the
 * workspace base.  Any output pointer may be NULL.  Errors: INVALID_ARG, PLAN_MISMATCH.
 */
int hcms_chunk_layout(const hcms_plan_t* plan, int c, size_t* bytes, size_t* q_off, size_t* k_off,
                      size_t* v_off, size_t* o_off);
/* Device address of the workspace (allocates the plan-owned one if none exists yet; NULL on failure); for tests
 * (NaN poisoning, inspection). */
void* hcms_plan_workspace(hcms_plan_t* plan);
/* Number of cuTensorMapEncodeTiled calls this plan has made so far: constant across repeated calls on the same
 * tensors (the descriptors live in the plan). */
long long hcms_plan_tensor_map_encodes(const hcms_plan_t* plan);

/* ---- the hot path ----------------------------------------------------------------------- */
/*
 * Algorithm 1 lines 4-26 for one layer: for every chunk c, scatter Q,K,V (input all-to-all,
 * line 8), attention O'_c = softmax(Q'_c K'_c^T * scale) V'_c per head, non-causal (line 15,
 * Eq. 2), gather O'_c into `out` (output all-to-all + Concat, lines 21, 26).
 *
 * q,k,v,out: device pointers, bf16, contiguous [S,H,D] = the P ranks' shards [S/P,H,D] in rank
 * order; 16-byte aligned; `out` must not overlap q,k,v.  S,H,D,P,C must equal the plan's
 * (PLAN_MISMATCH otherwise).  scale: finite, >= 0 (the paper's workloads use 1/sqrt(D)).
 *
 * Asynchronous: work is ordered after everything already enqueued on `stream` (E_main, Alg. 1
 * line 5) and `stream` is made to wait for the result (line 25); `out` is valid once the caller
 * synchronises `stream`.  Unless HCMS_FLAG_SERIAL is set, scatters/gathers run on the plan's
 * communication stream and attention on its compute stream, with Attn_c waiting on E_c^comm and
 * the gather of chunk c on E_c^comp (Eq. 6-7).  Numerics: bf16 operands, fp32 scores,
 * online softmax and accumulation in fp32, bf16 output (round to nearest even).  The result for
 * a given (q,k,v,scale) is bitwise independent of P and C (Table 14).
 * Errors: INVALID_ARG, PLAN_MISMATCH, MISALIGNED, ALIAS, UNSUPPORTED_DTYPE, CUDA.
 */
int hcms_attention_forward(hcms_plan_t* plan, const void* q, const void* k, const void* v, void* out,
                           int64_t S, int H, int D, int P, int C, float scale, void* stream);

/*
 * Same computation with HOST buffers (q,k,v,out: host pointers, bf16 [S,H,D]; pinned memory
 * makes the copies asynchronous) and SYNCHRONISES `stream` before returning.  Default: per head chunk,
 * strided host-to-device copies on S_comm deliver every rank's heads of the chunk directly into Q'_c, K'_c, V'_c
 * (the copy engines perform the input all-to-all), attention runs on S_comp as each chunk lands, strided
 * device-to-host copies on a second communication stream return O'_c into `out` (output all-to-all + Concat);
 * same events and ordering as hcms_attention_forward, same bits.  With HCMS_FLAG_HOST_STAGED (or SERIAL / GRAPH
 * plans): whole tensors go to plan-owned device staging (4*S*H*D*2 bytes, allocated on first use), the device
 * path runs on them, and `out` is copied back.
 */
int hcms_attention_forward_host(hcms_plan_t* plan, const void* q, const void* k, const void* v, void* out,
                                int64_t S, int H, int D, int P, int C, float scale, void* stream);

/* ---- single steps (tests time and compare each kernel on its own) ----------------------- */
/*
 * Input all-to-all of chunk c for up to three tensors in one launch (Alg. 1 line 8
 * "AllToAll(Q_c,K_c,V_c)"): dst_i[p][s][j][d] = src_i[s][p*Hl+o_c+j][d] for i < n_tensors
 * (1..3).  src_i: device [S,H,D]; dst_i: device [P][S][h_c][D]; any 2- or 4-byte element
 * type as given to hcms_plan; all 16-byte aligned; bits are copied untouched.
 */
int hcms_a2a_scatter(hcms_plan_t* plan, int n_tensors, const void* const* src, void* const* dst, int c,
                     void* stream);
/* Output all-to-all of chunk c: dst[s][p*Hl+o_c+j][d] = src[p][s][j][d]; writes only chunk c's heads. */
int hcms_a2a_gather(hcms_plan_t* plan, const void* src, void* dst, int c, void* stream);
/*
 * Attention of chunk c on head-sharded buffers qc,kc,vc -> oc, all device [P][S][h_c][D] bf16,
 * 16-byte aligned: for every p, j:  oc[p][:,j,:] = softmax(qc[p][:,j,:] kc[p][:,j,:]^T * scale) vc[p][:,j,:].
 */
int hcms_attention_chunk(hcms_plan_t* plan, const void* qc, const void* kc, const void* vc, void* oc, int c,
                         float scale, void* stream);

/* Number of kernels + async copies the last hcms_attention_forward on this plan enqueued. */
int hcms_plan_last_launch_count(const hcms_plan_t* plan);
/* How many times a HCMS_FLAG_GRAPH plan has captured its pipeline (1 after any number of calls on the same tensors). */
int hcms_plan_graph_captures(const hcms_plan_t* plan);

/*
 * Device durations, in milliseconds, of the steps of a recent hcms_attention_forward on a plan made
 * with HCMS_FLAG_PROFILE.  calls_back = 0 is the last call, 1 the one before, ... up to
 * HCMS_PROFILE_RING-1 calls are kept.  scatter_ms[c] = input all-to-all of chunk c (T_in share, incl.
 * the host route if any), attn_ms[c] = attention of chunk c, gather_ms[c] = output all-to-all of
 * chunk c; host arrays of C floats, any may be NULL.  Each is the elapsed time between two events
 * recorded on the stream the step ran on, so time spent queueing behind another stream's kernels
 * for the same SMs is included.  SYNCHRONISES the host with those events.
 * Errors: INVALID_ARG (NULL plan, plan without HCMS_FLAG_PROFILE, calls_back out of range or
 * older than the first call), CUDA.
 */
#define HCMS_PROFILE_RING 64
int hcms_plan_timings(hcms_plan_t* plan, int calls_back, float* scatter_ms, float* attn_ms, float* gather_ms);
/*
 * Same events, read as a span: *span_ms = time from the begin event of chunk 0 to the end event of chunk
 * C-1 of step kind `step` (0 = scatter, 1 = attention, 2 = gather) in that call.  Attention launches of
 * consecutive chunks may overlap (two alternating compute streams), so the attention time of a layer is
 * this span, not the sum of hcms_plan_timings' attn_ms.  SYNCHRONISES the host with those events.
 * Errors: as hcms_plan_timings, plus INVALID_ARG for step outside 0..2 or NULL span_ms.
 */
int hcms_plan_step_span(hcms_plan_t* plan, int calls_back, int step, float* span_ms);
/*
 * Same events, read as a timeline (the measured counterpart of Fig. 2): begin_ms[k*C + c] and
 * end_ms[k*C + c] are the begin / end of step kind k (0 = scatter, 1 = attention, 2 = gather) of chunk c,
 * in milliseconds after the begin event of chunk 0's scatter.  Host arrays of 3*C floats each.
 * SYNCHRONISES the host with those events.  Errors: as hcms_plan_timings, plus INVALID_ARG for NULL arrays.
 */
int hcms_plan_timeline(hcms_plan_t* plan, int calls_back, float* begin_ms, float* end_ms);

/* ---- adaptive chunk count (the paper's future work, L346) ------------------- */
/*
 * Measure hcms_attention_forward for every C in [1, min(max_C, H/P)] on the caller's tensors and
 * report the fastest: for each C a temporary plan (flags = `flags` without SERIAL/PROFILE) runs one
 * warm-up and `reps` timed calls between two CUDA events on `stream`; ms_per_call[C-1] = mean time
 * of a call (host array of max_C floats, may be NULL; entries beyond H/P are set to -1), *best_C = the
 * argmin (ties to the smaller C).  q,k,v,out as for hcms_attention_forward; `out` holds the result of
 * the last measured call (identical bits for every C).  SYNCHRONISES the host; allocates and frees one
 * workspace per C.  Errors: INVALID_ARG (NULL, max_C < 1, reps < 1), those of hcms_plan and of
 * hcms_attention_forward.
 */
int hcms_autotune_chunks(int64_t S, int H, int D, int P, int dtype, uint32_t flags, const void* q, const void* k,
                         const void* v, void* out, float scale, void* stream, int max_C, int reps, int* best_C,
                         float* ms_per_call);

/*
 * The same measurement through hcms_attention_forward_host: q,k,v,out are HOST pointers (pinned memory for
 * asynchronous copies), the chunks cross the host link, where the communication ratio is large and the chunk count
 * matters (measured on B200, cfg 3: C = 4 -> 23.6 ms, C = 6 -> 21.9 ms).  bf16 only; `flags` without SERIAL / PROFILE /
 * GRAPH.  Arguments, results and errors as hcms_autotune_chunks.
 */
int hcms_autotune_chunks_host(int64_t S, int H, int D, int P, uint32_t flags, const void* q, const void* k, const void* v,
                              void* out, float scale, void* stream, int max_C, int reps, int* best_C, float* ms_per_call);

/* ---- the attention layer around the hot path --------------------------------- */
/*
 * Section 3.1 (L59): "QKV projection -> RoPE positional encoding -> input all-to-all -> attention
 * computation -> output all-to-all -> output projection"; Algorithm 1 (L170) lines 2, 3 and 27.  These are
 * the T_other of Eq. 1 (L61).  Both projections are torch.nn.Linear-style maps without bias (the paper
 * names none):  C[M,N] = A[M,K] * B[N,K]^T, bf16 operands, fp32 accumulation, bf16 result (RNE).
 *
 * hcms_gemm_bf16_nt: the bare contraction.  a: device [M,K] bf16, b: device [N,K] bf16, c: device [M,N]
 * bf16, all row-major, 16-byte aligned, c not overlapping a or b.  K % 8 == 0, N % 128 == 0.
 * Asynchronous on `stream`.  Errors: INVALID_ARG, UNSUPPORTED_SHAPE, MISALIGNED, ALIAS,
 * UNSUPPORTED_DEVICE, CUDA.
 */
int hcms_gemm_bf16_nt(const void* a, const void* b, void* c, int64_t M, int N, int K, void* stream);
/*
 * Alg. 1 lines 2-3 in one kernel: [q|k|v] = x * w_qkv^T, then the rotary embedding on q and k.
 *   x: device [S, Dm] bf16 (the P ranks' token shards in rank order); w_qkv: device [3*H*D, Dm] bf16, row n =
 *   output feature n, features ordered q heads, k heads, v heads, D consecutive features per head;
 *   q,k,v: device [S,H,D] bf16 (the layout hcms_attention_forward takes).
 *   rope_cos, rope_sin: device [S, D/2] fp32 tables, or both NULL for no rotation.  For token s and pair
 *   i < D/2 of every head:  (x[2i], x[2i+1]) <- (x[2i]*c - x[2i+1]*s, x[2i]*s + x[2i+1]*c), c = cos[s][i],
 *   s = sin[s][i]  (adjacent-pair convention of RoFormer [34]; the caller's table fixes the position scheme,
 *   1-D or the 3-D grid of a video DiT).  The rotation is applied to the fp32 accumulators, then rounded once.
 * S,H,D are the plan's; Dm % 128 == 0 and H*D % 128 == 0.  Asynchronous on `stream`.
 * Errors: INVALID_ARG (NULL, only one table NULL, Dm <= 0), UNSUPPORTED_SHAPE, UNSUPPORTED_DTYPE (plan not
 * bf16), MISALIGNED, CUDA.
 */
int hcms_qkv_projection_rope(hcms_plan_t* plan, const void* x, const void* w_qkv, const void* rope_cos,
                             const void* rope_sin, void* q, void* k, void* v, int Dm, void* stream);
/* Alg. 1 line 27: y[S,Dm] = o[S,H*D] * w_o^T; o: device [S,H,D] bf16 (the Concat of line 26), w_o: device
 * [Dm, H*D] bf16, y: device [S,Dm] bf16.  Same rules and errors as above. */
int hcms_output_projection(hcms_plan_t* plan, const void* o, const void* w_o, void* y, int Dm, void* stream);
/*
 * Algorithm 1 lines 2-27 for one layer: hcms_qkv_projection_rope on `stream` (main stream), then
 * hcms_attention_forward (lines 4-26: E_main, S_comm / S_comp, events) on the plan-owned q,k,v,o buffers
 * (4*S*H*D*2 bytes, allocated on first use), then hcms_output_projection on `stream`.
 * x: device [S,Dm] bf16; y: device [S,Dm] bf16, not overlapping x; weights and tables as above.
 * S,H,D,P,C must equal the plan's.  Asynchronous: y is valid once the caller synchronises `stream`.
 * With HCMS_FLAG_PROFILE the three parts are bracketed by events (hcms_plan_layer_timings).
 * Errors: those of the three calls it makes.
 */
int hcms_layer_forward(hcms_plan_t* plan, const void* x, const void* w_qkv, const void* w_o, const void* rope_cos,
                       const void* rope_sin, void* y, int64_t S, int Dm, int H, int D, int P, int C, float scale,
                       void* stream);
/* Device address of the plan-owned layer buffer `which` (0 = q, 1 = k, 2 = v after RoPE, 3 = o) of
 * hcms_layer_forward, each [S,H,D] bf16; NULL before the first call.  For tests. */
void* hcms_plan_layer_buffer(const hcms_plan_t* plan, int which);
/* Device milliseconds of the last hcms_layer_forward on a HCMS_FLAG_PROFILE plan: QKV projection + RoPE,
 * lines 4-26 (all-to-alls and attention), output projection.  Any pointer may be NULL.  SYNCHRONISES the
 * host with those events.  Errors: INVALID_ARG (no profiled layer call yet), CUDA. */
int hcms_plan_layer_timings(hcms_plan_t* plan, float* qkv_ms, float* hcms_ms, float* out_ms);

/* ---- backward of the hot path ----------------------------------------------- */
/*
 * "HCMS is compatible with PyTorch autograd ... forward+backward combined execution" (L304; Table 15
 * L479-483; future work L346).  Autograd differentiates Alg. 1; the all-to-alls are permutations, so the
 * backward of lines 4-26 is the same pipeline run on the gradients: per head chunk c
 *     input all-to-all of dO (scatter)  ->  attention backward on every rank's heads  ->  output all-to-all
 *     of dQ'_c, dK'_c, dV'_c (one gather launch for the three),
 * with chunk c+1's all-to-all on S_comm overlapping chunk c's attention backward on S_comp, ordered by the
 * same events E_main, E_c^comm, E_c^comp (Eq. 6-7).  Per head, with P = softmax(scale Q K^T):
 *     dV = P^T dO,  dP = dO V^T,  dS = P o (dP - rowsum(dO o O)),  dQ = scale dS K,  dK = scale dS^T Q.
 * P is recomputed from the saved lse; two deterministic tcgen05 passes (dK/dV, then dQ) without atomics, so
 * the gradients are bitwise independent of P and C.  bf16 operands (P, dS rounded to bf16 for the MMAs), fp32
 * accumulation, bf16 gradients.
 *
 * hcms_attention_backward: `plan` must carry HCMS_FLAG_TRAINING and the last hcms_attention_forward on it must
 * be the forward being differentiated (its Q'_c, K'_c, V'_c, O'_c and lse are read from the workspace; `scale`
 * must be the same).  dout: device [S,H,D] bf16 = dL/d(out); dq, dk, dv: device [S,H,D] bf16, distinct, not
 * overlapping dout.  Asynchronous on `stream` like the forward.  HCMS_FLAG_SERIAL runs it on `stream` alone.
 * Errors: INVALID_ARG (NULL, plan without TRAINING, no forward yet or workspace replaced since, `scale` not
 * bit-equal to the forward's -- the saved lse belongs to that scale), PLAN_MISMATCH, MISALIGNED, ALIAS, CUDA.
 */
int hcms_attention_backward(hcms_plan_t* plan, const void* dout, void* dq, void* dk, void* dv, int64_t S, int H,
                            int D, int P, int C, float scale, void* stream);
/*
 * Single steps on caller-supplied chunk buffers ([P][S][h_c][D] bf16 unless stated; chunk c of the plan):
 * hcms_attention_chunk_lse = hcms_attention_chunk that also writes lse: device [P*h_c][S] fp32, natural log.
 * hcms_attention_backward_chunk: qc,kc,vc,oc,doc and lse in, dqc,dkc,dvc out (3 launches: delta/lse packing,
 * dK/dV pass, dQ pass); works on any bf16 plan (scratch for the packed statistics is allocated on first use).
 */
int hcms_attention_chunk_lse(hcms_plan_t* plan, const void* qc, const void* kc, const void* vc, void* oc, void* lse,
                             int c, float scale, void* stream);
int hcms_attention_backward_chunk(hcms_plan_t* plan, const void* qc, const void* kc, const void* vc, const void* oc,
                                  const void* doc, const void* lse, void* dqc, void* dkc, void* dvc, int c,
                                  float scale, void* stream);
/*
 * hcms_attention_backward_chunk for callers that may not allocate device memory: no plan, no cudaMalloc, no cudaFree,
 * no allocating library routine inside the call.  Meant for an operator embedded in a framework whose caching allocator
 * already owns the card (a raw cudaMalloc from a library fails there or escapes the host application's accounting), for
 * serving loops that cannot take cudaMalloc's device-wide synchronisation after start-up, and for processes whose memory
 * budget (MIG slice, MPS client limit) is fully committed at launch.
 *
 * Same three kernels, same bits as hcms_attention_backward_chunk (L304, Table 15; the formulas above).  The
 * packed row statistics {lse*log2(e), dO.O}, P*h_c*(S rounded up to 64)*8 bytes, go to a fixed array inside the
 * library's device image instead of plan-owned memory: HCMS_STATIC_SCRATCH_BYTES (4 MiB) that EVERY GPU loading
 * libhcms.so holds until the process exits.  Larger problems return HCMS_ERR_WORKSPACE_TOO_SMALL (checked first, before
 * any device work; nothing is enqueued): 4 MiB is 524288 (head, row) pairs, e.g. a 12-head chunk of BASELINE.json
 * config 3 (S = 32760), 8 heads of config 4 or 5 heads of config 5; split the heads over several calls beyond that.
 *
 * qc,kc,vc,oc,doc: device [P][S][h_c][D] bf16; lse: device [P*h_c][S] fp32 (as hcms_attention_chunk_lse writes it);
 * dqc,dkc,dvc: device outputs, same layout as qc; all 16-byte aligned, all owned by the caller.  D = 64 or 128.
 * Asynchronous on `stream`; the current device must be the one holding the tensors.
 *
 * First call on each device: looks up the array's device address (cudaGetSymbolAddress, once per device, cached) and
 * sets the kernels' attributes; the runtime may load the library's device image at that moment, so make that first
 * call during start-up, before any stream capture begins.  Later calls do neither.
 * The array is shared by every call in the process and keeps the previous call's contents.  Nothing in it needs
 * clearing (each call rewrites every entry it later reads), but two calls whose kernels can overlap on the GPU -- issued
 * on different streams without an event between them, or from two host threads -- RACE on it and produce garbage
 * gradients; order them on one stream or with events.  The TMA descriptors are re-encoded on the host at every call
 * (there is no plan to cache them).
 * Errors: INVALID_ARG (NULL, non-positive S/P/h_c, bad scale), UNSUPPORTED_SHAPE (D), WORKSPACE_TOO_SMALL, MISALIGNED,
 * UNSUPPORTED_DEVICE, CUDA.
 */
#define HCMS_STATIC_SCRATCH_BYTES (4u << 20)
int hcms_attention_backward_chunk_static(const void* qc, const void* kc, const void* vc, const void* oc, const void* doc,
                                         const void* lse, void* dqc, void* dkc, void* dvc, int64_t S, int P, int h_c,
                                         int D, float scale, void* stream);
/* Device address of the lse the last forward saved on a TRAINING plan: [H][S] fp32 in the order chunk 0's
 * P*h_0 heads (p-major), chunk 1's, ...; NULL otherwise.  For tests. */
void* hcms_plan_lse(const hcms_plan_t* plan);

/* ---- HCMS between P real ranks ---------------------------------------------------- */
/*
 * The paper's actual setting (L45, L59; Alg. 1 lines 8, 21; Table 1 "2 rounds"): P GPUs (one process each, or one
 * process driving several), rank r holding the sequence shard [S/P, H, D] of q, k, v and producing its shard of out.
 * Rank p owns global heads [p*H/P, (p+1)*H/P); head chunks are Eq. 3 on H/P as everywhere else.
 *
 * No library collective is on the data path.  Every rank owns an "exchange block" (its chunk buffers Q'_c, K'_c, V'_c,
 * O'_c, each [S][h_c][D], plus epoch flags) that the other ranks map through CUDA IPC (hcms_dist_export /
 * hcms_dist_attach; between GPUs of a node this is NVLink / NVSwitch peer memory) or, inside one process, through
 * peer access (hcms_dist_attach_local).  Per chunk c the input all-to-all is rank r's scatter kernel STORING its
 * [S/P][h_c][D] slices into every rank's Q'_c, K'_c, V'_c (rows [r*S/P, (r+1)*S/P)), the output all-to-all is rank
 * r's gather kernel LOADING its rows of every rank's O'_c into out[:, p*H/P + o_c + j, :].  E_c^comm and E_c^comp
 * (Eq. 6-7) are 32-bit epoch flags in the consumer's block: written by a one-warp kernel with system-scope
 * release stores after the producing kernel, awaited by the consumer's STREAM (cuStreamWaitValue32) -- no kernel spins
 * on another rank and the host is never blocked.  S_comm runs the pushes of all chunks and then the pulls, S_comp the
 * attention per chunk, exactly Alg. 1's three phases.  The attention kernel is the one of the single-device path, so
 * the concatenated outputs of the P ranks are BIT-EQUAL to hcms_attention_forward on the concatenated inputs.
 *
 * hcms_dist_plan: collective in spirit (every rank creates its own with the same S, H, D, P, C); allocates the
 * exchange block (4*S*(H/P)*D*2 bytes + flags) on the current device.  flags: 0 or any of HCMS_FLAG_ATTN_PAIR, HCMS_FLAG_DIST_FUSE_OUT (the exchange block then also holds this rank's output and 128 pad rows).  bf16 only.
 * There is no graph, profile (HCMS_FLAG_PROFILE), workspace-recycling or training form of the distributed path: those flags are refused.
 * hcms_dist_export: writes HCMS_DIST_HANDLE_BYTES opaque bytes that another PROCESS passes to hcms_dist_attach.
 * hcms_dist_attach: `handles` = P consecutive handles in rank order (this rank's own entry is checked, not opened);
 * the caller moves the bytes between processes with any host channel (torch.distributed, files).
 * hcms_dist_attach_local: the P plans live in this process (peers[r] = rank r's plan, peers[rank] = plan itself).
 * hcms_dist_attention_forward: q, k, v, out = this rank's device shards [S/P, H, D] bf16, 16-byte aligned, out not
 * overlapping the inputs; asynchronous on `stream` like hcms_attention_forward.  EVERY rank must make the call the
 * same number of times (a rank that does not leaves the others' streams waiting).
 * hcms_dist_attention_forward_group: the call for ranks that live in ONE process (attached with
 * hcms_dist_attach_local): plans[r], q[r], k[r], v[r], out[r], streams[r] for r < n = P, in rank order, DISTINCT caller
 * streams.  It enqueues phase by phase over all ranks (all pushes, then all attention, then all pulls), so that every
 * flag a stream waits on is produced by work already enqueued: a stream blocked on a flag holds its hardware work
 * queue, and a rank-by-rank enqueue could park rank 1's pushes behind rank 0's wait on a shared queue (measured: it
 * deadlocks).  hcms_dist_attention_forward therefore rejects locally attached plans (INVALID_ARG); one process per
 * rank -- the deployment the paper describes -- has no such constraint.  Switches to each plan's device for its part.
 * All ranks must have finished (a host barrier after synchronising the streams) before any plan is destroyed.
 * hcms_dist_layer_forward[_group]: the whole layer (Alg. 1 lines 2-27) between the ranks with BOTH all-to-alls inside
 * compute kernels; the plan must carry HCMS_FLAG_DIST_FUSE_OUT.  x = this rank's tokens [S/P, Dm] bf16, w_qkv [3*H*D, Dm]
 * and w_o [Dm, H*D] as in hcms_layer_forward (every rank holds the whole weights), rope_cos / rope_sin = this rank's
 * rows [S/P, D/2] fp32 or both NULL, y = [S/P, Dm].  The QKV projection's epilogue (RoPE, one rounding to bf16) TMA-stores
 * each 128 x 64 panel of q, k, v into the chunk buffer of the rank that owns its head (input all-to-all, peer memory); the
 * attention epilogue stores into the destination ranks' outputs (output all-to-all); the output projection reads the
 * assembled [S/P, H*D] output in place.  C + 2 kernels and 2C signals per rank.  The concatenated y of the P ranks is
 * BIT-EQUAL to hcms_layer_forward on the concatenated x.  Needs 3*C*P <= 96, H/P <= 64, Dm and H*D multiples of 128.
 * Failure of a forward call.  Every check that can refuse a call (NULLs, alignment, aliasing, shape, the plan's device being
 * current, a poisoned plan) runs before anything is enqueued and before the rank takes its next epoch: such an error leaves
 * the rank in step with its peers and the call may simply be repeated correctly.  A failure AFTER that point (a CUDA launch or
 * stream operation failing) stops the data path at once, still joins S_comm / S_comp back into the caller's stream -- so the
 * caller's stream and hcms_dist_plan_destroy never wait on a flag nobody will publish -- and POISONS the plan (for the group
 * calls: all n plans): this rank's epoch was consumed while its peers may never see its flags.  Every later forward call on a
 * poisoned plan returns INVALID_ARG.  The peers of a failed rank are not rescued: their streams keep waiting for its flags, as
 * with any collective one member of which died; tear the job down (destroying a plan whose streams are blocked blocks too).
 * Errors: INVALID_ARG, UNSUPPORTED_SHAPE (also P > 16), UNSUPPORTED_DTYPE, UNSUPPORTED_DEVICE, PLAN_MISMATCH (handle of
 * another shape / rank order, wrong device), MISALIGNED, ALIAS, CUDA.
 */
typedef struct hcms_dist_plan hcms_dist_plan_t;
#define HCMS_DIST_HANDLE_BYTES 128
int hcms_dist_plan(hcms_dist_plan_t** plan, int64_t S, int H, int D, int P, int C, int dtype, uint32_t flags, int rank);
int hcms_dist_plan_destroy(hcms_dist_plan_t* plan); /* synchronises the plan's streams, unmaps the peers; NULL is a no-op */
int hcms_dist_export(hcms_dist_plan_t* plan, void* handle);
int hcms_dist_attach(hcms_dist_plan_t* plan, const void* handles, int n);
int hcms_dist_attach_local(hcms_dist_plan_t* plan, hcms_dist_plan_t* const* peers, int n);
int hcms_dist_attention_forward(hcms_dist_plan_t* plan, const void* q, const void* k, const void* v, void* out,
                                float scale, void* stream);
/* The same call with HOST shards (q, k, v, out: host pointers, bf16 [S/P, H, D]; pinned memory makes the copies asynchronous):
 * H2D copies of the three input shards into plan-owned device staging (4 * S/P*H*D*2 bytes, allocated on first use) on
 * `stream`, hcms_dist_attention_forward on the staging, D2H copy of this rank's output shard, then SYNCHRONISES `stream`.
 * Every rank must make the call like the device form.  Same bits.  Errors: those of hcms_dist_attention_forward. */
int hcms_dist_attention_forward_host(hcms_dist_plan_t* plan, const void* q, const void* k, const void* v, void* out,
                                     float scale, void* stream);
int hcms_dist_attention_forward_group(hcms_dist_plan_t* const* plans, int n, const void* const* q, const void* const* k,
                                      const void* const* v, void* const* out, float scale, void* const* streams);
int hcms_dist_layer_forward(hcms_dist_plan_t* plan, const void* x, const void* w_qkv, const void* w_o, const void* rope_cos,
                            const void* rope_sin, void* y, int Dm, float scale, void* stream);
int hcms_dist_layer_forward_group(hcms_dist_plan_t* const* plans, int n, const void* const* x, const void* w_qkv,
                                  const void* w_o, const void* const* rope_cos, const void* const* rope_sin, void* const* y,
                                  int Dm, float scale, void* const* streams);
/* Bytes of the rank's exchange block; kernels + signal launches of the last forward (C pushes + C attention + C pulls
 * + 2C signals).  0 for a NULL plan. */
size_t hcms_dist_block_bytes(const hcms_dist_plan_t* plan);
int hcms_dist_last_launch_count(const hcms_dist_plan_t* plan);

#ifdef __cplusplus
}
#endif
#endif /* HCMS_H_ */
