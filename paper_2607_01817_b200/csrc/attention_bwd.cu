// Backward of the non-causal bf16 attention of one HCMS head chunk on sm_100a (tcgen05 / TMEM / TMA).
//
// PAPER.md L304 / Table 15 (L479-483): HCMS runs under autograd for forward+backward; L346 names the backward
// as the extension.  The gradient of Eq. 2 (L76) per head, with P = softmax(scale Q K^T), dO = dL/dO:
//     dV = P^T dO            dP = dO V^T            delta_i = dO_i . O_i
//     dS = P o (dP - delta)  dQ = scale dS K        dK = scale dS^T Q
// P is recomputed from the saved row statistic lse_i = log sum_k exp(scale q_i . k_k) (no S x S tensor is kept).
//
// Two deterministic passes (no atomics, so the gradients are bitwise independent of the chunking, like the
// forward: Table 14), both instances of ONE kernel template:
//   kDQ = false  "dK/dV pass": a CTA owns 128 keys (R1 = K_j, R2 = V_j resident) and streams 32-query tiles
//                (X = Q_t, Y = dO_t):  T1 = K_j Q_t^T = S^T, T2 = V_j dO_t^T = dP^T  (M = 128 keys, N = 32 queries);
//                P^T = exp2(T1*c - lse2[col]), dS^T = P^T o (T2 - delta[col]);  dV += P^T dO_t,  dK += dS^T Q_t.
//   kDQ = true   "dQ pass": a CTA owns 128 queries (R1 = Q_i, R2 = dO_i resident) and streams 64-key tiles
//                (X = K_t, Y = V_t):  T1 = Q_i K_t^T = S, T2 = dO_i V_t^T = dP  (M = 128 queries, N = 64 keys);
//                dS = exp2(T1*c - lse2[row]) o (T2 - delta[row]);  dQ += dS K_t.
// Computing the TRANSPOSED scores in the dK/dV pass makes every A operand K-major and every accumulating B
// operand MN-major, the two descriptor forms the forward kernel already uses (QK^T and PV).
//
// One CTA = 384 threads: warp 0 TMA producer, warp 1 MMA issuer, warp 2 TMEM allocator, warps 4-7 / 8-11 two
// softmax warpgroups that take the streamed tiles alternately (tile t -> warpgroup t & 1), each with its own
// T1/T2 columns in TMEM.  P and dS are written back INTO those columns as packed bf16 and feed the accumulating
// MMAs as TMEM A operands (tcgen05.mma with A in TMEM): the kernel is bound by shared-memory operand traffic
// (ncu: tensor queue always full at 52 % pipe activity with P/dS staged in shared memory), and this removes the
// P/dS stores and their re-reads from it.  The RESIDENT operands (K_j, V_j / Q_i, dO_i) are copied into TMEM once per
// CTA as well, so every T1 / T2 MMA reads only the streamed tile from shared memory.  In the dK/dV pass that is what
// fits 512 columns only with 32-query tiles: T1[2], T2[2] 4 x 32 + K_j, V_j 2 x D/2 + dV, dK 2 x D (round 1 used
// 64-query tiles with K_j, V_j as shared-memory operands: the shared-memory pipe was 100 % busy at 71 % tensor activity).
// TMEM columns: T1[2] at 0, T2[2] at 2*kC, R1 at 4*kC, R2 at 4*kC + D/2, accumulators at 4*kC + D.
#include <cuda_bf16.h>

#include "hcms_internal.h"
#include "ptx.cuh"

namespace hcms {
using namespace ptx;

namespace {

constexpr int kRows = 128;        // resident rows per CTA (UMMA M)
constexpr int kPad = 64;          // the packed statistics are padded to a multiple of this many rows
constexpr int kThreads = 384;
constexpr int kTmemCols = 512;

// kCols = streamed rows per iteration (UMMA N of T1/T2, K extent of the accumulating GEMMs): 32 in the dK/dV pass,
// 64 in the dQ pass
template <int D, bool kDQ>
struct Cfg {
  static constexpr int kCols = kDQ ? 64 : 32;
  static constexpr int kPanels = D / 64;
  static constexpr int kResBytes = kPanels * kRows * 128;      // one resident tile
  static constexpr int kStrPanelBytes = kCols * 128;           // one 64-element-wide panel of a streamed tile
  static constexpr int kStrBytes = kPanels * kStrPanelBytes;   // one streamed tile
  static constexpr int kStageBytes = 2 * kStrBytes;            // X_t and Y_t
  static constexpr int kStages = (D == 128 ? 5 : 8) * (64 / kCols);
  static constexpr int kSmemBytes = 2 * kResBytes + kStages * kStageBytes + 1024 + 512;
  static constexpr int kTmemT1 = 0, kTmemT2 = 2 * kCols;
  static constexpr int kTmemR1 = 4 * kCols, kTmemR2 = 4 * kCols + D / 2;   // resident operands as packed bf16 (D/2 columns each)
  static constexpr int kTmemAcc = 4 * kCols + D;
  static_assert(kTmemAcc + (kDQ ? D : 2 * D) <= kTmemCols, "TMEM budget");
};

struct alignas(64) BwdMaps {
  CUtensorMap r1, r2;     // resident operands, box {64, 1, 128, 1} over {D, h_c, S, P}
  CUtensorMap x, y;       // streamed operands, box {64, 1, kCols, 1}
  CUtensorMap out1, out2; // dV, dK (dK/dV pass) or dQ, unused (dQ pass); box {64, 1, 128, 1}
};

struct BwdParams {
  int S;
  int n_iter;             // s_pad / kCols
  int h_c;
  int s_pad;              // row pitch of `stats` (multiple of 64, >= S)
  float scale;
  float scale_log2;
  const float2* stats;    // [P*h_c][s_pad]: {lse * log2(e), delta}; rows >= S hold {+inf, 0}
};

__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ void ld_shared_v4(uint32_t addr, uint32_t& a, uint32_t& b, uint32_t& c, uint32_t& d) {
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(a), "=r"(b), "=r"(c), "=r"(d) : "r"(addr) : "memory");
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

template <int D, bool kDQ>
__global__ void __launch_bounds__(kThreads, 1)
attention_bwd_kernel(const __grid_constant__ BwdMaps maps, const BwdParams prm) {
  using C = Cfg<D, kDQ>;
  constexpr int kStages = C::kStages;
  constexpr int kCols = C::kCols;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t r1_smem = smem_base;
  const uint32_t r2_smem = r1_smem + C::kResBytes;
  const uint32_t ring = r2_smem + C::kResBytes;                      // kStages x (X_t, Y_t)
  const uint32_t bar_base = ring + kStages * C::kStageBytes;
  const uint32_t bar_r_full = bar_base;                      // TMA -> MMA: resident tiles
  const uint32_t bar_x_full = bar_r_full + 8;                // [kStages] TMA -> MMA
  const uint32_t bar_x_empty = bar_x_full + 8 * kStages;     // [kStages] MMA -> TMA
  const uint32_t bar_t_full = bar_x_empty + 8 * kStages;     // [2] MMA -> warpgroup: T1, T2 of its tile are in TMEM
  const uint32_t bar_pd_full = bar_t_full + 16;              // [2] warpgroup -> MMA: P / dS of its tile are in TMEM
  const uint32_t bar_done = bar_pd_full + 16;                // MMA -> all: every accumulation has completed
  const uint32_t bar_rt_full = bar_done + 8;                 // warpgroups -> MMA: the resident tiles are copied into TMEM
  const uint32_t tmem_slot = bar_rt_full + 8;

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
  const int lane = threadIdx.x & 31;
  const int head = blockIdx.y;                 // p*h_c + j
  const int rank = head / prm.h_c;
  const int hj = head - rank * prm.h_c;
  const int row0 = blockIdx.x * kRows;         // first resident row (key in the dK/dV pass, query in the dQ pass)
  const int n_iter = prm.n_iter;

  if (threadIdx.x == 0) {
    mbar_init(bar_r_full, 1);
    mbar_init(bar_done, 1);
    mbar_init(bar_rt_full, 8);            // one elected lane per softmax warp
    for (int s = 0; s < kStages; ++s) {
      mbar_init(bar_x_full + 8 * s, 1);
      mbar_init(bar_x_empty + 8 * s, 1);
    }
    for (int g = 0; g < 2; ++g) {
      mbar_init(bar_t_full + 8 * g, 1);
      mbar_init(bar_pd_full + 8 * g, 4);    // one elected lane per warp of the warpgroup
    }
    fence_mbar_init();
    fence_proxy_async_smem();
  }
  if (warp == 2) {
    tmem_alloc(tmem_slot, kTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  if (warp < 4) {
    setmaxnreg_dec<56>();
    if (warp == 0) {
      // ---------------- TMA producer ----------------
      const bool leader = elect_one();
      if (leader) {
        prefetch_tensormap(&maps.r1);
        prefetch_tensormap(&maps.r2);
        prefetch_tensormap(&maps.x);
        prefetch_tensormap(&maps.y);
        mbar_expect_tx(bar_r_full, 2 * C::kResBytes);
#pragma unroll
        for (int pn = 0; pn < C::kPanels; ++pn) {
          tma_load_4d(r1_smem + pn * kRows * 128, &maps.r1, bar_r_full, pn * 64, hj, row0, rank);
          tma_load_4d(r2_smem + pn * kRows * 128, &maps.r2, bar_r_full, pn * 64, hj, row0, rank);
        }
      }
      __syncwarp();
      int stage = 0;
      uint32_t phase = 0;
      for (int t = 0; t < n_iter; ++t) {
        mbar_wait(bar_x_empty + 8 * stage, phase ^ 1);
        if (leader) {
          const uint32_t dst = ring + stage * C::kStageBytes;
          mbar_expect_tx(bar_x_full + 8 * stage, C::kStageBytes);
#pragma unroll
          for (int pn = 0; pn < C::kPanels; ++pn) {
            tma_load_4d(dst + pn * C::kStrPanelBytes, &maps.x, bar_x_full + 8 * stage, pn * 64, hj, t * kCols, rank);
            tma_load_4d(dst + C::kStrBytes + pn * C::kStrPanelBytes, &maps.y, bar_x_full + 8 * stage, pn * 64, hj,
                        t * kCols, rank);
          }
        }
        __syncwarp();
        if (++stage == kStages) {
          stage = 0;
          phase ^= 1;
        }
      }
    } else if (warp == 1) {
      // ---------------- MMA issuer ----------------
      const bool leader = elect_one();
      constexpr uint32_t idesc_t = umma_idesc_bf16(kRows, kCols, false, false);   // T = R X^T, both K-major
      constexpr uint32_t idesc_acc = umma_idesc_bf16(kRows, D, false, true);      // acc += PD * X, B MN-major
      constexpr uint32_t hi = umma_desc_hi(1024);
      // T1 = R1 X^T and T2 = R2 Y^T of one streamed tile into TMEM buffer b
      auto issue_t = [&](int b, uint32_t stage_addr) {
        const uint32_t x_lo = umma_desc_lo(stage_addr, 16), y_lo = umma_desc_lo(stage_addr + C::kStrBytes, 16);
#pragma unroll
        for (int ks = 0; ks < D / 16; ++ks) {
          const uint32_t s_off = ((ks >> 2) * C::kStrPanelBytes + (ks & 3) * 32) >> 4;
          // A = the resident operand from TMEM: it costs no shared-memory bandwidth
          mma_ts(tmem_base + C::kTmemT1 + b * kCols, tmem_base + C::kTmemR1 + ks * 8,
                 (static_cast<uint64_t>(hi) << 32) | (x_lo + s_off), idesc_t, ks > 0 ? 1u : 0u);
        }
#pragma unroll
        for (int ks = 0; ks < D / 16; ++ks) {
          const uint32_t s_off = ((ks >> 2) * C::kStrPanelBytes + (ks & 3) * 32) >> 4;
          mma_ts(tmem_base + C::kTmemT2 + b * kCols, tmem_base + C::kTmemR2 + ks * 8,
                 (static_cast<uint64_t>(hi) << 32) | (y_lo + s_off), idesc_t, ks > 0 ? 1u : 0u);
        }
      };
      // acc[128 x D] += PD[128 x kCols] * B[kCols x D]: A = P or dS as packed bf16 in TMEM (8 columns per K step of 16),
      // B MN-major in shared memory: 64-wide D panels kStrPanelBytes apart (LBO), 8-row groups 1024 B apart (SBO),
      // 16 rows (one K step) = 2048 B
      auto issue_acc = [&](uint32_t d_tmem, uint32_t a_tmem, uint32_t b_tile, bool accumulate) {
#pragma unroll
        for (int ks = 0; ks < kCols / 16; ++ks) {
          const uint64_t b_desc = (static_cast<uint64_t>(hi) << 32) | (umma_desc_lo(b_tile, C::kStrPanelBytes) + ks * (2048 >> 4));
          mma_ts(d_tmem, a_tmem + ks * 8, b_desc, idesc_acc, (accumulate || ks > 0) ? 1u : 0u);
        }
      };
      mbar_wait(bar_r_full, 0);
      mbar_wait(bar_rt_full, 0);
      tc_fence_after();
      // ring bookkeeping: tile t lives in stage t % kStages, its full-barrier phase is (t / kStages) & 1
      auto wait_tile = [&](int t) -> uint32_t {
        const int s = t % kStages;
        mbar_wait(bar_x_full + 8 * s, (t / kStages) & 1);
        tc_fence_after();
        return ring + s * C::kStageBytes;
      };
      for (int t = 0; t < 2 && t < n_iter; ++t) {
        const uint32_t addr = wait_tile(t);
        if (leader) {
          issue_t(t, addr);
          tc_commit(bar_t_full + 8 * t);
        }
        __syncwarp();
      }
      for (int t = 0; t < n_iter; ++t) {
        const int b = t & 1;
        const uint32_t addr = ring + (t % kStages) * C::kStageBytes;
        mbar_wait(bar_pd_full + 8 * b, (t >> 1) & 1);     // P / dS of tile t sit in the columns of T1/T2[b]
        tc_fence_after();
        if (leader) {
          const uint32_t p_tmem = tmem_base + C::kTmemT1 + b * kCols, ds_tmem = tmem_base + C::kTmemT2 + b * kCols;
          if (kDQ) {
            issue_acc(tmem_base + C::kTmemAcc, ds_tmem, addr, t > 0);                        // dQ += dS K_t
          } else {
            issue_acc(tmem_base + C::kTmemAcc, p_tmem, addr + C::kStrBytes, t > 0);          // dV += P^T dO_t
            issue_acc(tmem_base + C::kTmemAcc + D, ds_tmem, addr, t > 0);                    // dK += dS^T Q_t
          }
          tc_commit(bar_x_empty + 8 * (t % kStages));
          if (t == n_iter - 1) tc_commit(bar_done);
        }
        __syncwarp();
        // T1/T2 of tile t+2 overwrite buffer b: issued after the accumulations that read P / dS from it (the
        // tensor pipe executes one thread's MMAs in issue order)
        if (t + 2 < n_iter) {
          const uint32_t next = wait_tile(t + 2);
          if (leader) {
            issue_t(b, next);
            tc_commit(bar_t_full + 8 * b);
          }
          __syncwarp();
        }
      }
    }
    __syncwarp();
  } else {
    // ================================ softmax warpgroups ================================
    setmaxnreg_inc<224>();
    const int g = (warp >> 2) - 1;                       // warpgroup: tiles t = g, g+2, ...
    const int row = (warp & 3) * 32 + lane;              // resident row == TMEM lane
    const uint32_t lane_addr = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t t1_tmem = tmem_base + lane_addr + C::kTmemT1 + g * kCols;
    const uint32_t t2_tmem = tmem_base + lane_addr + C::kTmemT2 + g * kCols;
    const uint32_t swz = static_cast<uint32_t>(row & 7);
    const float scale_log2 = prm.scale_log2;
    const float2* stats = prm.stats + static_cast<size_t>(head) * prm.s_pad;
    float row_lse2 = 0.f, row_delta = 0.f;
    if (kDQ) {
      const int r = min(row0 + row, prm.s_pad - 1);
      const float2 st = __ldg(stats + r);                // rows >= S: {+inf, 0} -> P = 0 (never stored anyway)
      row_lse2 = st.x;
      row_delta = st.y;
    }

    {
      // warpgroup 0 copies R1 (Q_i / K_j), warpgroup 1 R2 (dO_i / V_j) from the swizzled shared-memory tile into TMEM
      // (row = lane, column c = elements 2c, 2c+1): the A operand of every T1 / T2 MMA of this CTA
      mbar_wait(bar_r_full, 0);
      const uint32_t src = (g == 0 ? r1_smem : r2_smem) + row * 128;
      const uint32_t dst = tmem_base + lane_addr + (g == 0 ? C::kTmemR1 : C::kTmemR2);
#pragma unroll
      for (int pn = 0; pn < C::kPanels; ++pn) {
        uint32_t w[32];
#pragma unroll
        for (int ch = 0; ch < 8; ++ch)
          ld_shared_v4(src + pn * (kRows * 128) + ((static_cast<uint32_t>(ch) ^ swz) << 4), w[ch * 4], w[ch * 4 + 1],
                       w[ch * 4 + 2], w[ch * 4 + 3]);
        tmem_st32(dst + pn * 32, w);
      }
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_rt_full);
    }

    for (int t = g, k = 0; t < n_iter; t += 2, ++k) {
      mbar_wait(bar_t_full + 8 * g, k & 1);
      tc_fence_after();
      uint32_t s[kCols], dp[kCols];
#pragma unroll
      for (int c4 = 0; c4 < kCols / 32; ++c4) tmem_ld32(t1_tmem + c4 * 32, &s[c4 * 32]);
#pragma unroll
      for (int c4 = 0; c4 < kCols / 32; ++c4) tmem_ld32(t2_tmem + c4 * 32, &dp[c4 * 32]);
      tmem_wait_ld();
      const int valid = prm.S - t * kCols;                        // streamed rows of this tile that exist (dQ pass mask)
      // P and dS go back into the first 32 columns of T1 / T2 as packed bf16 (element 2c in the low half): the
      // accumulating MMAs read their A operand from TMEM, so neither costs shared-memory bandwidth
      uint32_t pw[kCols / 2], dw[kCols / 2];
#pragma unroll
      for (int ch = 0; ch < kCols / 8; ++ch) {
#pragma unroll
        for (int pr = 0; pr < 4; ++pr) {
          const int c = ch * 8 + pr * 2;
          float l0, d0, l1, d1;
          if (kDQ) {
            l0 = l1 = row_lse2;
            d0 = d1 = row_delta;
          } else {
            const float4 st = __ldg(reinterpret_cast<const float4*>(stats + t * kCols + c));   // warp-uniform address
            l0 = st.x; d0 = st.y; l1 = st.z; d1 = st.w;
          }
          float p0 = ex2(fmaf(__uint_as_float(s[c]), scale_log2, -l0));
          float p1 = ex2(fmaf(__uint_as_float(s[c + 1]), scale_log2, -l1));
          if (kDQ) {                       // keys beyond S do not exist (their K rows are TMA zero fill)
            if (c >= valid) p0 = 0.f;
            if (c + 1 >= valid) p1 = 0.f;
          }
          const float e0 = p0 * (__uint_as_float(dp[c]) - d0);
          const float e1 = p1 * (__uint_as_float(dp[c + 1]) - d1);
          if (!kDQ) pw[ch * 4 + pr] = pack_bf16(p0, p1);
          dw[ch * 4 + pr] = pack_bf16(e0, e1);
        }
      }
      // kCols / 2 packed columns each
      if constexpr (kCols == 64) {
        if (!kDQ) tmem_st32(t1_tmem, pw);
        tmem_st32(t2_tmem, dw);
      } else {
        if (!kDQ) tmem_st16(t1_tmem, pw);
        tmem_st16(t2_tmem, dw);
      }
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_pd_full + 8 * g);
    }

    // ---------------- epilogue ----------------
    mbar_wait(bar_done, 0);
    tc_fence_after();
    if (kDQ) {
      // dQ = scale * acc: warpgroup g converts columns [g*D/2, (g+1)*D/2) into R1's space (Q_i is dead), one TMA store
#pragma unroll
      for (int c4 = g * (D / 64); c4 < (g + 1) * (D / 64); ++c4) {
        uint32_t r[32];
        tmem_ld32(tmem_base + lane_addr + C::kTmemAcc + c4 * 32, r);
        tmem_wait_ld();
#pragma unroll
        for (int q4 = 0; q4 < 4; ++q4) {
          uint32_t w[4];
#pragma unroll
          for (int e = 0; e < 4; ++e)
            w[e] = pack_bf16(__uint_as_float(r[q4 * 8 + 2 * e]) * prm.scale, __uint_as_float(r[q4 * 8 + 2 * e + 1]) * prm.scale);
          const uint32_t chunk = (c4 & 1) * 4 + q4;
          st_shared_v4(r1_smem + (c4 >> 1) * (kRows * 128) + row * 128 + ((chunk ^ swz) << 4), w[0], w[1], w[2], w[3]);
        }
      }
      fence_proxy_async_smem();
      named_bar_sync(1, 256);
      if (threadIdx.x == 128 && row0 < prm.S) {
#pragma unroll
        for (int pn = 0; pn < C::kPanels; ++pn)
          tma_store_4d(&maps.out1, r1_smem + pn * (kRows * 128), pn * 64, hj, row0, rank);
        bulk_commit();
        bulk_wait<0>();
      }
    } else {
      // warpgroup 0: dV = acc1 -> R1's space; warpgroup 1: dK = scale * acc2 -> R2's space (K_j, V_j are dead)
      const float mul = g == 0 ? 1.0f : prm.scale;
      const uint32_t stage = g == 0 ? r1_smem : r2_smem;
#pragma unroll
      for (int c4 = 0; c4 < D / 32; ++c4) {
        uint32_t r[32];
        tmem_ld32(tmem_base + lane_addr + C::kTmemAcc + g * D + c4 * 32, r);
        tmem_wait_ld();
#pragma unroll
        for (int q4 = 0; q4 < 4; ++q4) {
          uint32_t w[4];
#pragma unroll
          for (int e = 0; e < 4; ++e)
            w[e] = pack_bf16(__uint_as_float(r[q4 * 8 + 2 * e]) * mul, __uint_as_float(r[q4 * 8 + 2 * e + 1]) * mul);
          const uint32_t chunk = (c4 & 1) * 4 + q4;
          st_shared_v4(stage + (c4 >> 1) * (kRows * 128) + row * 128 + ((chunk ^ swz) << 4), w[0], w[1], w[2], w[3]);
        }
      }
      fence_proxy_async_smem();
      named_bar_sync(1 + g, 128);
      if ((warp & 3) == 0 && lane == 0 && row0 < prm.S) {
        const CUtensorMap* om = g == 0 ? &maps.out1 : &maps.out2;
#pragma unroll
        for (int pn = 0; pn < C::kPanels; ++pn) tma_store_4d(om, stage + pn * (kRows * 128), pn * 64, hj, row0, rank);
        bulk_commit();
        bulk_wait<0>();
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem_base, kTmemCols);
}

// delta_i = dO_i . O_i and lse_i * log2(e) for every (head, row) of a chunk, packed for the two passes; the
// padding rows [S, s_pad) of every head get {+inf, 0} so that a query that does not exist has P = 0.
// o, dO: [P][S][h_c][D] bf16; lse: [P*h_c][S] fp32 (natural log, as the forward wrote it); stats: [P*h_c][s_pad].
template <int D>
__global__ void __launch_bounds__(256)
attention_bwd_prep_kernel(const uint4* __restrict__ o, const uint4* __restrict__ d_o, const float* __restrict__ lse,
                          float2* __restrict__ stats, int S, int h_c, int P, int s_pad) {
  constexpr int kLanes = D / 8;                 // lanes per row, 8 bf16 (16 bytes) each
  constexpr int kRowsPerBlock = 256 / kLanes;
  const int64_t n_rows = static_cast<int64_t>(P) * S * h_c;
  const int64_t L = static_cast<int64_t>(blockIdx.x) * kRowsPerBlock + threadIdx.x / kLanes;   // row in memory order
  const int sub = threadIdx.x % kLanes;
  float acc = 0.f;
  if (L < n_rows) {
    const uint4 a = __ldg(o + L * kLanes + sub), b = __ldg(d_o + L * kLanes + sub);
    const uint32_t aw[4] = {a.x, a.y, a.z, a.w}, bw[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      acc = fmaf(__uint_as_float(aw[e] << 16), __uint_as_float(bw[e] << 16), acc);
      acc = fmaf(__uint_as_float(aw[e] & 0xffff0000u), __uint_as_float(bw[e] & 0xffff0000u), acc);
    }
  }
#pragma unroll
  for (int m = kLanes / 2; m > 0; m >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, m);
  if (L < n_rows && sub == 0) {
    const int j = static_cast<int>(L % h_c);
    const int64_t ps = L / h_c;
    const int s = static_cast<int>(ps % S);
    const int head = static_cast<int>(ps / S) * h_c + j;
    stats[static_cast<size_t>(head) * s_pad + s] =
        make_float2(lse[static_cast<size_t>(head) * S + s] * 1.4426950408889634f, acc);
  }
  if (blockIdx.x == 0) {
    const int pad = s_pad - S;
    for (int i = threadIdx.x; i < P * h_c * pad; i += 256)
      stats[static_cast<size_t>(i / pad) * s_pad + S + i % pad] = make_float2(INFINITY, 0.f);
  }
}

cudaError_t map4d(CUtensorMap* m, const void* base, const AttnBwdArgs& a, uint32_t box_rows) {
  const uint64_t dims[4] = {static_cast<uint64_t>(a.D), static_cast<uint64_t>(a.h_c), static_cast<uint64_t>(a.S),
                            static_cast<uint64_t>(a.P)};
  const uint64_t strides[3] = {static_cast<uint64_t>(a.D) * 2, static_cast<uint64_t>(a.h_c) * a.D * 2,
                               static_cast<uint64_t>(a.S) * a.h_c * a.D * 2};
  const uint32_t box[4] = {64, 1, box_rows, 1};
  return encode_tensor_map(a.cache, m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, base, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
}

template <int D>
cudaError_t launch(const AttnBwdArgs& a, cudaStream_t stream) {
  const int heads = a.P * a.h_c;
  const int s_pad = static_cast<int>((a.S + kPad - 1) / kPad * kPad);
  float2* stats = static_cast<float2*>(a.stats);
  {
    constexpr int kRowsPerBlock = 256 / (D / 8);
    const int64_t n_rows = static_cast<int64_t>(heads) * a.S;
    const unsigned blocks = static_cast<unsigned>((n_rows + kRowsPerBlock - 1) / kRowsPerBlock);
    attention_bwd_prep_kernel<D><<<blocks, 256, 0, stream>>>(static_cast<const uint4*>(a.o), static_cast<const uint4*>(a.d_o),
                                                             a.lse, stats, static_cast<int>(a.S), a.h_c, a.P, s_pad);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  if (D == 128 && a.dq_acc && a.dq_turn) return launch_attention_bwd_1pass(a, stats, s_pad, stream);
  BwdParams prm;
  prm.S = static_cast<int>(a.S);
  prm.h_c = a.h_c;
  prm.s_pad = s_pad;
  prm.scale = a.scale;
  prm.scale_log2 = fmaxf(a.scale * 1.4426950408889634f, 1e-30f);
  prm.stats = stats;
  const dim3 grid(static_cast<unsigned>((a.S + kRows - 1) / kRows), static_cast<unsigned>(heads));
  cudaError_t e;
  BwdMaps kv;   // dK/dV pass: R = K, V; streamed Q, dO; out dV, dK
  constexpr int kColsKV = Cfg<D, false>::kCols, kColsQ = Cfg<D, true>::kCols;
  if ((e = map4d(&kv.r1, a.k, a, kRows)) != cudaSuccess) return e;
  if ((e = map4d(&kv.r2, a.v, a, kRows)) != cudaSuccess) return e;
  if ((e = map4d(&kv.x, a.q, a, kColsKV)) != cudaSuccess) return e;
  if ((e = map4d(&kv.y, a.d_o, a, kColsKV)) != cudaSuccess) return e;
  if ((e = map4d(&kv.out1, a.dv, a, kRows)) != cudaSuccess) return e;
  if ((e = map4d(&kv.out2, a.dk, a, kRows)) != cudaSuccess) return e;
  prm.n_iter = s_pad / kColsKV;
  attention_bwd_kernel<D, false><<<grid, kThreads, Cfg<D, false>::kSmemBytes, stream>>>(kv, prm);
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  BwdMaps qm;   // dQ pass: R = Q, dO; streamed K, V; out dQ
  if ((e = map4d(&qm.r1, a.q, a, kRows)) != cudaSuccess) return e;
  if ((e = map4d(&qm.r2, a.d_o, a, kRows)) != cudaSuccess) return e;
  if ((e = map4d(&qm.x, a.k, a, kColsQ)) != cudaSuccess) return e;
  if ((e = map4d(&qm.y, a.v, a, kColsQ)) != cudaSuccess) return e;
  if ((e = map4d(&qm.out1, a.dq, a, kRows)) != cudaSuccess) return e;
  qm.out2 = qm.out1;
  prm.n_iter = s_pad / kColsQ;
  attention_bwd_kernel<D, true><<<grid, kThreads, Cfg<D, true>::kSmemBytes, stream>>>(qm, prm);
  return cudaGetLastError();
}

}  // namespace

static cudaError_t bwd_set_attributes() {
  cudaError_t e;
#define HCMS_SET(fn, bytes) \
  if ((e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes)) != cudaSuccess) return e;
  HCMS_SET((attention_bwd_kernel<128, false>), (Cfg<128, false>::kSmemBytes))
  HCMS_SET((attention_bwd_kernel<128, true>), (Cfg<128, true>::kSmemBytes))
  HCMS_SET((attention_bwd_kernel<64, false>), (Cfg<64, false>::kSmemBytes))
  HCMS_SET((attention_bwd_kernel<64, true>), (Cfg<64, true>::kSmemBytes))
#undef HCMS_SET
  return cudaSuccess;
}

cudaError_t attention_bwd_init() {
  static PerDeviceOnce once;
  return once_per_device(&once, bwd_set_attributes);
}

size_t attention_bwd_stats_bytes(int64_t S, int heads) {
  const int64_t s_pad = (S + kPad - 1) / kPad * kPad;
  return static_cast<size_t>(heads) * s_pad * sizeof(float2);
}

// Three launches: delta/lse packing, the dK/dV pass, the dQ pass.
cudaError_t launch_attention_bwd(const AttnBwdArgs& a, cudaStream_t stream) {
  if (a.D == 128) return launch<128>(a, stream);
  if (a.D == 64) return launch<64>(a, stream);
  return cudaErrorInvalidValue;
}

}  // namespace hcms
