// Single-pass backward of the non-causal bf16 attention of one HCMS head chunk on sm_100a, D = 128 (tcgen05 / TMEM / TMA).
//
// PAPER.md L304 / Table 15 (L479-483), L346: forward + backward under HCMS.  attention_bwd.cu computes the gradient of
// Eq. 2 (L76) in two passes (a dK/dV pass and a dQ pass: 7 contractions for 5 algorithmic ones, because S = QK^T and
// dP = dO V^T are formed in both).  This kernel forms them once: a CTA owns 128 keys of one head (dK_j, dV_j stay in
// tensor memory), streams 64-query tiles, and sends its partial dQ of every tile to an fp32 accumulator in global memory
// IN A FIXED ORDER over the key tiles, so that the gradients stay bitwise independent of the chunking (Table 14's
// "max error 0", L472-477) and of the run.
//
// Per step t (queries [64 t, 64 t + 64)), with K_j, V_j [128 x D] resident in shared memory:
//     M1  S^T  [128 k x 64 q] = K_j Q_t^T            (SS, both K-major)
//     M2  dP^T [128 k x 64 q] = V_j dO_t^T           (SS)
//         P^T = exp2(S^T c - lse2[q]),  dS^T = P^T o (dP^T - delta[q])              (two softmax warpgroups, alternating steps)
//     M3  dV   [128 k x D]   += P^T  dO_t            (TS: A = P^T as packed bf16 in TMEM, B = dO_t MN-major)
//     M4  dK   [128 k x D]   += dS^T Q_t             (TS)
//     M5  dQ^T [D x 64 q]     = K_j^T dS^T           (SS: A = the SAME K_j tile read MN-major, B = dS^T [128 k x 64 q] MN-major
//                                                     from shared memory, where the softmax warpgroup also put it)
//         dQ_acc[q][d] (+)= dQ^T                     (drain warpgroup: tcgen05.ld, then one coalesced red.global.add.f32 per
//                                                     query row; the CTA of key tile 0 stores, tile j adds after tile j-1)
//
// TMEM (512 columns): S^T 0 | dP^T 64 | dQ^T 128 | P^T 192 (32) | dS^T 224 (32) | dV 256 | dK 384.  S^T, dP^T and dQ^T are
// single buffers handed back and forth (the tensor pipe runs the accumulations of step t-1 while a warpgroup works on
// step t); there is no room for K_j, V_j as TMEM operands (attention_bwd.cu's dK/dV pass), so M1, M2 and M5 read their A
// operand from shared memory (224 KB of operand, TMA and dS traffic per step = 1792 shared-memory-pipe cycles against
// 1280 tensor cycles).
//
// Order of the dQ reduction: one counter per (head, query tile).  The CTA of key tile j waits until the counter equals
// j, issues its 64 x 128 reds (tile 0: stores), and sets the counter to j + 1 one step later, after a fence (by then the
// reds have been performed, so the fence costs its fixed latency only).
// Forward progress: a CTA spins on a counter that another CTA of the same launch advances, so that other CTA must already
// be running.  CUDA does not promise that CTAs start in blockIdx order (another kernel may hold SMs, the two compute
// streams may each have such a grid in flight, MPS, a debugger), so the key tile is NOT blockIdx.x: every CTA draws a
// ticket from a per-head counter when it starts (atomicAdd, zeroed with the turn counters) and works on key tile
// `ticket`.  The CTA of key tile j therefore waits only for CTAs that drew j-1, j-2, ... before it -- CTAs that are
// resident and waiting on nobody newer -- whatever order the hardware starts them in.  The reduction order (ascending
// key tile) and with it every bit of dQ is unchanged.
//
// MEASURED (cfg 3 backward, one B200, profiles/r2k_bwd_one_pass.md): two-pass kernels 59.2-60.0 ms; this kernel without
// any dQ output 48.4 ms (the contraction pipeline alone: the 5-vs-7 saving is real), with unordered reds 60.9 ms, with the
// ordered reduction 82.3 ms (97.9 ms when the fence followed the reds directly).  The 172 GB of fp32 reduction traffic
// per layer (32 KB per step, 19 cycles per red instruction in the LSU, 40 % of L2 throughput) costs what the two
// saved contractions gain, and ordering it costs more.  Hence opt-in (HCMS_FLAG_BWD_ONE_PASS), not the default.
#include <cuda_bf16.h>

#include "hcms_internal.h"
#include "ptx.cuh"

namespace hcms {
using namespace ptx;

namespace {

constexpr int kD = 128;
constexpr int kRows = 128;        // keys per CTA (UMMA M of M1-M4)
constexpr int kQ = 64;            // queries per step (UMMA N of M1, M2, M5; K extent of M3, M4)
constexpr int kThreads = 512;
constexpr int kTmemCols = 512;
constexpr int kPanels = kD / 64;
constexpr int kResBytes = kPanels * kRows * 128;        // K_j or V_j: 32 KB
constexpr int kStrPanelBytes = kQ * 128;                // one 64-wide panel of a streamed tile
constexpr int kStrBytes = kPanels * kStrPanelBytes;     // Q_t or dO_t: 16 KB
constexpr int kStageBytes = 2 * kStrBytes;
constexpr int kStages = 4;
constexpr int kDsBytes = kRows * 128;                   // dS^T: 128 key rows x 64 queries bf16
constexpr int kSmemBytes = 2 * kResBytes + kStages * kStageBytes + 2 * kDsBytes + 1024 + 512;
static_assert(kSmemBytes <= 227 * 1024, "shared memory budget");
constexpr int kTmemT1 = 0, kTmemT2 = 64, kTmemDQ = 128, kTmemP = 192, kTmemDS = 224, kTmemDV = 256, kTmemDK = 384;

struct alignas(64) Bwd1Maps {
  CUtensorMap k, v;       // resident, box {64, 1, 128, 1} over {D, h_c, S, P}
  CUtensorMap q, d_o;     // streamed, box {64, 1, 64, 1}
  CUtensorMap dv, dk;     // outputs, box {64, 1, 128, 1}
};

struct Bwd1Params {
  int S;
  int n_iter;             // s_pad / 64
  int h_c;
  int s_pad;
  float scale;
  float scale_log2;
  const float2* stats;    // [P*h_c][s_pad]: {lse * log2(e), delta}; rows >= S hold {+inf, 0}
  float* dq_acc;          // [P*h_c][s_pad][D] fp32
  int* dq_turn;           // [P*h_c][n_iter], zero before the launch
  int* dq_ticket;         // [P*h_c], zero before the launch: next key tile of the head to hand out
};

__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_gpu(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void red_add_f32(float* p, float v) {
  asm volatile("red.relaxed.gpu.global.add.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory");
}

__global__ void __launch_bounds__(kThreads, 1)
attention_bwd_1pass_kernel(const __grid_constant__ Bwd1Maps maps, const Bwd1Params prm) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t k_smem = smem_base;
  const uint32_t v_smem = k_smem + kResBytes;
  const uint32_t ring = v_smem + kResBytes;                          // kStages x (Q_t, dO_t)
  const uint32_t ds_smem = ring + kStages * kStageBytes;             // 2 x dS^T (one per softmax warpgroup)
  const uint32_t bar_base = ds_smem + 2 * kDsBytes;
  const uint32_t bar_r_full = bar_base;                      // TMA -> MMA: K_j, V_j
  const uint32_t bar_x_full = bar_r_full + 8;                // [kStages] TMA -> MMA
  const uint32_t bar_x_empty = bar_x_full + 8 * kStages;     // [kStages] MMA -> TMA
  // A waiter that sees only every other completion of a barrier cannot tell phases apart by parity, so the barriers the
  // alternating warpgroups wait on exist once per step parity; the MMA warp and the drain see every step.
  const uint32_t bar_t_full = bar_x_empty + 8 * kStages;     // [2] MMA -> warpgroup t & 1: S^T, dP^T of step t are in TMEM
  const uint32_t bar_t_free = bar_t_full + 16;               // warpgroup -> MMA: they are in registers
  const uint32_t bar_pd_full = bar_t_free + 8;               // warpgroup -> MMA: P^T, dS^T (TMEM) and dS^T (shared) of step t
  const uint32_t bar_acc = bar_pd_full + 8;                  // [2] MMA -> warpgroups: M3, M4, M5 of step t have completed
  const uint32_t bar_dq_free = bar_acc + 16;                 // drain -> MMA: dQ^T of step t is in registers
  const uint32_t bar_done = bar_dq_free + 8;                 // MMA -> all: every accumulation has completed
  const uint32_t tmem_slot = bar_done + 8;
  const uint32_t ticket_slot = tmem_slot + 4;

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
  const int lane = threadIdx.x & 31;
  const int head = blockIdx.y;                 // p*h_c + j
  const int rank = head / prm.h_c;
  const int hj = head - rank * prm.h_c;
  const int n_iter = prm.n_iter;

  if (threadIdx.x == 0) {
    // the key tile is the order in which this head's CTAs actually start (see "Forward progress" above)
    const int ticket = atomicAdd(prm.dq_ticket + head, 1);
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(ticket_slot), "r"(ticket) : "memory");
    mbar_init(bar_r_full, 1);
    for (int b = 0; b < 2; ++b) {
      mbar_init(bar_t_full + 8 * b, 1);
      mbar_init(bar_acc + 8 * b, 1);
    }
    mbar_init(bar_t_free, 4);             // one elected lane per warp of the warpgroup that owns the step
    mbar_init(bar_pd_full, 4);
    mbar_init(bar_dq_free, 4);
    mbar_init(bar_done, 1);
    for (int s = 0; s < kStages; ++s) {
      mbar_init(bar_x_full + 8 * s, 1);
      mbar_init(bar_x_empty + 8 * s, 1);
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
  int key_tile;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(key_tile) : "r"(ticket_slot));
  const int row0 = key_tile * kRows;

  if (warp < 4) {
    setmaxnreg_dec<56>();
    if (warp == 0) {
      // ---------------- TMA producer ----------------
      const bool leader = elect_one();
      if (leader) {
        prefetch_tensormap(&maps.k);
        prefetch_tensormap(&maps.v);
        prefetch_tensormap(&maps.q);
        prefetch_tensormap(&maps.d_o);
        mbar_expect_tx(bar_r_full, 2 * kResBytes);
#pragma unroll
        for (int pn = 0; pn < kPanels; ++pn) {
          tma_load_4d(k_smem + pn * kRows * 128, &maps.k, bar_r_full, pn * 64, hj, row0, rank);
          tma_load_4d(v_smem + pn * kRows * 128, &maps.v, bar_r_full, pn * 64, hj, row0, rank);
        }
      }
      __syncwarp();
      int stage = 0;
      uint32_t phase = 0;
      for (int t = 0; t < n_iter; ++t) {
        mbar_wait(bar_x_empty + 8 * stage, phase ^ 1);
        if (leader) {
          const uint32_t dst = ring + stage * kStageBytes;
          mbar_expect_tx(bar_x_full + 8 * stage, kStageBytes);
#pragma unroll
          for (int pn = 0; pn < kPanels; ++pn) {
            tma_load_4d(dst + pn * kStrPanelBytes, &maps.q, bar_x_full + 8 * stage, pn * 64, hj, t * kQ, rank);
            tma_load_4d(dst + kStrBytes + pn * kStrPanelBytes, &maps.d_o, bar_x_full + 8 * stage, pn * 64, hj, t * kQ, rank);
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
      constexpr uint32_t idesc_t = umma_idesc_bf16(kRows, kQ, false, false);    // S^T / dP^T: both operands K-major
      constexpr uint32_t idesc_acc = umma_idesc_bf16(kRows, kD, false, true);   // dV / dK: A in TMEM, B MN-major
      constexpr uint32_t idesc_dq = umma_idesc_bf16(kD, kQ, true, true);        // dQ^T: A = K_j^T and B = dS^T, both MN-major
      constexpr uint32_t hi = umma_desc_hi(1024);
      const uint32_t k_lo = umma_desc_lo(k_smem, 16), v_lo = umma_desc_lo(v_smem, 16);
      const uint32_t kt_lo = umma_desc_lo(k_smem, kRows * 128);        // MN-major: 64-wide d panels 16 KB apart
      // S^T = K_j Q_t^T and dP^T = V_j dO_t^T of one streamed tile
      auto issue_t = [&](uint32_t stage_addr) {
        const uint32_t x_lo = umma_desc_lo(stage_addr, 16), y_lo = umma_desc_lo(stage_addr + kStrBytes, 16);
#pragma unroll
        for (int ks = 0; ks < kD / 16; ++ks) {
          const uint32_t r_off = ((ks >> 2) * (kRows * 128) + (ks & 3) * 32) >> 4;
          const uint32_t s_off = ((ks >> 2) * kStrPanelBytes + (ks & 3) * 32) >> 4;
          mma_ss_lohi(tmem_base + kTmemT1, k_lo + r_off, x_lo + s_off, hi, hi, idesc_t, ks > 0 ? 1u : 0u);
        }
#pragma unroll
        for (int ks = 0; ks < kD / 16; ++ks) {
          const uint32_t r_off = ((ks >> 2) * (kRows * 128) + (ks & 3) * 32) >> 4;
          const uint32_t s_off = ((ks >> 2) * kStrPanelBytes + (ks & 3) * 32) >> 4;
          mma_ss_lohi(tmem_base + kTmemT2, v_lo + r_off, y_lo + s_off, hi, hi, idesc_t, ks > 0 ? 1u : 0u);
        }
      };
      // acc[128 x D] += PD[128 x 64] * B[64 x D]: A packed bf16 in TMEM (8 columns per K step of 16 queries), B MN-major
      auto issue_acc = [&](uint32_t d_tmem, uint32_t a_tmem, uint32_t b_tile, bool accumulate) {
        const uint32_t b_lo = umma_desc_lo(b_tile, kStrPanelBytes);
#pragma unroll
        for (int ks = 0; ks < kQ / 16; ++ks)
          mma_ts_lohi(d_tmem, a_tmem + ks * 8, b_lo + ks * (2048 >> 4), hi, idesc_acc, (accumulate || ks > 0) ? 1u : 0u);
      };
      // dQ^T[D x 64] = K_j^T[D x 128 keys] dS^T[128 keys x 64]: K steps of 16 keys = 2048 B in both tiles
      auto issue_dq = [&](uint32_t ds_tile) {
        const uint32_t b_lo = umma_desc_lo(ds_tile, kDsBytes);
#pragma unroll
        for (int ks = 0; ks < kRows / 16; ++ks)
          mma_ss_lohi(tmem_base + kTmemDQ, kt_lo + ks * (2048 >> 4), b_lo + ks * (2048 >> 4), hi, hi, idesc_dq, ks > 0 ? 1u : 0u);
      };
      auto wait_tile = [&](int t) -> uint32_t {
        const int s = t % kStages;
        mbar_wait(bar_x_full + 8 * s, (t / kStages) & 1);
        return ring + s * kStageBytes;
      };
      mbar_wait(bar_r_full, 0);
      {
        const uint32_t addr = wait_tile(0);
        tc_fence_after();
        if (leader) {
          issue_t(addr);
          tc_commit(bar_t_full);                  // step 0 -> warpgroup 0
        }
        __syncwarp();
      }
      for (int t = 0; t < n_iter; ++t) {
        if (t + 1 < n_iter) {
          // S^T, dP^T of step t+1 overwrite the buffers once the warpgroup of step t has them in registers
          const uint32_t next = wait_tile(t + 1);
          mbar_wait(bar_t_free, t & 1);
          tc_fence_after();
          if (leader) {
            issue_t(next);
            tc_commit(bar_t_full + 8 * ((t + 1) & 1));
          }
          __syncwarp();
        }
        const uint32_t addr = ring + (t % kStages) * kStageBytes;
        mbar_wait(bar_pd_full, t & 1);                          // P^T, dS^T of step t are in place
        if (t >= 1) mbar_wait(bar_dq_free, (t - 1) & 1);        // dQ^T of step t-1 has left its buffer
        tc_fence_after();
        if (leader) {
          issue_acc(tmem_base + kTmemDV, tmem_base + kTmemP, addr + kStrBytes, t > 0);     // dV += P^T dO_t
          issue_acc(tmem_base + kTmemDK, tmem_base + kTmemDS, addr, t > 0);                // dK += dS^T Q_t
          issue_dq(ds_smem + (t & 1) * kDsBytes);                                          // dQ^T = K_j^T dS^T
          tc_commit(bar_acc + 8 * (t & 1));
          tc_commit(bar_x_empty + 8 * (t % kStages));
          if (t == n_iter - 1) tc_commit(bar_done);
        }
        __syncwarp();
      }
    }
    __syncwarp();
  } else if (warp < 12) {
    // ================================ softmax warpgroups (steps t = g, g+2, ...) ================================
    setmaxnreg_inc<176>();
    const int g = (warp >> 2) - 1;
    const int row = (warp & 3) * 32 + lane;              // key row == TMEM lane
    const uint32_t lane_addr = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t t1_tmem = tmem_base + lane_addr + kTmemT1;
    const uint32_t t2_tmem = tmem_base + lane_addr + kTmemT2;
    const uint32_t swz = static_cast<uint32_t>(row & 7);
    const float scale_log2 = prm.scale_log2;
    const float2* stats = prm.stats + static_cast<size_t>(head) * prm.s_pad;
    const uint32_t ds_row = ds_smem + g * kDsBytes + row * 128;

    for (int t = g; t < n_iter; t += 2) {
      mbar_wait(bar_t_full + 8 * g, (t >> 1) & 1);
      tc_fence_after();
      uint32_t pw[kQ / 2], dw[kQ / 2];
#pragma unroll
      for (int h = 0; h < 2; ++h) {                      // two halves of 32 queries: 64 live accumulator registers at a time
        uint32_t s[32], dp[32];
        tmem_ld32(t1_tmem + h * 32, s);
        tmem_ld32(t2_tmem + h * 32, dp);
        tmem_wait_ld();
        if (h == 1) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(bar_t_free);        // the MMA warp may overwrite S^T, dP^T with step t+1
        }
#pragma unroll
        for (int c = 0; c < 32; c += 2) {
          const float4 st = __ldg(reinterpret_cast<const float4*>(stats + t * kQ + h * 32 + c));   // warp-uniform address
          const float p0 = ex2(fmaf(__uint_as_float(s[c]), scale_log2, -st.x));
          const float p1 = ex2(fmaf(__uint_as_float(s[c + 1]), scale_log2, -st.z));
          const float e0 = p0 * (__uint_as_float(dp[c]) - st.y);
          const float e1 = p1 * (__uint_as_float(dp[c + 1]) - st.w);
          pw[h * 16 + c / 2] = pack_bf16(p0, p1);
          dw[h * 16 + c / 2] = pack_bf16(e0, e1);
        }
      }
      // P^T / dS^T columns and this warpgroup's dS^T tile are free once M3, M4, M5 of step t-1 have completed
      if (t >= 1) {
        mbar_wait(bar_acc + 8 * ((t - 1) & 1), ((t - 1) >> 1) & 1);
        tc_fence_after();
      }
      tmem_st32(tmem_base + lane_addr + kTmemP, pw);
      tmem_st32(tmem_base + lane_addr + kTmemDS, dw);
#pragma unroll
      for (int ch = 0; ch < 8; ++ch)                      // row `row` of dS^T: 64 queries = 8 chunks of 16 B, 128-byte swizzle
        st_shared_v4(ds_row + ((static_cast<uint32_t>(ch) ^ swz) << 4), dw[ch * 4], dw[ch * 4 + 1], dw[ch * 4 + 2], dw[ch * 4 + 3]);
      tmem_wait_st();
      fence_proxy_async_smem();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_pd_full);
    }

    // ---------------- epilogue: warpgroup 0 stores dV, warpgroup 1 dK = scale * acc (K_j, V_j are dead) ----------------
    mbar_wait(bar_done, 0);
    tc_fence_after();
    const float mul = g == 0 ? 1.0f : prm.scale;
    const uint32_t stage = g == 0 ? k_smem : v_smem;
#pragma unroll
    for (int c4 = 0; c4 < kD / 32; ++c4) {
      uint32_t r[32];
      tmem_ld32(tmem_base + lane_addr + (g == 0 ? kTmemDV : kTmemDK) + c4 * 32, r);
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
      const CUtensorMap* om = g == 0 ? &maps.dv : &maps.dk;
#pragma unroll
      for (int pn = 0; pn < kPanels; ++pn) tma_store_4d(om, stage + pn * (kRows * 128), pn * 64, hj, row0, rank);
      bulk_commit();
      bulk_wait<0>();
    }
  } else {
    // ================================ dQ drain warpgroup ================================
    setmaxnreg_dec<96>();
    const int d = (warp & 3) * 32 + lane;                // head-dim index == TMEM lane of dQ^T
    const uint32_t dq_tmem = tmem_base + (static_cast<uint32_t>((warp & 3) * 32) << 16) + kTmemDQ;
    float* acc = prm.dq_acc + static_cast<size_t>(head) * prm.s_pad * kD + d;
    int* turn = prm.dq_turn + static_cast<size_t>(head) * n_iter;
    const bool first = key_tile == 0;
    const bool poller = threadIdx.x == kThreads - 128;
    int seen = poller ? ld_acquire_gpu(turn) : 0;           // whose turn it is at query tile 0
    for (int t = 0; t < n_iter; ++t) {
      mbar_wait(bar_acc + 8 * (t & 1), (t >> 1) & 1);
      tc_fence_after();
      uint32_t r[kQ];
      tmem_ld32(dq_tmem, r);
      tmem_ld32(dq_tmem + 32, r + 32);
      tmem_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_dq_free);
      // Publish step t-1 one step late: its reds were issued a whole step ago, so the fence that must precede the
      // flag finds them performed and costs its fixed latency only (fencing right after the reds put their L2 round
      // trip into every step: 97.9 ms instead of 61 ms per cfg 3 backward).
      if (t > 0) {
        __threadfence();
        named_bar_sync(3, 128);
        if (poller) st_release_gpu(turn + t - 1, key_tile + 1);
      }
      // this CTA's turn: key tiles add to dQ_acc[t] in ascending order
      if (poller) {
        while (seen != key_tile) seen = ld_acquire_gpu(turn + t);
      }
      named_bar_sync(3, 128);
      float* dst = acc + static_cast<size_t>(t) * kQ * kD;
      if (first) {
#pragma unroll
        for (int c = 0; c < kQ; ++c) dst[static_cast<size_t>(c) * kD] = __uint_as_float(r[c]);
      } else {
#pragma unroll
        for (int c = 0; c < kQ; ++c) red_add_f32(dst + static_cast<size_t>(c) * kD, __uint_as_float(r[c]));
      }
      if (poller && t + 1 < n_iter) seen = ld_acquire_gpu(turn + t + 1);    // next tile's turn, fetched while this one drains
    }
    __threadfence();
    named_bar_sync(3, 128);
    if (poller) st_release_gpu(turn + n_iter - 1, key_tile + 1);
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem_base, kTmemCols);
}

// dQ'_c[p][s][j][:] = bf16(scale * dq_acc[p*h_c + j][s][:]) -- the fp32 accumulator into the chunk-buffer layout
__global__ void __launch_bounds__(256)
attention_bwd_dq_convert_kernel(const float4* __restrict__ acc, uint4* __restrict__ dq, int S, int h_c, int P, int s_pad, float scale) {
  constexpr int kLanes = kD / 8;                          // 8 elements per thread
  const int64_t n = static_cast<int64_t>(P) * S * h_c * kLanes;
  const int64_t i = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
  if (i >= n) return;
  const int sub = static_cast<int>(i % kLanes);
  const int64_t L = i / kLanes;                           // output row in memory order: (p*S + s)*h_c + j
  const int j = static_cast<int>(L % h_c);
  const int64_t ps = L / h_c;
  const int s = static_cast<int>(ps % S);
  const int head = static_cast<int>(ps / S) * h_c + j;
  const float4* src = acc + (static_cast<size_t>(head) * s_pad + s) * (kD / 4) + sub * 2;
  const float4 a = __ldcs(src), b = __ldcs(src + 1);
  uint4 o;
  o.x = pack_bf16(a.x * scale, a.y * scale);
  o.y = pack_bf16(a.z * scale, a.w * scale);
  o.z = pack_bf16(b.x * scale, b.y * scale);
  o.w = pack_bf16(b.z * scale, b.w * scale);
  dq[i] = o;
}

cudaError_t map4d(CUtensorMap* m, const void* base, const AttnBwdArgs& a, uint32_t box_rows) {
  const uint64_t dims[4] = {static_cast<uint64_t>(a.D), static_cast<uint64_t>(a.h_c), static_cast<uint64_t>(a.S),
                            static_cast<uint64_t>(a.P)};
  const uint64_t strides[3] = {static_cast<uint64_t>(a.D) * 2, static_cast<uint64_t>(a.h_c) * a.D * 2,
                               static_cast<uint64_t>(a.S) * a.h_c * a.D * 2};
  const uint32_t box[4] = {64, 1, box_rows, 1};
  return encode_tensor_map(a.cache, m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, base, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
}

}  // namespace

cudaError_t attention_bwd_1pass_init() {
  static PerDeviceOnce once;
  return once_per_device(&once, [] {
    return cudaFuncSetAttribute(attention_bwd_1pass_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
  });
}

size_t attention_bwd_1pass_acc_bytes(int64_t S, int heads) {
  const int64_t s_pad = (S + kQ - 1) / kQ * kQ;
  return static_cast<size_t>(heads) * s_pad * kD * sizeof(float);
}
size_t attention_bwd_1pass_turn_bytes(int64_t S, int heads) {
  const int64_t s_pad = (S + kQ - 1) / kQ * kQ;
  return static_cast<size_t>(heads) * (s_pad / kQ + 1) * sizeof(int);     // turn counters, then one ticket counter per head
}

// After the statistics kernel: zero the turn counters, the single-pass kernel, the dQ conversion (3 stream operations).
cudaError_t launch_attention_bwd_1pass(const AttnBwdArgs& a, const void* stats, int s_pad, cudaStream_t stream) {
  if (a.D != kD || !a.dq_acc || !a.dq_turn) return cudaErrorInvalidValue;
  cudaError_t e = attention_bwd_1pass_init();
  if (e != cudaSuccess) return e;
  const int heads = a.P * a.h_c;
  Bwd1Maps m;
  if ((e = map4d(&m.k, a.k, a, kRows)) != cudaSuccess) return e;
  if ((e = map4d(&m.v, a.v, a, kRows)) != cudaSuccess) return e;
  if ((e = map4d(&m.q, a.q, a, kQ)) != cudaSuccess) return e;
  if ((e = map4d(&m.d_o, a.d_o, a, kQ)) != cudaSuccess) return e;
  if ((e = map4d(&m.dv, a.dv, a, kRows)) != cudaSuccess) return e;
  if ((e = map4d(&m.dk, a.dk, a, kRows)) != cudaSuccess) return e;
  Bwd1Params prm;
  prm.S = static_cast<int>(a.S);
  prm.n_iter = s_pad / kQ;
  prm.h_c = a.h_c;
  prm.s_pad = s_pad;
  prm.scale = a.scale;
  prm.scale_log2 = fmaxf(a.scale * 1.4426950408889634f, 1e-30f);
  prm.stats = static_cast<const float2*>(stats);
  prm.dq_acc = a.dq_acc;
  prm.dq_turn = a.dq_turn;
  prm.dq_ticket = a.dq_turn + static_cast<size_t>(heads) * (s_pad / kQ);
  if ((e = cudaMemsetAsync(a.dq_turn, 0, attention_bwd_1pass_turn_bytes(a.S, heads), stream)) != cudaSuccess) return e;
  const dim3 grid(static_cast<unsigned>((a.S + kRows - 1) / kRows), static_cast<unsigned>(heads));
  attention_bwd_1pass_kernel<<<grid, kThreads, kSmemBytes, stream>>>(m, prm);
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  const int64_t n = static_cast<int64_t>(heads) * a.S * (kD / 8);
  attention_bwd_dq_convert_kernel<<<static_cast<unsigned>((n + 255) / 256), 256, 0, stream>>>(
      reinterpret_cast<const float4*>(a.dq_acc), static_cast<uint4*>(a.dq), static_cast<int>(a.S), a.h_c, a.P, s_pad, a.scale);
  return cudaGetLastError();
}

}  // namespace hcms
