// Non-causal bf16 attention forward for one HCMS head chunk on sm_100a (tcgen05 / TMEM / TMA).
//
// Computes, for every logical rank p and local head j of the chunk (Eq. 2,
// Algorithm 1 line 15, bidirectional L43):
//     O'[p][i][j][:] = sum_k softmax_k(scale * Q'[p][i][j] . K'[p][k][j]) V'[p][k][j][:]
// on head-sharded buffers [P][S][h_c][D] (bf16 in, fp32 scores/softmax/accumulate, bf16 out).
//
// One CTA = one head x 256 query rows (two 128-row Q tiles that ping-pong), 384 threads:
//   warp 0      TMA producer: Q tiles once, then K_j / V_j tiles through a shared-memory ring
//   warp 1      MMA issuer (one lane): S_t = Q_t K_j^T (SS, M=128,N=128), O_t += P_t V_j (TS: P read from TMEM)
//   warp 2      TMEM allocator (512 columns: S_0,S_1 at 0/128 (P_t aliases S_t as packed bf16), O_0,O_1 at 256+)
//   warps 4-7   softmax warpgroup of tile 0: one thread per query row, online softmax in fp32 with lazy
//   warps 8-11  softmax warpgroup of tile 1    rescaling of O (only when the row max grew by > 2^8), epilogue
// While softmax_t works on S_t(j) the tensor core runs PV_{1-t}(j-1) and QK_{1-t}(j).
//
// The KV iteration order per (head, query tile) is fixed (j = 0..ceil(S/128)-1) and does not depend
// on how many heads a launch holds, so the output is bitwise independent of the chunking
// (the paper's "max error 0" claim, L304 / Table 14).
#include <cuda_bf16.h>

#include "hcms_internal.h"
#include "ptx.cuh"

namespace hcms {
using namespace ptx;

namespace {

constexpr int kBM = 128;          // query rows per tile (UMMA M)
constexpr int kBN = 128;          // keys per KV tile (UMMA N of QK^T, K extent of PV)
constexpr int kQTiles = 2;        // Q tiles per CTA
constexpr int kStages = 4;        // KV ring stages (each holds one K tile or one V tile)
constexpr int kThreads = 384;
constexpr int kTmemCols = 512;
constexpr float kRescaleThreshold = 8.0f;  // log2 units: rescale O only if the max grew by > 2^8

template <int D>
struct Cfg {
  static constexpr int kPanels = D / 64;                 // 128-byte swizzle panels along D
  static constexpr int kPanelBytes = 128 * 128;          // 128 rows x 128 B
  static constexpr int kTileBytes = kPanels * kPanelBytes;  // one Q / K / V tile
  static constexpr int kSmemBytes = (kQTiles + kStages) * kTileBytes + 1024 /*align*/ + 256 /*barriers*/;
  static constexpr int kTmemS = 0;                       // S_t at kTmemS + t*128
  static constexpr int kTmemO = 256;                     // O_t at kTmemO + t*D
};

// Shared-memory matrix descriptor, 128-byte swizzle (cute::UMMA::SmemDescriptor bit layout):
// [0,14) start>>4, [16,30) LBO>>4, [32,46) SBO>>4, [46,48) version=1, [61,64) layout=2 (SWIZZLE_128B).
__device__ __forceinline__ uint64_t make_desc(uint32_t smem_addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= static_cast<uint64_t>((smem_addr >> 4) & 0x3FFF);
  d |= static_cast<uint64_t>((lbo_bytes >> 4) & 0x3FFF) << 16;
  d |= static_cast<uint64_t>((sbo_bytes >> 4) & 0x3FFF) << 32;
  d |= 1ull << 46;
  d |= 2ull << 61;
  return d;
}

// Instruction descriptor for kind::f16: fp32 accumulate, bf16 A and B.
__host__ __device__ constexpr uint32_t make_idesc(int M, int N, bool b_mn_major) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn_major ? 1u : 0u) << 16) |
         (static_cast<uint32_t>(N >> 3) << 17) | (static_cast<uint32_t>(M >> 4) << 24);
}

struct alignas(64) AttnMaps {
  CUtensorMap q, k, v, o;   // rank-4 {D, h_c, S, P}, box {64, 1, 128, 1}, SWIZZLE_128B
};

struct AttnParams {
  int S;
  int n_kv;          // ceil(S/128)
  int h_c;
  float scale_log2;  // scale * log2(e)
};

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}

template <int D>
__global__ void __launch_bounds__(kThreads, 1)
attention_fwd_kernel(const __grid_constant__ AttnMaps maps, const AttnParams prm) {
  using C = Cfg<D>;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t q_smem = smem_base;                                  // kQTiles tiles
  const uint32_t kv_smem = smem_base + kQTiles * C::kTileBytes;       // kStages tiles
  const uint32_t bar_base = kv_smem + kStages * C::kTileBytes;        // 8-byte barriers
  // barrier indices
  const uint32_t bar_q_full = bar_base;                // [2]
  const uint32_t bar_kv_full = bar_base + 16;          // [kStages]
  const uint32_t bar_kv_empty = bar_kv_full + 8 * kStages;
  const uint32_t bar_s_full = bar_kv_empty + 8 * kStages;  // [2]
  const uint32_t bar_p_full = bar_s_full + 16;             // [2]
  const uint32_t bar_o_full = bar_p_full + 16;             // [2]
  const uint32_t tmem_slot = bar_o_full + 16;              // 4 bytes

  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  const int head = blockIdx.y;                 // p*h_c + j
  const int rank = head / prm.h_c;
  const int hj = head - rank * prm.h_c;
  const int q_row0 = blockIdx.x * (kQTiles * kBM);
  const int n_kv = prm.n_kv;

  if (threadIdx.x == 0) {
    for (int t = 0; t < kQTiles; ++t) {
      mbar_init(bar_q_full + 8 * t, 1);
      mbar_init(bar_s_full + 8 * t, 1);
      mbar_init(bar_p_full + 8 * t, kBM);
      mbar_init(bar_o_full + 8 * t, 1);
    }
    for (int s = 0; s < kStages; ++s) {
      mbar_init(bar_kv_full + 8 * s, 1);
      mbar_init(bar_kv_empty + 8 * s, 1);
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
    // ================================ producer / MMA warpgroup ================================
    setmaxnreg_dec<56>();
    if (warp == 0 && lane == 0) {
      // ---------------- TMA producer ----------------
      prefetch_tensormap(&maps.q);
      prefetch_tensormap(&maps.k);
      prefetch_tensormap(&maps.v);
      auto load_tile = [&](const CUtensorMap* tm, uint32_t dst, uint32_t bar, int row0) {
        mbar_expect_tx(bar, C::kTileBytes);
#pragma unroll
        for (int pn = 0; pn < C::kPanels; ++pn)
          tma_load_4d(dst + pn * C::kPanelBytes, tm, bar, pn * 64, hj, row0, rank);
      };
      load_tile(&maps.q, q_smem, bar_q_full, q_row0);
      int it = 0;  // ring item: K_j is item 2j, V_j is item 2j+1
      for (int j = 0; j < n_kv; ++j) {
#pragma unroll
        for (int kv = 0; kv < 2; ++kv, ++it) {
          const int stage = it % kStages;
          const uint32_t round = it / kStages;
          mbar_wait(bar_kv_empty + 8 * stage, (round & 1) ^ 1);
          load_tile(kv == 0 ? &maps.k : &maps.v, kv_smem + stage * C::kTileBytes, bar_kv_full + 8 * stage,
                    j * kBN);
          if (it == 0) load_tile(&maps.q, q_smem + C::kTileBytes, bar_q_full + 8, q_row0 + kBM);
        }
      }
    } else if (warp == 1 && lane == 0) {
      // ---------------- MMA issuer ----------------
      constexpr uint32_t idesc_qk = make_idesc(kBM, kBN, false);
      constexpr uint32_t idesc_pv = make_idesc(kBM, D, true);
      auto issue_qk = [&](int t, uint32_t k_tile) {
        // S_t[128 x 128] = Q_t[128 x D] * K_j[128 x D]^T ; both operands K-major, 128B-swizzled panels
        const uint32_t d_tmem = tmem_base + C::kTmemS + t * kBN;
        const uint32_t q_tile = q_smem + t * C::kTileBytes;
#pragma unroll
        for (int ks = 0; ks < D / 16; ++ks) {
          const uint32_t off = (ks >> 2) * C::kPanelBytes + (ks & 3) * 32;
          mma_ss(d_tmem, make_desc(q_tile + off, 16, 1024), make_desc(k_tile + off, 16, 1024), idesc_qk,
                 ks > 0 ? 1u : 0u);
        }
      };
      auto issue_pv = [&](int t, uint32_t v_tile, bool accumulate) {
        // O_t[128 x D] += P_t[128 x 128 (TMEM, packed bf16)] * V_j[128 keys x D] ; B is MN-major:
        // 64-wide D panels (LBO = panel stride), 8-key groups 1024 B apart (SBO)
        const uint32_t d_tmem = tmem_base + C::kTmemO + t * D;
        const uint32_t p_tmem = tmem_base + C::kTmemS + t * kBN;
#pragma unroll
        for (int ks = 0; ks < kBN / 16; ++ks) {
          mma_ts(d_tmem, p_tmem + ks * 8, make_desc(v_tile + ks * 2048, C::kPanelBytes, 1024), idesc_pv,
                 (accumulate || ks > 0) ? 1u : 0u);
        }
      };
      auto kv_wait = [&](int it) -> uint32_t {
        const int stage = it % kStages;
        mbar_wait(bar_kv_full + 8 * stage, (it / kStages) & 1);
        return kv_smem + stage * C::kTileBytes;
      };
      auto kv_release = [&](int it) { tc_commit(bar_kv_empty + 8 * (it % kStages)); };

      // prologue: S_0(0), S_1(0)
      {
        const uint32_t k_tile = kv_wait(0);
        mbar_wait(bar_q_full, 0);
        tc_fence_after();
        issue_qk(0, k_tile);
        tc_commit(bar_s_full);
        mbar_wait(bar_q_full + 8, 0);
        tc_fence_after();
        issue_qk(1, k_tile);
        tc_commit(bar_s_full + 8);
        kv_release(0);
      }
      for (int j = 0; j < n_kv; ++j) {
        const uint32_t v_tile = kv_wait(2 * j + 1);
        uint32_t k_next = 0;
#pragma unroll
        for (int t = 0; t < kQTiles; ++t) {
          mbar_wait(bar_p_full + 8 * t, j & 1);   // P_t(j) written, O_t rescaled if needed
          tc_fence_after();
          issue_pv(t, v_tile, j > 0);
          tc_commit(bar_o_full + 8 * t);
          if (t == kQTiles - 1) kv_release(2 * j + 1);
          if (j + 1 < n_kv) {
            if (t == 0) {
              k_next = kv_wait(2 * j + 2);
              tc_fence_after();
            }
            issue_qk(t, k_next);
            tc_commit(bar_s_full + 8 * t);
            if (t == kQTiles - 1) kv_release(2 * j + 2);
          }
        }
      }
    }
    __syncwarp();
  } else {
    // ================================ softmax warpgroups ================================
    setmaxnreg_inc<224>();
    const int t = (warp >> 2) - 1;                       // Q tile of this warpgroup
    const int row = (warp & 3) * 32 + lane;              // row inside the tile == TMEM lane
    const uint32_t lane_addr = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t s_tmem = tmem_base + lane_addr + C::kTmemS + t * kBN;
    const uint32_t o_tmem = tmem_base + lane_addr + C::kTmemO + t * D;
    const float scale_log2 = prm.scale_log2;
    const int tail_valid = prm.S - (n_kv - 1) * kBN;     // valid keys in the last KV tile (1..128)

    float m_run = -INFINITY;   // running (possibly stale) row max, raw score units
    float l_run = 0.f;         // running row sum of exp2((s - m_run)*scale_log2)

    for (int j = 0; j < n_kv; ++j) {
      mbar_wait(bar_s_full + 8 * t, j & 1);
      tc_fence_after();
      uint32_t sr[kBN];
#pragma unroll
      for (int c4 = 0; c4 < kBN / 32; ++c4) tmem_ld32(s_tmem + c4 * 32, &sr[c4 * 32]);
      tmem_wait_ld();
      if (j == n_kv - 1 && tail_valid < kBN) {
#pragma unroll
        for (int c = 0; c < kBN; ++c)
          if (c >= tail_valid) sr[c] = 0xff800000u;   // -inf: keys beyond S do not exist
      }
      float mx0 = __uint_as_float(sr[0]), mx1 = __uint_as_float(sr[1]);
      float mx2 = __uint_as_float(sr[2]), mx3 = __uint_as_float(sr[3]);
#pragma unroll
      for (int c = 4; c < kBN; c += 4) {
        mx0 = fmaxf(mx0, __uint_as_float(sr[c]));
        mx1 = fmaxf(mx1, __uint_as_float(sr[c + 1]));
        mx2 = fmaxf(mx2, __uint_as_float(sr[c + 2]));
        mx3 = fmaxf(mx3, __uint_as_float(sr[c + 3]));
      }
      const float m_tile = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3));
      if (j == 0) {
        m_run = m_tile;
      } else {
        const bool need = (m_tile - m_run) * scale_log2 > kRescaleThreshold;
        if (__any_sync(0xffffffffu, need)) {
          // O_t currently holds sum_k p_k V_k relative to m_run: wait for PV_t(j-1), then rescale
          mbar_wait(bar_o_full + 8 * t, (j - 1) & 1);
          tc_fence_after();
          const float alpha = need ? ex2((m_run - m_tile) * scale_log2) : 1.0f;
          if (need) {
            l_run *= alpha;
            m_run = m_tile;
          }
#pragma unroll
          for (int c4 = 0; c4 < D / 32; ++c4) {
            uint32_t orr[32];
            tmem_ld32(o_tmem + c4 * 32, orr);
            tmem_wait_ld();
#pragma unroll
            for (int c = 0; c < 32; ++c) orr[c] = __float_as_uint(__uint_as_float(orr[c]) * alpha);
            tmem_st32(o_tmem + c4 * 32, orr);
          }
        }
      }
      const float neg_m = -m_run * scale_log2;
      float sum0 = 0.f, sum1 = 0.f, sum2 = 0.f, sum3 = 0.f;
      uint32_t pr[kBN / 2];
#pragma unroll
      for (int c = 0; c < kBN; c += 4) {
        const float p0 = ex2(fmaf(__uint_as_float(sr[c]), scale_log2, neg_m));
        const float p1 = ex2(fmaf(__uint_as_float(sr[c + 1]), scale_log2, neg_m));
        const float p2 = ex2(fmaf(__uint_as_float(sr[c + 2]), scale_log2, neg_m));
        const float p3 = ex2(fmaf(__uint_as_float(sr[c + 3]), scale_log2, neg_m));
        sum0 += p0;
        sum1 += p1;
        sum2 += p2;
        sum3 += p3;
        pr[c / 2] = pack_bf16(p0, p1);
        pr[c / 2 + 1] = pack_bf16(p2, p3);
      }
      l_run += (sum0 + sum1) + (sum2 + sum3);
      // P_t aliases the first 64 columns of S_t (two bf16 per 32-bit column, element 2c in the low half)
      tmem_st32(s_tmem, &pr[0]);
      tmem_st32(s_tmem + 32, &pr[32]);
      tmem_wait_st();
      tc_fence_before();
      mbar_arrive(bar_p_full + 8 * t);
    }

    // ---------------- epilogue: O_t / l -> bf16 -> swizzled smem (Q_t's buffer) -> TMA store ----------------
    mbar_wait(bar_o_full + 8 * t, (n_kv - 1) & 1);
    tc_fence_after();
    const float inv_l = 1.0f / l_run;
    const uint32_t o_smem = q_smem + t * C::kTileBytes;   // all QK_t MMAs have completed
#pragma unroll
    for (int c4 = 0; c4 < D / 32; ++c4) {
      uint32_t orr[32];
      tmem_ld32(o_tmem + c4 * 32, orr);
      tmem_wait_ld();
      const uint32_t panel = c4 >> 1;
#pragma unroll
      for (int q4 = 0; q4 < 4; ++q4) {
        uint32_t w[4];
#pragma unroll
        for (int e = 0; e < 4; ++e)
          w[e] = pack_bf16(__uint_as_float(orr[q4 * 8 + 2 * e]) * inv_l,
                           __uint_as_float(orr[q4 * 8 + 2 * e + 1]) * inv_l);
        const uint32_t chunk = (c4 & 1) * 4 + q4;                  // 16-byte chunk inside the 128-byte row
        const uint32_t addr = o_smem + panel * C::kPanelBytes + row * 128 + ((chunk ^ (row & 7)) << 4);
        asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(w[0]), "r"(w[1]), "r"(w[2]),
                     "r"(w[3])
                     : "memory");
      }
    }
    fence_proxy_async_smem();
    named_bar_sync(1 + t, kBM);
    if ((warp & 3) == 0 && lane == 0) {
      const int row0 = q_row0 + t * kBM;
      if (row0 < prm.S) {
#pragma unroll
        for (int pn = 0; pn < C::kPanels; ++pn)
          tma_store_4d(&maps.o, o_smem + pn * C::kPanelBytes, pn * 64, hj, row0, rank);
        bulk_commit();
        bulk_wait<0>();
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem_base, kTmemCols);
}

cudaError_t make_maps(const AttnArgs& a, AttnMaps* m) {
  const uint64_t dims[4] = {static_cast<uint64_t>(a.D), static_cast<uint64_t>(a.h_c), static_cast<uint64_t>(a.S),
                            static_cast<uint64_t>(a.P)};
  const uint64_t strides[3] = {static_cast<uint64_t>(a.D) * 2, static_cast<uint64_t>(a.h_c) * a.D * 2,
                               static_cast<uint64_t>(a.S) * a.h_c * a.D * 2};
  const uint32_t box[4] = {64, 1, 128, 1};
  const void* ptrs[4] = {a.q, a.k, a.v, a.o};
  CUtensorMap* outs[4] = {&m->q, &m->k, &m->v, &m->o};
  for (int i = 0; i < 4; ++i) {
    cudaError_t e = encode_tensor_map(outs[i], CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, ptrs[i], dims, strides, box,
                                      CU_TENSOR_MAP_SWIZZLE_128B);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

}  // namespace

cudaError_t attention_init() {
  cudaError_t e = cudaFuncSetAttribute(attention_fwd_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       Cfg<128>::kSmemBytes);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(attention_fwd_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              Cfg<64>::kSmemBytes);
}

cudaError_t launch_attention(const AttnArgs& a, cudaStream_t stream) {
  AttnMaps maps;
  cudaError_t e = make_maps(a, &maps);
  if (e != cudaSuccess) return e;
  AttnParams prm;
  prm.S = static_cast<int>(a.S);
  prm.n_kv = static_cast<int>((a.S + kBN - 1) / kBN);
  prm.h_c = a.h_c;
  // scale == 0 is legal (uniform softmax); a tiny positive factor keeps (-inf)*scale_log2 = -inf for
  // masked tail keys while exp2(s*1e-30) is exactly 1 in fp32.
  prm.scale_log2 = fmaxf(a.scale * 1.4426950408889634f, 1e-30f);
  dim3 grid(static_cast<unsigned>((a.S + kQTiles * kBM - 1) / (kQTiles * kBM)), static_cast<unsigned>(a.P * a.h_c));
  if (a.D == 128)
    attention_fwd_kernel<128><<<grid, kThreads, Cfg<128>::kSmemBytes, stream>>>(maps, prm);
  else if (a.D == 64)
    attention_fwd_kernel<64><<<grid, kThreads, Cfg<64>::kSmemBytes, stream>>>(maps, prm);
  else
    return cudaErrorInvalidValue;
  return cudaGetLastError();
}

}  // namespace hcms
