// bf16 projection GEMMs of the HCMS attention layer on sm_100a (tcgen05 / TMEM / TMA).
//
// PAPER.md section 3.1 (L59) and Algorithm 1 (L170): line 2 "Q,K,V <- QKVProjection(X)", line 3
// "Q,K <- ApplyRoPE(Q,K)", line 27 "Y <- OutputProjection(O)" -- the T_other of Eq. 1 (L61).
// Both projections are  C[M,N] = A[M,K] * B[N,K]^T  (activations [tokens, features] times a
// torch.nn.Linear-style weight [out_features, in_features]), bf16 operands, fp32 accumulation in
// TMEM, bf16 output.  The QKV variant splits the N = 3*H*D output features over three tensors
// q,k,v [S,H,D] and applies the rotary embedding to q and k in the epilogue, on the fp32
// accumulators, before the single rounding to bf16: adjacent pairs (x[2i], x[2i+1]) of a head are
// rotated by the angle whose cos/sin the caller tabulates per (token, i)  (reading R-23).
//
// Two kernels: the CTA-pair kernel below (cta_group::2, 256 x 256 tiles; default when the output width allows) and this
// single-CTA kernel (128 x 256 or 128 x 128 tiles), which also serves as the fallback (HCMS_FLAG_GEMM_1CTA).
// Persistent kernel, one CTA per SM, 256 threads:
//   warp 0     TMA producer: A tile [128 x 64] and B tile [BN x 64] per k-block into a shared-memory ring
//   warp 1     MMA issuer (one elected lane): tcgen05.mma.cta_group::1.kind::f16, M=128, N=BN, K=16, SS
//   warp 2     TMEM allocator: 2 accumulators of BN fp32 columns (the epilogue of tile i overlaps the
//              main loop of tile i+1)
//   warps 4-7  epilogue: tcgen05.ld -> (RoPE) -> bf16 -> 128-byte-swizzled staging -> TMA store (rows >= M clipped)
// Tiles are visited in bands of 16 m-tiles x all n-tiles so that the ~148 tiles in flight share A and B
// panels through L2.
#include <cuda_bf16.h>

#include "hcms_internal.h"
#include "ptx.cuh"


namespace hcms {
using namespace ptx;

namespace {

constexpr int kBM = 128;          // UMMA M
constexpr int kBK = 64;           // one 128-byte swizzle panel of bf16 along K
constexpr int kThreads = 256;
constexpr int kABytes = kBM * kBK * 2;
constexpr int kEpiPanelBytes = kBM * 128;     // 128 rows x 64 bf16

template <int BN>
struct Cfg {
  static constexpr int kBBytes = BN * kBK * 2;
  static constexpr int kStageBytes = kABytes + kBBytes;
  static constexpr int kStages = BN == 256 ? 4 : 6;
  static constexpr int kSmemBytes = kStages * kStageBytes + 2 * kEpiPanelBytes + 1024 /*align*/ + 256 /*barriers*/;
  static constexpr int kTmemCols = 2 * BN;
};

struct alignas(64) GemmMaps {
  CUtensorMap a;        // {K, M}, box {64, 128}, SWIZZLE_128B
  CUtensorMap b;        // {K, N}, box {64, BN}
  CUtensorMap out[3];   // {n_per_out, M}, box {64, 128}
};

// Fused all-to-all (SURVEY 8(f3) "scatter fused into the QKV epilogue"): one rank-4 map {D, h_c, S, P}, box
// {64, 1, 128, 1}, per (tensor, head chunk) over the head-sharded chunk buffers [P][S][h_c][D] of the plan.
constexpr int kMaxChunks = 16;
constexpr int kMaxFusedMaps = 96;   // 3 tensors x 16 chunks on one device, or 3 x C x P <= 96 between real ranks (12 KB of kernel parameters)
constexpr int kMaxLocalHeads = 64;
struct alignas(64) ChunkMaps {
  CUtensorMap m[kMaxFusedMaps];   // [tensor * C + chunk], or [(tensor * C + chunk) * P + destination rank] between real ranks
};
enum { kPlain = 0, kFusedOut = 1, kFusedA = 2 };

struct GemmParams {
  int M, N, K;
  // fused modes: heads -> (logical rank, chunk, index in chunk); D = 1 << d_shift
  int d_shift, Hl, C;
  uint8_t chunk_of[kMaxLocalHeads], j_of[kMaxLocalHeads];
  int n_per_out;        // output features per output tensor (N for a plain GEMM, H*D for the QKV projection)
  int rope_outs;        // the first rope_outs output tensors get the rotary embedding (2 = q and k; 0 = none)
  int half_d;           // D/2 = pairs per head
  int d_mask;           // D-1 (D is a power of two >= 64)
  const float* cos;     // [M, D/2]
  const float* sin;
  int m_tiles, n_tiles;
  int group_m;          // m-tiles per band of the tile walk
  // kFusedOut between real ranks (hcms_dist): one map per (tensor, chunk, destination rank) instead of one per (tensor,
  // chunk) with the rank as its 4th coordinate: map index = (t * C + c) * peer_n + rank * peer_on
  int peer_n, peer_on;  // (P, 1) with peer maps, (1, 0) without
};

__device__ __forceinline__ void tile_coords(int tile, const GemmParams& p, int& m0, int& n0) {
  const int per_band = p.group_m * p.n_tiles;
  const int band = tile / per_band;
  const int r = tile - band * per_band;
  const int left = p.m_tiles - band * p.group_m;
  const int rows = left < p.group_m ? left : p.group_m;
  const int n = r / rows;
  m0 = (band * p.group_m + (r - n * rows)) * kBM;
  n0 = n;  // caller multiplies by BN
}

__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

// kMode: kPlain = A [M,K] in, outputs [M, n_per_out] out; kFusedOut = output column n belongs to head n / D of its
// tensor and is stored straight into that head's chunk buffer (the input all-to-all happens in the epilogue's TMA
// store); kFusedA = A's k-block kb is columns of head kb*64 / D and is loaded straight from that head's chunk buffer
// (the output all-to-all + Concat happen in the producer's TMA load).
template <int BN, int kMode>
__global__ void __launch_bounds__(kThreads, 1)
gemm_bf16_nt_kernel(const __grid_constant__ GemmMaps maps, const __grid_constant__ ChunkMaps cmaps, const GemmParams prm) {
  using C = Cfg<BN>;
  constexpr int kStages = C::kStages;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t ring = smem_base;                                   // kStages x (A tile, B tile)
  const uint32_t epi = ring + kStages * C::kStageBytes;              // 2 staging panels
  const uint32_t bar_base = epi + 2 * kEpiPanelBytes;
  const uint32_t bar_full = bar_base;                                // [kStages] TMA -> MMA
  const uint32_t bar_empty = bar_full + 8 * kStages;                 // [kStages] MMA -> TMA
  const uint32_t bar_acc_full = bar_empty + 8 * kStages;             // [2] MMA -> epilogue
  const uint32_t bar_acc_empty = bar_acc_full + 16;                  // [2] epilogue -> MMA
  const uint32_t tmem_slot = bar_acc_empty + 16;

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
  const int lane = threadIdx.x & 31;
  const int total_tiles = prm.m_tiles * prm.n_tiles;
  const int n_kb = (prm.K + kBK - 1) / kBK;

  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) {
      mbar_init(bar_full + 8 * s, 1);
      mbar_init(bar_empty + 8 * s, 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(bar_acc_full + 8 * a, 1);
      mbar_init(bar_acc_empty + 8 * a, 4);   // one elected lane per epilogue warp
    }
    fence_mbar_init();
    fence_proxy_async_smem();
  }
  if (warp == 2) {
    tmem_alloc(tmem_slot, C::kTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  if (warp == 0) {
    // ---------------- TMA producer ----------------
    const bool leader = elect_one();
    if (leader) {
      prefetch_tensormap(&maps.a);
      prefetch_tensormap(&maps.b);
    }
    int stage = 0;
    uint32_t phase = 0;
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
      int m0, n0;
      tile_coords(tile, prm, m0, n0);
      n0 *= BN;
      for (int kb = 0; kb < n_kb; ++kb) {
        mbar_wait(bar_empty + 8 * stage, phase ^ 1);
        if (leader) {
          const uint32_t dst = ring + stage * C::kStageBytes;
          mbar_expect_tx(bar_full + 8 * stage, C::kStageBytes);
          if (kMode == kFusedA) {
            const int head = (kb * kBK) >> prm.d_shift, rank = head / prm.Hl, lh = head - rank * prm.Hl;
            tma_load_4d(dst, &cmaps.m[prm.chunk_of[lh]], bar_full + 8 * stage, (kb * kBK) & prm.d_mask, prm.j_of[lh], m0, rank);
          } else {
            tma_load_2d(dst, &maps.a, bar_full + 8 * stage, kb * kBK, m0);
          }
          tma_load_2d(dst + kABytes, &maps.b, bar_full + 8 * stage, kb * kBK, n0);
        }
        __syncwarp();
        if (++stage == kStages) {
          stage = 0;
          phase ^= 1;
        }
      }
    }
  } else if (warp == 1) {
    // ---------------- MMA issuer ----------------
    const bool leader = elect_one();
    constexpr uint32_t idesc = umma_idesc_bf16(kBM, BN, false, false);
    constexpr uint32_t hi = umma_desc_hi(1024);      // 8 rows x 128 B between core-matrix groups
    int stage = 0;
    uint32_t phase = 0;
    int it = 0;
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x, ++it) {
      const int acc = it & 1;
      mbar_wait(bar_acc_empty + 8 * acc, ((it >> 1) & 1) ^ 1);   // the epilogue has drained this accumulator
      tc_fence_after();
      const uint32_t d_tmem = tmem_base + acc * BN;
      for (int kb = 0; kb < n_kb; ++kb) {
        mbar_wait(bar_full + 8 * stage, phase);
        tc_fence_after();
        if (leader) {
          const uint32_t a_lo = umma_desc_lo(ring + stage * C::kStageBytes, 16);
          const uint32_t b_lo = umma_desc_lo(ring + stage * C::kStageBytes + kABytes, 16);
#pragma unroll
          for (int ks = 0; ks < kBK / 16; ++ks)     // 16 bf16 = 32 bytes along the swizzled row
            mma_ss_lohi(d_tmem, a_lo + ks * 2, b_lo + ks * 2, hi, hi, idesc, (kb > 0 || ks > 0) ? 1u : 0u);
          tc_commit(bar_empty + 8 * stage);
          if (kb == n_kb - 1) tc_commit(bar_acc_full + 8 * acc);
        }
        __syncwarp();
        if (++stage == kStages) {
          stage = 0;
          phase ^= 1;
        }
      }
    }
  } else if (warp >= 4) {
    // ---------------- epilogue ----------------
    const int ew = warp & 3;                       // TMEM lane quarter this warp may read
    const int row = ew * 32 + lane;
    const uint32_t lane_addr = static_cast<uint32_t>(ew * 32) << 16;
    const uint32_t swz = static_cast<uint32_t>(row & 7);
    const bool issuer = threadIdx.x == 128;
    int it = 0;
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x, ++it) {
      const int acc = it & 1;
      int m0, n0;
      tile_coords(tile, prm, m0, n0);
      n0 *= BN;
      const int t_out = n0 / prm.n_per_out;
      const int col0 = n0 - t_out * prm.n_per_out;
      const bool rope = t_out < prm.rope_outs;
      const int grow = min(m0 + row, prm.M - 1);   // tail rows compute on a valid row; the TMA store clips them
      mbar_wait(bar_acc_full + 8 * acc, (it >> 1) & 1);
      tc_fence_after();
#pragma unroll 1
      for (int ch = 0; ch < BN / 64; ++ch) {
        const uint32_t buf = epi + (ch & 1) * kEpiPanelBytes;
        if (issuer) bulk_wait_read<1>();           // the store that last read this panel has drained
        named_bar_sync(1, 128);
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          uint32_t r[32];
          tmem_ld32(tmem_base + lane_addr + acc * BN + ch * 64 + half * 32, r);
          tmem_wait_ld();
          if (rope) {
            const int pair0 = (((col0 + ch * 64 + half * 32) & prm.d_mask) >> 1);
            const float4* cp = reinterpret_cast<const float4*>(prm.cos + static_cast<size_t>(grow) * prm.half_d + pair0);
            const float4* sp = reinterpret_cast<const float4*>(prm.sin + static_cast<size_t>(grow) * prm.half_d + pair0);
#pragma unroll
            for (int g = 0; g < 4; ++g) {
              const float4 c4 = __ldg(cp + g), s4 = __ldg(sp + g);
              const float cs[4] = {c4.x, c4.y, c4.z, c4.w}, sn[4] = {s4.x, s4.y, s4.z, s4.w};
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                const float a = __uint_as_float(r[g * 8 + 2 * e]), b = __uint_as_float(r[g * 8 + 2 * e + 1]);
                r[g * 8 + 2 * e] = __float_as_uint(a * cs[e] - b * sn[e]);
                r[g * 8 + 2 * e + 1] = __float_as_uint(a * sn[e] + b * cs[e]);
              }
            }
          }
#pragma unroll
          for (int q4 = 0; q4 < 4; ++q4) {
            uint32_t w[4];
#pragma unroll
            for (int e = 0; e < 4; ++e)
              w[e] = pack_bf16(__uint_as_float(r[q4 * 8 + 2 * e]), __uint_as_float(r[q4 * 8 + 2 * e + 1]));
            const uint32_t chunk = half * 4 + q4;     // 16-byte chunk inside the 128-byte row
            st_shared_v4(buf + row * 128 + ((chunk ^ swz) << 4), w[0], w[1], w[2], w[3]);
          }
        }
        if (ch == BN / 64 - 1) {                      // every column of this accumulator is in registers / smem
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(bar_acc_empty + 8 * acc);
        }
        fence_proxy_async_smem();
        named_bar_sync(1, 128);
        if (issuer) {
          if (kMode == kFusedOut) {
            const int within = col0 + ch * 64;
            const int head = within >> prm.d_shift, rank = head / prm.Hl, lh = head - rank * prm.Hl;
            tma_store_4d(&cmaps.m[(t_out * prm.C + prm.chunk_of[lh]) * prm.peer_n + rank * prm.peer_on], buf, within & prm.d_mask, prm.j_of[lh], m0,
                         prm.peer_on ? 0 : rank);
          } else {
            tma_store_2d(&maps.out[t_out], buf, col0 + ch * 64, m0);
          }
          bulk_commit();
        }
      }
    }
    if (issuer) bulk_wait<0>();
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem_base, C::kTmemCols);
}

}  // namespace

// ------------------------------------------------------------------------------------------
// CTA-pair variant (tcgen05 cta_group::2): a cluster of two CTAs on one TPC computes a 256 x 256 tile.  Each CTA
// loads its own 128 rows of A and HALF of the B tile (128 of the 256 weight rows); one thread of the leader CTA issues
// M=256 MMAs that read A and B from both CTAs' shared memory and write each CTA's 128 accumulator rows into its own
// TMEM.  Per CTA this halves the B traffic into and out of shared memory and the number of MMA instructions.
// Barriers: `full` lives in the leader (both CTAs' TMA bytes are counted there), `empty` and `acc_full` are signalled
// in both CTAs by multicast commits, `acc_empty` lives in the leader and collects the epilogue warps of both CTAs.
// ------------------------------------------------------------------------------------------
struct Cfg2 {
  static constexpr int kBN = 256;
  static constexpr int kBHalfBytes = (kBN / 2) * kBK * 2;
  static constexpr int kStageBytes = kABytes + kBHalfBytes;     // per CTA
  static constexpr int kStages = 6;
  static constexpr int kSmemBytes = kStages * kStageBytes + 2 * kEpiPanelBytes + 1024 + 256;
  static constexpr int kTmemCols = 2 * kBN;
};

template <int kMode>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
gemm_bf16_nt_2cta_kernel(const __grid_constant__ GemmMaps maps, const __grid_constant__ ChunkMaps cmaps, const GemmParams prm) {
  using C = Cfg2;
  constexpr int BN = C::kBN;
  constexpr int kStages = C::kStages;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t ring = smem_base;
  const uint32_t epi = ring + kStages * C::kStageBytes;
  const uint32_t bar_base = epi + 2 * kEpiPanelBytes;
  const uint32_t bar_full = bar_base;                       // [kStages] leader only: TMA of both CTAs -> MMA
  const uint32_t bar_empty = bar_full + 8 * kStages;        // [kStages] per CTA: MMA -> TMA (multicast commit)
  const uint32_t bar_acc_full = bar_empty + 8 * kStages;    // [2] per CTA: MMA -> epilogue (multicast commit)
  const uint32_t bar_acc_empty = bar_acc_full + 16;         // [2] leader only: epilogue warps of both CTAs -> MMA
  const uint32_t tmem_slot = bar_acc_empty + 16;

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);
  const int lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int cluster_id = blockIdx.x >> 1, n_clusters = gridDim.x >> 1;
  const int total_tiles = prm.m_tiles * prm.n_tiles;       // m_tiles counts 256-row cluster tiles here
  const int n_kb = (prm.K + kBK - 1) / kBK;

  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) {
      mbar_init(bar_full + 8 * s, 1);
      mbar_init(bar_empty + 8 * s, 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(bar_acc_full + 8 * a, 1);
      mbar_init(bar_acc_empty + 8 * a, 8);   // 4 epilogue warps x 2 CTAs
    }
    fence_mbar_init();
    fence_proxy_async_smem();
  }
  if (warp == 2) {
    tmem_alloc_2sm(tmem_slot, C::kTmemCols);
    tmem_relinquish_2sm();
  }
  tc_fence_before();
  cluster_sync();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  if (warp == 0) {
    // ---------------- TMA producer (both CTAs) ----------------
    const bool leader = elect_one();
    if (leader) {
      prefetch_tensormap(&maps.a);
      prefetch_tensormap(&maps.b);
    }
    // L2 policy (swept on B200, profiles/r2e_gemm_l2.md): operand tiles are re-read by the other clusters of the wave (B)
    // and of the band (A), so both loads ask for evict_last; the output, written once, asks for evict_first below
    const uint64_t pol_a = l2_policy_evict_last(), pol_b = pol_a;
    int stage = 0;
    uint32_t phase = 0;
    for (int tile = cluster_id; tile < total_tiles; tile += n_clusters) {
      int m0, n0;
      tile_coords(tile, prm, m0, n0);
      m0 = 2 * m0 + static_cast<int>(rank) * kBM;            // tile_coords counted in units of kBM
      n0 = n0 * BN + static_cast<int>(rank) * (BN / 2);
      for (int kb = 0; kb < n_kb; ++kb) {
        mbar_wait(bar_empty + 8 * stage, phase ^ 1);
        if (leader) {
          const uint32_t dst = ring + stage * C::kStageBytes;
          const uint32_t full0 = mapa(bar_full + 8 * stage, 0);
          if (rank == 0) mbar_expect_tx(bar_full + 8 * stage, 2 * C::kStageBytes);
          if (kMode == kFusedA) {
            const int head = (kb * kBK) >> prm.d_shift, hr = head / prm.Hl, lh = head - hr * prm.Hl;
            tma_load_4d_2sm(dst, &cmaps.m[prm.chunk_of[lh]], full0, (kb * kBK) & prm.d_mask, prm.j_of[lh], m0, hr);
          } else {
            tma_load_2d_2sm_hint(dst, &maps.a, full0, kb * kBK, m0, pol_a);
          }
          tma_load_2d_2sm_hint(dst + kABytes, &maps.b, full0, kb * kBK, n0, pol_b);
        }
        __syncwarp();
        if (++stage == kStages) {
          stage = 0;
          phase ^= 1;
        }
      }
    }
  } else if (warp == 1 && rank == 0) {
    // ---------------- MMA issuer (leader CTA) ----------------
    const bool leader = elect_one();
    constexpr uint32_t idesc = umma_idesc_bf16(2 * kBM, BN, false, false);
    constexpr uint32_t hi = umma_desc_hi(1024);
    int stage = 0;
    uint32_t phase = 0;
    int it = 0;
    for (int tile = cluster_id; tile < total_tiles; tile += n_clusters, ++it) {
      const int acc = it & 1;
      mbar_wait(bar_acc_empty + 8 * acc, ((it >> 1) & 1) ^ 1);
      tc_fence_after();
      const uint32_t d_tmem = tmem_base + acc * BN;
      for (int kb = 0; kb < n_kb; ++kb) {
        mbar_wait(bar_full + 8 * stage, phase);
        tc_fence_after();
        if (leader) {
          const uint32_t a_lo = umma_desc_lo(ring + stage * C::kStageBytes, 16);
          const uint32_t b_lo = umma_desc_lo(ring + stage * C::kStageBytes + kABytes, 16);
#pragma unroll
          for (int ks = 0; ks < kBK / 16; ++ks)
            mma_ss_lohi_2sm(d_tmem, a_lo + ks * 2, b_lo + ks * 2, hi, hi, idesc, (kb > 0 || ks > 0) ? 1u : 0u);
          tc_commit_2sm(bar_empty + 8 * stage, 3);
          if (kb == n_kb - 1) tc_commit_2sm(bar_acc_full + 8 * acc, 3);
        }
        __syncwarp();
        if (++stage == kStages) {
          stage = 0;
          phase ^= 1;
        }
      }
    }
  } else if (warp >= 4) {
    // ---------------- epilogue (both CTAs, each its own 128 rows) ----------------
    const int ew = warp & 3;
    const int row = ew * 32 + lane;
    const uint32_t lane_addr = static_cast<uint32_t>(ew * 32) << 16;
    const uint32_t swz = static_cast<uint32_t>(row & 7);
    const bool issuer = threadIdx.x == 128;
    const uint64_t pol_out = l2_policy_evict_first();   // the output is written once and not read again here
    int it = 0;
    for (int tile = cluster_id; tile < total_tiles; tile += n_clusters, ++it) {
      const int acc = it & 1;
      int m0, n0;
      tile_coords(tile, prm, m0, n0);
      m0 = 2 * m0 + static_cast<int>(rank) * kBM;
      n0 *= BN;
      const int t_out = n0 / prm.n_per_out;
      const int col0 = n0 - t_out * prm.n_per_out;
      const bool rope = t_out < prm.rope_outs;
      const int grow = min(m0 + row, prm.M - 1);
      mbar_wait(bar_acc_full + 8 * acc, (it >> 1) & 1);
      tc_fence_after();
#pragma unroll 1
      for (int ch = 0; ch < BN / 64; ++ch) {
        const uint32_t buf = epi + (ch & 1) * kEpiPanelBytes;
        if (issuer) bulk_wait_read<1>();
        named_bar_sync(1, 128);
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          uint32_t r[32];
          tmem_ld32(tmem_base + lane_addr + acc * BN + ch * 64 + half * 32, r);
          tmem_wait_ld();
          if (rope) {
            const int pair0 = (((col0 + ch * 64 + half * 32) & prm.d_mask) >> 1);
            const float4* cp = reinterpret_cast<const float4*>(prm.cos + static_cast<size_t>(grow) * prm.half_d + pair0);
            const float4* sp = reinterpret_cast<const float4*>(prm.sin + static_cast<size_t>(grow) * prm.half_d + pair0);
#pragma unroll
            for (int g = 0; g < 4; ++g) {
              const float4 c4 = __ldg(cp + g), s4 = __ldg(sp + g);
              const float cs[4] = {c4.x, c4.y, c4.z, c4.w}, sn[4] = {s4.x, s4.y, s4.z, s4.w};
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                const float a = __uint_as_float(r[g * 8 + 2 * e]), b = __uint_as_float(r[g * 8 + 2 * e + 1]);
                r[g * 8 + 2 * e] = __float_as_uint(a * cs[e] - b * sn[e]);
                r[g * 8 + 2 * e + 1] = __float_as_uint(a * sn[e] + b * cs[e]);
              }
            }
          }
#pragma unroll
          for (int q4 = 0; q4 < 4; ++q4) {
            uint32_t w[4];
#pragma unroll
            for (int e = 0; e < 4; ++e)
              w[e] = pack_bf16(__uint_as_float(r[q4 * 8 + 2 * e]), __uint_as_float(r[q4 * 8 + 2 * e + 1]));
            const uint32_t chunk = half * 4 + q4;
            st_shared_v4(buf + row * 128 + ((chunk ^ swz) << 4), w[0], w[1], w[2], w[3]);
          }
        }
        if (ch == BN / 64 - 1) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(mapa(bar_acc_empty + 8 * acc, 0));
        }
        fence_proxy_async_smem();
        named_bar_sync(1, 128);
        if (issuer && m0 < prm.M) {
          if (kMode == kFusedOut) {
            const int within = col0 + ch * 64;
            const int head = within >> prm.d_shift, hr = head / prm.Hl, lh = head - hr * prm.Hl;
            tma_store_4d(&cmaps.m[(t_out * prm.C + prm.chunk_of[lh]) * prm.peer_n + hr * prm.peer_on], buf, within & prm.d_mask, prm.j_of[lh], m0,
                         prm.peer_on ? 0 : hr);
          } else {
            tma_store_2d_hint(&maps.out[t_out], buf, col0 + ch * 64, m0, pol_out);
          }
        }
        if (issuer) bulk_commit();
      }
    }
    if (issuer) bulk_wait<0>();
  }

  tc_fence_before();
  cluster_sync();
  if (warp == 2) tmem_dealloc_2sm(tmem_base, C::kTmemCols);
}

// ------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------
namespace {

cudaError_t map2d(TmapCache* cache, CUtensorMap* m, const void* base, uint64_t inner, uint64_t outer, uint32_t box_inner,
                  uint32_t box_outer) {
  const uint64_t dims[2] = {inner, outer};
  const uint64_t strides[1] = {inner * 2};
  const uint32_t box[2] = {box_inner, box_outer};
  return encode_tensor_map(cache, m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, base, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_128B);
}

// m-tiles per band: the ~148 tiles in flight cover kGroupM x (148 / kGroupM) tiles, and the whole B matrix is streamed
// from HBM once per band.  Swept on B200: 8 / 16 / 32 / 64 -> 1374 / 1415 / 1382 / 1322 TFLOP/s.
constexpr int kGroupM = 16;
// CTA-pair kernel: 16 bands of 256-row tiles = 4096 rows (a 42 MB A band at K = 5120).  Swept on B200 at the cfg 3 QKV
// shape (profiles/r2e_gemm_l2.md), DRAM reads / TFLOP/s: 8 -> 4.7 GB / 1449, 12 -> 3.7 / 1458, 16 -> 3.0-3.4 / 1497,
// 20 -> 5.8 / 1406, 24 -> 6.2 / 1411, 32 -> 12.9 / 1348 (a band beyond ~45 MB no longer stays in L2).
constexpr int kGroupM2 = 16;

template <int BN, int kMode, bool k2Cta>
cudaError_t launch(const GemmArgs& a, cudaStream_t stream) {
  GemmMaps maps;
  ChunkMaps cmaps;
  cudaError_t e = map2d(a.cache, &maps.b, a.b, static_cast<uint64_t>(a.K), static_cast<uint64_t>(a.N), kBK, k2Cta ? BN / 2 : BN);
  if (e != cudaSuccess) return e;
  GemmParams p{};
  const int n_out = a.N / a.n_per_out;
  if (kMode == kPlain) {
    e = map2d(a.cache, &maps.a, a.a, static_cast<uint64_t>(a.K), static_cast<uint64_t>(a.M), kBK, kBM);
    if (e != cudaSuccess) return e;
    for (int t = 0; t < 3; ++t) {
      // unused slots repeat slot 0 so that the struct holds valid descriptors only
      void* base = a.out[t < n_out ? t : 0];
      e = map2d(a.cache, &maps.out[t], base, static_cast<uint64_t>(a.n_per_out), static_cast<uint64_t>(a.M), 64, kBM);
      if (e != cudaSuccess) return e;
    }
    for (auto& m : cmaps.m) m = maps.b;
  } else {
    const GemmChunks& ck = *a.chunks;
    if (ck.C > kMaxChunks || ck.Hl > kMaxLocalHeads) return cudaErrorInvalidValue;
    if (kMode == kFusedOut) {
      e = map2d(a.cache, &maps.a, a.a, static_cast<uint64_t>(a.K), static_cast<uint64_t>(a.M), kBK, kBM);
    } else {
      maps.a = maps.b;
      e = map2d(a.cache, &maps.out[0], a.out[0], static_cast<uint64_t>(a.n_per_out), static_cast<uint64_t>(a.M), 64, kBM);
    }
    if (e != cudaSuccess) return e;
    for (int t = 0; t < 3; ++t)
      if (kMode == kFusedOut || t > 0) maps.out[t] = kMode == kFusedOut ? maps.a : maps.out[0];
    const int n_tensors = kMode == kFusedOut ? n_out : 1;
    for (auto& m : cmaps.m) m = maps.b;
    if (ck.peer) {
      // hcms_dist: tensor t, chunk c, destination rank p -> that rank's [rows][h_c][D] slice for THIS rank's tokens
      // (ck.peer[(t * C + c) * P + p], a.M rows: rows past the shard are clipped by the map)
      if (kMode != kFusedOut || n_tensors * ck.C * ck.P > kMaxFusedMaps) return cudaErrorInvalidValue;
      for (int i = 0; i < n_tensors * ck.C * ck.P; ++i) {
        const int c = (i / ck.P) % ck.C;
        const uint64_t dims[4] = {static_cast<uint64_t>(a.D), static_cast<uint64_t>(ck.h[c]), static_cast<uint64_t>(a.M), 1};
        const uint64_t strides[3] = {static_cast<uint64_t>(a.D) * 2, static_cast<uint64_t>(ck.h[c]) * a.D * 2,
                                     static_cast<uint64_t>(a.M) * ck.h[c] * a.D * 2};
        const uint32_t box[4] = {64, 1, kBM, 1};
        e = encode_tensor_map(a.cache, &cmaps.m[i], CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, ck.peer[i], dims, strides, box,
                              CU_TENSOR_MAP_SWIZZLE_128B);
        if (e != cudaSuccess) return e;
      }
    }
    for (int t = 0; t < n_tensors && !ck.peer; ++t)
      for (int c = 0; c < ck.C; ++c) {
        const uint64_t dims[4] = {static_cast<uint64_t>(a.D), static_cast<uint64_t>(ck.h[c]), static_cast<uint64_t>(a.M),
                                  static_cast<uint64_t>(ck.P)};
        const uint64_t strides[3] = {static_cast<uint64_t>(a.D) * 2, static_cast<uint64_t>(ck.h[c]) * a.D * 2,
                                     static_cast<uint64_t>(a.M) * ck.h[c] * a.D * 2};
        const uint32_t box[4] = {64, 1, kBM, 1};
        e = encode_tensor_map(a.cache, &cmaps.m[t * ck.C + c], CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, ck.base[t][c], dims, strides, box,
                              CU_TENSOR_MAP_SWIZZLE_128B);
        if (e != cudaSuccess) return e;
      }
    p.Hl = ck.Hl;
    p.C = ck.C;
    p.peer_n = ck.peer ? ck.P : 1;
    p.peer_on = ck.peer ? 1 : 0;
    for (int c = 0; c < ck.C; ++c)
      for (int j = 0; j < ck.h[c]; ++j) {
        p.chunk_of[ck.o[c] + j] = static_cast<uint8_t>(c);
        p.j_of[ck.o[c] + j] = static_cast<uint8_t>(j);
      }
  }
  p.d_shift = a.D == 128 ? 7 : 6;
  p.M = static_cast<int>(a.M);
  p.N = a.N;
  p.K = a.K;
  p.n_per_out = a.n_per_out;
  p.rope_outs = a.rope_outs;
  p.half_d = a.D / 2;
  p.d_mask = a.D - 1;
  p.cos = a.cos;
  p.sin = a.sin;
  p.n_tiles = a.N / BN;
  if (k2Cta) {
    p.m_tiles = static_cast<int>((a.M + 2 * kBM - 1) / (2 * kBM));     // 256-row tiles of a CTA pair
    p.group_m = kGroupM2;
    const int total = p.m_tiles * p.n_tiles, pairs = a.num_sms / 2;
    const int grid = 2 * (total < pairs ? total : pairs);
    gemm_bf16_nt_2cta_kernel<kMode><<<grid, kThreads, Cfg2::kSmemBytes, stream>>>(maps, cmaps, p);
  } else {
    p.m_tiles = static_cast<int>((a.M + kBM - 1) / kBM);
    p.group_m = kGroupM;
    const int total = p.m_tiles * p.n_tiles;
    const int grid = total < a.num_sms ? total : a.num_sms;
    gemm_bf16_nt_kernel<BN, kMode><<<grid, kThreads, Cfg<BN>::kSmemBytes, stream>>>(maps, cmaps, p);
  }
  return cudaGetLastError();
}

}  // namespace

static cudaError_t gemm_set_attributes() {
  cudaError_t status = cudaSuccess;
  auto set = [&](auto fn, int bytes) {
    if (status == cudaSuccess) status = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  };
  set(gemm_bf16_nt_kernel<256, kPlain>, Cfg<256>::kSmemBytes);
  set(gemm_bf16_nt_kernel<128, kPlain>, Cfg<128>::kSmemBytes);
  set(gemm_bf16_nt_kernel<256, kFusedOut>, Cfg<256>::kSmemBytes);
  set(gemm_bf16_nt_kernel<128, kFusedOut>, Cfg<128>::kSmemBytes);
  set(gemm_bf16_nt_kernel<256, kFusedA>, Cfg<256>::kSmemBytes);
  set(gemm_bf16_nt_kernel<128, kFusedA>, Cfg<128>::kSmemBytes);
  set(gemm_bf16_nt_2cta_kernel<kPlain>, Cfg2::kSmemBytes);
  set(gemm_bf16_nt_2cta_kernel<kFusedOut>, Cfg2::kSmemBytes);
  set(gemm_bf16_nt_2cta_kernel<kFusedA>, Cfg2::kSmemBytes);
  return status;
}

cudaError_t gemm_init() {
  static PerDeviceOnce once;
  return once_per_device(&once, gemm_set_attributes);
}

// Shape rules (checked by the callers in hcms_api.cu): K % 8 == 0 (16-byte row pitch), n_per_out % 128 == 0,
// N % n_per_out == 0, N / n_per_out <= 3, and with RoPE or a fused mode D in {64, 128}; fused modes: C <= 16, H/P <= 64.
cudaError_t launch_gemm(const GemmArgs& a, cudaStream_t stream) {
  cudaError_t e = gemm_init();
  if (e != cudaSuccess) return e;
  const bool wide = a.n_per_out % 256 == 0;
  if (wide && !a.one_cta) {   // CTA pairs (cta_group::2), 256 x 256 tiles: 1527 vs 1416 TFLOP/s on the cfg 3 QKV projection
    if (a.fuse == 1) return launch<256, kFusedOut, true>(a, stream);
    if (a.fuse == 2) return launch<256, kFusedA, true>(a, stream);
    return launch<256, kPlain, true>(a, stream);
  }
  if (a.fuse == 1) return wide ? launch<256, kFusedOut, false>(a, stream) : launch<128, kFusedOut, false>(a, stream);
  if (a.fuse == 2) return wide ? launch<256, kFusedA, false>(a, stream) : launch<128, kFusedA, false>(a, stream);
  return wide ? launch<256, kPlain, false>(a, stream) : launch<128, kPlain, false>(a, stream);
}

}  // namespace hcms
