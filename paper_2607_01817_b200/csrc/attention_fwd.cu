// Non-causal bf16 attention forward for one HCMS head chunk on sm_100a (tcgen05 / TMEM / TMA).
//
// Computes, for every logical rank p and local head j of the chunk (Eq. 2,
// Algorithm 1 line 15, bidirectional L43):
//     O'[p][i][j][:] = sum_k softmax_k(scale * Q'[p][i][j] . K'[p][k][j]) V'[p][k][j][:]
// on head-sharded buffers [P][S][h_c][D] (bf16 in, fp32 scores/softmax/accumulate, bf16 out).
//
// One CTA = one head x 256 query rows (two 128-row Q tiles), 384 threads:
//   warp 0      TMA producer: Q tiles once, then K/V tiles through a shared-memory ring, in the order the
//               tensor core first touches them (K_0, K_1, V_0, K_2, V_1, ...)
//   warp 1      MMA issuer (one lane): S_t = Q_t K_n^T (SS, M=128, N=128) and O_t += P_t V_n (TS: P_t is the A operand
//               in TENSOR memory, V_n MN-major in shared memory)
//   warp 2      TMEM allocator (512 columns: S at 0, P_0 / P_1 at 128 / 192, O_0 / O_1 at 256 / 256+D)
//   warps 4-7   softmax warpgroup of tile 0: one thread per query row; online softmax in fp32 with lazy
//   warps 8-11  softmax warpgroup of tile 1   rescaling of O (only when the row max grew by > 2^8); epilogue
//
// Why P lives in tensor memory.  With P staged in shared memory (round 1) the kernel sat at 98 % of the shared-memory
// data pipe (ncu: tensor-core operand reads 77 % + P stores 21 % of l1tex__data_pipe_*_wavefronts_mem_shared), i.e. 1280
// wavefronts per 1024 tensor-pipe cycles of every (Q tile, KV tile) pair: tensor activity could not exceed 80 %, and it
// measured 77-81 %.  As a TMEM A operand P costs neither the 32 KB store nor the 32 KB operand read: 768 wavefronts.
// TMEM has 512 columns and O_0, O_1 take 256 (D = 128), so the two P tiles (64 columns each, bf16 pairs) fit only if
// the two Q tiles SHARE one 128-column score buffer S.  They can, because a softmax warpgroup pulls S into registers
// within ~150 cycles and the tensor pipe runs a PV in between: the issue order per KV tile n is
//     QK_0(n) -> S     PV_1(n-2)     QK_1(n) -> S     PV_0(n-1)
// so that (a) the PV between two QKs covers the time the previous owner needs to empty S, and (b) every softmax has
// three MMA slots plus a whole iteration (~3000 cycles) between its scores and the PV that consumes its P.  P_t(n) is
// kept in registers until PV_t(n-1) has completed (pv_done), then written with two tcgen05.st.  V_m is used by PV_0(m)
// in iteration m+1 and PV_1(m) in iteration m+2, so K_n, V_{n-2}, V_{n-1} are live while K_{n+1}, V_n load: the ring has 5
// stages at D = 128 (the shared memory P used to take).
// Pair variant: the softmax warps of the peer CTA signal the leader's barriers with RELAXED cluster-scope arrives.  A
// release.cluster arrive costs a cluster-wide fence per warp and iteration (measured: 20.7 ms instead of 16.4 ms at
// BASELINE config 3).  What the leader's MMAs touch after the arrive is tensor memory of the arriving CTA (S columns
// already pulled out, ordered by tcgen05.wait::ld; P columns written, ordered by tcgen05.wait::st) followed by
// tcgen05.fence::before_thread_sync and the __syncwarp that precedes the arrive; the leader waits with acquire.cluster.
// tests/test_gpu_attention.py compares the pair kernel bit for bit with the single-CTA kernel at full size under NaN
// poisoning.
// The exponentials are split between the MUFU pipe (ex2.approx) and a degree-3 polynomial on the FMA pipe
// (packed f32x2 arithmetic), since 16 ex2/clk/SM would otherwise co-limit the kernel at exactly the MMA time.
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
constexpr int kThreads = 384;
constexpr int kTmemCols = 512;
constexpr float kRescaleThreshold = 8.0f;  // log2 units: rescale O only if the max grew by > 2^8
constexpr int kPanelBytes = 128 * 128;     // one 128-byte-swizzle panel: 128 rows x 128 B
constexpr int kPCols = kBN / 2;            // P_t in TMEM: 128 keys as bf16 pairs

// kPair: the CTA-pair variant (tcgen05 cta_group::2, D = 128 only).  Two CTAs of a cluster share every K_n / V_n tile:
// each loads HALF of it (64 of the 128 keys of K_n; 64 of the 128 head-dim columns of V_n) and the leader CTA issues
// M = 256 MMAs over both CTAs' query tiles, so per CTA the K/V traffic into and out of shared memory and the number
// of MMA instructions are halved.
template <int D, bool kPair = false>
struct Cfg {
  static constexpr int kPanels = D / 64;                    // 128-byte swizzle panels along D
  static constexpr int kTileBytes = kPanels * kPanelBytes;  // one Q / K / V tile
  static constexpr int kKvBytes = kPair ? kTileBytes / 2 : kTileBytes;   // what one ring stage holds
  static constexpr int kStages = D == 128 ? (kPair ? 10 : 5) : 8;         // KV ring stages (one K or one V (half) tile each)
  static constexpr int kSmemBytes = kQTiles * kTileBytes + kStages * kKvBytes + 1024 /*align*/ + 256 /*barriers*/;
  static constexpr int kTmemS = 0;                          // the score buffer both Q tiles take turns in
  static constexpr int kTmemP = kBN;                        // P_t at kTmemP + t*64
  static constexpr int kTmemO = 256;                        // O_t at kTmemO + t*D
  static_assert(kSmemBytes <= 227 * 1024, "shared memory budget");
};

// Shared-memory matrix descriptor, 128-byte swizzle (cute::UMMA::SmemDescriptor bit layout):
// [0,14) start>>4, [16,30) LBO>>4, [32,46) SBO>>4, [46,48) version=1, [61,64) layout=2 (SWIZZLE_128B),
// built as two 32-bit words: the high word is a constant, so per-MMA address stepping is one
// 32-bit add on the low word (shared-memory addresses are < 2^18, the start field never carries).
__host__ __device__ constexpr uint32_t desc_hi(uint32_t sbo_bytes) {
  return ((sbo_bytes >> 4) & 0x3FFF) | (1u << 14) | (2u << 29);
}
__device__ __forceinline__ uint32_t desc_lo(uint32_t smem_addr, uint32_t lbo_bytes) {
  return ((smem_addr >> 4) & 0x3FFF) | (((lbo_bytes >> 4) & 0x3FFF) << 16);
}

// Instruction descriptor for kind::f16: fp32 accumulate, bf16 A and B.
__host__ __device__ constexpr uint32_t make_idesc(int M, int N, bool b_mn_major) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn_major ? 1u : 0u) << 16) |
         (static_cast<uint32_t>(N >> 3) << 17) | (static_cast<uint32_t>(M >> 4) << 24);
}

struct alignas(64) AttnMaps {
  CUtensorMap q, k, v, o;   // rank-4 {D, h_c, S, P}, box {64, 1, 128, 1}, SWIZZLE_128B
  CUtensorMap kh;           // K with box {64, 1, 64, 1}: the half tile a CTA of a pair loads
  CUtensorMap op[kMaxPeers];   // fused output all-to-all: rank r's [push_rows][push_heads][D] output, rank-3 {D, heads, rows},
                               // box {64, 1, 128} (copies of o when unused)
};

struct AttnParams {
  int S;
  int n_kv;          // ceil(S/128)
  int h_c;
  float scale_log2;  // scale * log2(e)
  float* lse;        // optional [P*h_c][S]: log sum_k exp(scale q.k) per query row (natural log), for the backward
  int n_push;        // > 0: output tiles go to the n_push ranks' sequence-sharded outputs (AttnMaps::op), not to o
  int push_rows;     // tokens per rank
  int push_head0;    // global head of this launch's head 0
};

// ---- packed fp32x2 arithmetic (FFMA2 / FADD2 on sm_100) and helpers ----------------------------------
__device__ __forceinline__ uint64_t pack2(float lo, float hi) {
  uint64_t r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack2(uint64_t v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c) {
  uint64_t d;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
  return d;
}
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ uint64_t add2_rm(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("add.rm.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ uint64_t sub2(uint64_t a, uint64_t b) {
  uint64_t d;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
  return d;
}
__device__ __forceinline__ float max3(float a, float b, float c) {
  float d;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
  return d;
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

// 2^x for a pair on the FMA pipe: x = n + f (n = floor x via the 1.5*2^23 round-down trick), 2^f by a
// degree-3 polynomial with p(0) = 1 (max relative error 8.6e-5, far below P's bf16 rounding 2^-9), and
// n added into the exponent field.  x is clamped to >= -126 so that the exponent never underflows.
struct PolyConsts {
  uint64_t magic, c1, c2, c3, one;
};
__device__ __forceinline__ PolyConsts poly_consts() {
  PolyConsts c;
  c.magic = pack2(12582912.f, 12582912.f);
  c.c1 = pack2(0.6951168179512024f, 0.6951168179512024f);
  c.c2 = pack2(0.22764474153518677f, 0.22764474153518677f);
  c.c3 = pack2(0.07706727087497711f, 0.07706727087497711f);
  c.one = pack2(1.0f, 1.0f);
  return c;
}
__device__ __forceinline__ uint64_t exp2_poly2(float x0, float x1, const PolyConsts& c) {
  const uint64_t x = pack2(fmaxf(x0, -126.f), fmaxf(x1, -126.f));
  const uint64_t t = add2_rm(x, c.magic);
  const uint64_t f = sub2(x, sub2(t, c.magic));
  uint64_t p = fma2(f, c.c3, c.c2);
  p = fma2(p, f, c.c1);
  p = fma2(p, f, c.one);
  float p0, p1, t0, t1;
  unpack2(p, p0, p1);
  unpack2(t, t0, t1);
  p0 = __uint_as_float(__float_as_uint(p0) + (__float_as_uint(t0) << 23));
  p1 = __uint_as_float(__float_as_uint(p1) + (__float_as_uint(t1) << 23));
  return pack2(p0, p1);
}

__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}

// kPoly: of every 8 consecutive column pairs, this many take the polynomial path (the rest MUFU).
template <int D, int kPoly, bool kPair>
__global__ void __launch_bounds__(kThreads, 1)
attention_fwd_kernel(const __grid_constant__ AttnMaps maps, const AttnParams prm) {
  using C = Cfg<D, kPair>;
  constexpr int kStages = C::kStages;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t q_smem = smem_base;                                  // kQTiles Q tiles
  const uint32_t kv_smem = q_smem + kQTiles * C::kTileBytes;          // kStages K/V tiles
  const uint32_t bar_base = kv_smem + kStages * C::kKvBytes;          // 8-byte barriers
  const uint32_t bar_q_full = bar_base;                       // [2]  TMA -> MMA
  const uint32_t bar_kv_full = bar_q_full + 16;               // [kStages] TMA -> MMA
  const uint32_t bar_kv_empty = bar_kv_full + 8 * kStages;    // [kStages] MMA -> TMA
  const uint32_t bar_s_full = bar_kv_empty + 8 * kStages;     // [2]  MMA -> softmax: S_t(n) is in the score buffer
  const uint32_t bar_s_free = bar_s_full + 16;                // [2]  softmax -> MMA: S_t(n) is in registers, the buffer is free
  const uint32_t bar_p_full = bar_s_free + 16;                // [2]  softmax -> MMA: P_t(n) is in TMEM (O_t rescaled if needed)
  const uint32_t bar_pv_done = bar_p_full + 16;               // [2]  MMA -> softmax: PV_t(n) has completed
  const uint32_t tmem_slot = bar_pv_done + 16;                // 4 bytes

  const int warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);   // warp-uniform by construction
  const int lane = threadIdx.x & 31;
  const uint32_t cr = kPair ? cluster_ctarank() : 0u;   // rank in the CTA pair; the leader (0) issues the MMAs
  const int head = blockIdx.y;                 // p*h_c + j
  const int rank = head / prm.h_c;
  const int hj = head - rank * prm.h_c;
  const int q_row0 = blockIdx.x * (kQTiles * kBM);
  const int n_kv = prm.n_kv;

  if (threadIdx.x == 0) {
    for (int t = 0; t < kQTiles; ++t) {
      mbar_init(bar_q_full + 8 * t, 1);
      mbar_init(bar_s_full + 8 * t, 1);
      mbar_init(bar_s_free + 8 * t, kPair ? 8 : 4);     // one elected lane per softmax warp (of both CTAs of a pair)
      mbar_init(bar_p_full + 8 * t, kPair ? 8 : 4);
      mbar_init(bar_pv_done + 8 * t, 1);
    }
    for (int s = 0; s < kStages; ++s) {
      mbar_init(bar_kv_full + 8 * s, 1);
      mbar_init(bar_kv_empty + 8 * s, 1);
    }
    fence_mbar_init();
    fence_proxy_async_smem();
  }
  if (warp == 2) {
    if (kPair) {
      tmem_alloc_2sm(tmem_slot, kTmemCols);
      tmem_relinquish_2sm();
    } else {
      tmem_alloc(tmem_slot, kTmemCols);
      tmem_relinquish();
    }
  }
  tc_fence_before();
  if (kPair) cluster_sync(); else __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  if (warp < 4) {
    // ================================ producer / MMA warpgroup ================================
    // Both roles run warp-uniformly (all 32 lanes walk the loops and poll the barriers); only the TMA /
    // tcgen05 instructions themselves are guarded by elect.sync.  A whole role under `lane == 0` makes
    // ptxas wrap every uniform-datapath instruction in a divergence loop (~100 clk per MMA issue).
    setmaxnreg_dec<56>();
    if (warp == 0) {
      // ---------------- TMA producer ----------------
      const bool leader = elect_one();
      if (leader) {
        prefetch_tensormap(&maps.q);
        prefetch_tensormap(&maps.k);
        prefetch_tensormap(&maps.v);
      }
      // Pair: every byte count lives on the LEADER's barrier (both CTAs' TMA complete there); each CTA loads its own
      // Q rows, keys [j*128 + cr*64, +64) of K_j (D/64 panels of 64 rows) and head-dim columns [cr*64, +64) of V_j.
      auto load_tile = [&](const CUtensorMap* tm, uint32_t dst, uint32_t bar, int row0) {
        if (leader) {
          if (kPair) {
            if (cr == 0) mbar_expect_tx(bar, 2 * C::kTileBytes);
            const uint32_t bar0 = mapa(bar, 0);
#pragma unroll
            for (int pn = 0; pn < C::kPanels; ++pn) tma_load_4d_2sm(dst + pn * kPanelBytes, tm, bar0, pn * 64, hj, row0, rank);
          } else {
            mbar_expect_tx(bar, C::kTileBytes);
#pragma unroll
            for (int pn = 0; pn < C::kPanels; ++pn) tma_load_4d(dst + pn * kPanelBytes, tm, bar, pn * 64, hj, row0, rank);
          }
        }
        __syncwarp();
      };
      int stage = 0;
      uint32_t phase = 0;  // ring items are loaded in consumption order
      auto load_kv = [&](bool is_v, int j) {
        mbar_wait(bar_kv_empty + 8 * stage, phase ^ 1);
        const uint32_t dst = kv_smem + stage * C::kKvBytes, bar = bar_kv_full + 8 * stage;
        if (kPair) {
          if (leader) {
            if (cr == 0) mbar_expect_tx(bar, 2 * C::kKvBytes);
            const uint32_t bar0 = mapa(bar, 0);
            if (is_v) {
              tma_load_4d_2sm(dst, &maps.v, bar0, static_cast<int>(cr) * 64, hj, j * kBN, rank);
            } else {
#pragma unroll
              for (int pn = 0; pn < C::kPanels; ++pn)
                tma_load_4d_2sm(dst + pn * (kPanelBytes / 2), &maps.kh, bar0, pn * 64, hj, j * kBN + static_cast<int>(cr) * 64, rank);
            }
          }
          __syncwarp();
        } else {
          load_tile(is_v ? &maps.v : &maps.k, dst, bar, j * kBN);
        }
        if (++stage == kStages) {
          stage = 0;
          phase ^= 1;
        }
      };
      load_tile(&maps.q, q_smem, bar_q_full, q_row0);
      load_kv(false, 0);
      load_tile(&maps.q, q_smem + C::kTileBytes, bar_q_full + 8, q_row0 + kBM);
      for (int j = 0; j < n_kv; ++j) {
        if (j + 1 < n_kv) load_kv(false, j + 1);
        load_kv(true, j);
      }
    } else if (warp == 1 && (!kPair || cr == 0)) {
      // ---------------- MMA issuer (pair: the leader CTA issues M = 256 MMAs over both CTAs' query tiles) ----------------
      const bool leader = elect_one();
      constexpr uint32_t idesc_qk = make_idesc(kPair ? 2 * kBM : kBM, kBN, false);
      constexpr uint32_t idesc_pv = make_idesc(kPair ? 2 * kBM : kBM, D, true);
      constexpr uint32_t hi = desc_hi(1024);                 // SBO = 1024 B for every operand
      auto mma = [&](uint32_t d, uint32_t a_lo, uint32_t b_lo, uint32_t idesc, uint32_t acc) {
        if (kPair) mma_ss_lohi_2sm(d, a_lo, b_lo, hi, hi, idesc, acc); else mma_ss_lohi(d, a_lo, b_lo, hi, hi, idesc, acc);
      };
      auto commit = [&](uint32_t bar) {          // pair: the barrier at this offset in BOTH CTAs
        if (kPair) tc_commit_2sm(bar, 3); else tc_commit(bar);
      };
      auto wait_softmax = [&](uint32_t bar, uint32_t parity) {   // pair: arrivals come from both CTAs' softmax warps
        if (kPair) mbar_wait_cluster(bar, parity); else mbar_wait(bar, parity);
      };
      constexpr uint32_t kKPanel = kPair ? kPanelBytes / 2 : kPanelBytes;   // a K panel holds 64 or 128 keys
      auto issue_qk = [&](int t, uint32_t k_tile) {
        // S[128 x 128] = Q_t[128 x D] * K_n[128 x D]^T ; both operands K-major, 128B-swizzled panels
        const uint32_t d_tmem = tmem_base + C::kTmemS;
        const uint32_t q_lo = desc_lo(q_smem + t * C::kTileBytes, 16);
        const uint32_t k_lo = desc_lo(k_tile, 16);
#pragma unroll
        for (int ks = 0; ks < D / 16; ++ks) {
          const uint32_t off = ((ks >> 2) * kPanelBytes + (ks & 3) * 32) >> 4;
          const uint32_t k_off = ((ks >> 2) * kKPanel + (ks & 3) * 32) >> 4;
          mma(d_tmem, q_lo + off, k_lo + k_off, idesc_qk, ks > 0 ? 1u : 0u);
        }
      };
      auto issue_pv = [&](int t, uint32_t v_tile, bool accumulate) {
        // O_t[128 x D] += P_t[128 x 128 keys] * V_n[128 keys x D]; A = P_t in TMEM (bf16 pairs: 8 columns per K step of
        // 16 keys), B = V_n MN-major: 64-wide D panels (LBO = panel stride), 8-key groups 1024 B apart
        const uint32_t d_tmem = tmem_base + C::kTmemO + t * D;
        const uint32_t a_tmem = tmem_base + C::kTmemP + t * kPCols;
        const uint32_t v_lo = desc_lo(v_tile, kPanelBytes);
#pragma unroll
        for (int ks = 0; ks < kBN / 16; ++ks) {
          const uint32_t acc = (accumulate || ks > 0) ? 1u : 0u;
          if (kPair) mma_ts_lohi_2sm(d_tmem, a_tmem + ks * 8, v_lo + ks * (2048 >> 4), hi, idesc_pv, acc);
          else mma_ts_lohi(d_tmem, a_tmem + ks * 8, v_lo + ks * (2048 >> 4), hi, idesc_pv, acc);
        }
      };
      // The ring is a FIFO: tiles are first touched in load order (K_0, K_1, V_0, K_2, V_1, ...) and released in the same
      // order (K_n after QK_1(n); V_m after PV_1(m), two iterations after its K), so acquire and release keep their own
      // positions.
      int stage = 0, rel_stage = 0;
      uint32_t phase = 0;
      auto kv_acquire = [&]() -> uint32_t {
        mbar_wait(bar_kv_full + 8 * stage, phase);
        const uint32_t addr = kv_smem + stage * C::kKvBytes;
        if (++stage == kStages) {
          stage = 0;
          phase ^= 1;
        }
        return addr;
      };
      auto kv_release = [&]() {       // the oldest tile still held: free once every MMA issued so far has completed
        if (leader) commit(bar_kv_empty + 8 * rel_stage);
        __syncwarp();
        if (++rel_stage == kStages) rel_stage = 0;
      };
      auto qk_step = [&](int t, uint32_t k_tile) {
        tc_fence_after();
        if (leader) {
          issue_qk(t, k_tile);
          commit(bar_s_full + 8 * t);
        }
        __syncwarp();
      };
      auto pv_step = [&](int t, uint32_t v_tile, int m) {     // PV_t(m)
        wait_softmax(bar_p_full + 8 * t, m & 1);                // P_t(m) is in TMEM, O_t rescaled if needed
        tc_fence_after();
        if (leader) {
          issue_pv(t, v_tile, m > 0);
          commit(bar_pv_done + 8 * t);
        }
        __syncwarp();
      };

      mbar_wait(bar_q_full, 0);
      mbar_wait(bar_q_full + 8, 0);
      uint32_t v_prev = 0;                                      // V_{n-2} while iteration n runs: PV_1 still needs it
      for (int n = 0; n < n_kv; ++n) {
        const uint32_t k_tile = kv_acquire();
        if (n >= 1) wait_softmax(bar_s_free + 8, (n - 1) & 1);  // S_1(n-1) has left the score buffer
        qk_step(0, k_tile);
        if (n >= 2) {
          pv_step(1, v_prev, n - 2);
          kv_release();                                         // V_{n-2}
        }
        wait_softmax(bar_s_free, n & 1);                        // S_0(n) has left the score buffer
        qk_step(1, k_tile);
        kv_release();                                           // K_n
        if (n >= 1) {
          v_prev = kv_acquire();                                // V_{n-1}
          pv_step(0, v_prev, n - 1);
        }
      }
      if (n_kv >= 2) {
        pv_step(1, v_prev, n_kv - 2);
        kv_release();
      }
      {
        const uint32_t v_tile = kv_acquire();                   // V_{n_kv-1}
        pv_step(0, v_tile, n_kv - 1);
        pv_step(1, v_tile, n_kv - 1);
        kv_release();
      }
    }
    __syncwarp();
  } else {
    // ================================ softmax warpgroups ================================
    setmaxnreg_inc<224>();
    const int t = (warp >> 2) - 1;                       // Q tile of this warpgroup
    const int row = (warp & 3) * 32 + lane;              // row inside the tile == TMEM lane
    const uint32_t lane_addr = static_cast<uint32_t>((warp & 3) * 32) << 16;
    const uint32_t s_tmem = tmem_base + lane_addr + C::kTmemS;
    const uint32_t p_tmem = tmem_base + lane_addr + C::kTmemP + t * kPCols;
    const uint32_t o_tmem = tmem_base + lane_addr + C::kTmemO + t * D;
    const uint32_t swz = static_cast<uint32_t>(row & 7);
    const float scale_log2 = prm.scale_log2;
    const uint64_t scale2 = pack2(scale_log2, scale_log2);
    const int tail_valid = prm.S - (n_kv - 1) * kBN;     // valid keys in the last KV tile (1..128)
    const PolyConsts pc = poly_consts();

    float m_run = -INFINITY;   // running (possibly stale) row max, raw score units
    uint64_t l2 = pack2(0.f, 0.f), l2b = pack2(0.f, 0.f);   // running row sum, four partial lanes

    for (int j = 0; j < n_kv; ++j) {
      mbar_wait(bar_s_full + 8 * t, j & 1);
      tc_fence_after();
      uint32_t sr[kBN];
#pragma unroll
      for (int c4 = 0; c4 < kBN / 32; ++c4) tmem_ld32(s_tmem + c4 * 32, &sr[c4 * 32]);
      tmem_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {                                   // the other tile's QK may overwrite the score buffer now
        if (kPair) mbar_arrive_cluster_relaxed(mapa(bar_s_free + 8 * t, 0)); else mbar_arrive(bar_s_free + 8 * t);
      }
      if (j == n_kv - 1 && tail_valid < kBN) {
#pragma unroll
        for (int c = 0; c < kBN; ++c)
          if (c >= tail_valid) sr[c] = 0xff800000u;   // -inf: keys beyond S do not exist
      }
      float mx0 = __uint_as_float(sr[0]), mx1 = __uint_as_float(sr[1]);
      float mx2 = __uint_as_float(sr[2]), mx3 = __uint_as_float(sr[3]);
#pragma unroll
      for (int c = 4; c < kBN; c += 8) {
        mx0 = max3(mx0, __uint_as_float(sr[c]), __uint_as_float(sr[c + 1]));
        mx1 = max3(mx1, __uint_as_float(sr[c + 2]), __uint_as_float(sr[c + 3]));
        if (c + 4 < kBN) {
          mx2 = max3(mx2, __uint_as_float(sr[c + 4]), __uint_as_float(sr[c + 5]));
          mx3 = max3(mx3, __uint_as_float(sr[c + 6]), __uint_as_float(sr[c + 7]));
        }
      }
      const float m_tile = max3(mx0, mx1, fmaxf(mx2, mx3));
      if (j > 0) {
        const bool need = (m_tile - m_run) * scale_log2 > kRescaleThreshold;
        if (__any_sync(0xffffffffu, need)) {
          // O_t holds sum_k p_k V_k relative to m_run: once PV_t(j-1) has landed, rescale it to the new max
          mbar_wait(bar_pv_done + 8 * t, (j - 1) & 1);
          tc_fence_after();
          const float alpha = need ? ex2((m_run - m_tile) * scale_log2) : 1.0f;
          if (need) {
            l2 = fma2(l2, pack2(alpha, alpha), pack2(0.f, 0.f));
            l2b = fma2(l2b, pack2(alpha, alpha), pack2(0.f, 0.f));
            m_run = m_tile;
          }
          // 16 columns at a time: the 128 scores of the tile stay in registers beside them
#pragma unroll 1
          for (int c16 = 0; c16 < D / 16; ++c16) {
            uint32_t orr[16];
            tmem_ld16(o_tmem + c16 * 16, orr);
            tmem_wait_ld();
#pragma unroll
            for (int c = 0; c < 16; ++c) orr[c] = __float_as_uint(__uint_as_float(orr[c]) * alpha);
            tmem_st16(o_tmem + c16 * 16, orr);
          }
          tmem_wait_st();
          tc_fence_before();
        }
      } else {
        m_run = m_tile;
      }
      const float neg_m = -m_run * scale_log2;
      const uint64_t neg_m2 = pack2(neg_m, neg_m);
      // 64 key pairs: x = s*scale_log2 - m*scale_log2, p = 2^x, row sum in fp32, P rounded to bf16.  The packed tile
      // (64 registers, taking the place of the scores as they die) waits in registers for PV_t(j-1) to finish with
      // P_t's columns; by then that has normally happened (it was issued one to two iterations ago).
      uint32_t pw[kPCols];
#pragma unroll
      for (int pair = 0; pair < kPCols; ++pair) {
        const int c = pair * 2;
        const uint64_t x = fma2(pack2(__uint_as_float(sr[c]), __uint_as_float(sr[c + 1])), scale2, neg_m2);
        float x0, x1;
        unpack2(x, x0, x1);
        const uint64_t p = (pair & 7) < kPoly ? exp2_poly2(x0, x1, pc) : pack2(ex2(x0), ex2(x1));
        if (pair & 1) l2b = add2(l2b, p); else l2 = add2(l2, p);
        float p0, p1;
        unpack2(p, p0, p1);
        pw[pair] = pack_bf16(p0, p1);       // key 2*pair in the low half: column `pair` of the TMEM A operand
      }
      if (j > 0) {
        mbar_wait(bar_pv_done + 8 * t, (j - 1) & 1);
        tc_fence_after();
      }
      tmem_st32(p_tmem, pw);
      tmem_st32(p_tmem + 32, pw + 32);
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (kPair) mbar_arrive_cluster_relaxed(mapa(bar_p_full + 8 * t, 0)); else mbar_arrive(bar_p_full + 8 * t);
      }
    }

    // ---------------- epilogue: O_t / l -> bf16 -> swizzled smem (Q_t's tile: every QK_t has completed) -> TMA store ----------------
    mbar_wait(bar_pv_done + 8 * t, (n_kv - 1) & 1);
    tc_fence_after();
    float la, lb, lc, ld;
    unpack2(l2, la, lb);
    unpack2(l2b, lc, ld);
    const float l_sum = (la + lb) + (lc + ld);
    const float inv_l = 1.0f / l_sum;
    if (prm.lse != nullptr && q_row0 + t * kBM + row < prm.S)      // sum_k exp(s_k) = l * exp(m): lse = m*scale + log l
      prm.lse[static_cast<size_t>(head) * prm.S + q_row0 + t * kBM + row] =
          (m_run * scale_log2 + log2f(l_sum)) * 0.6931471805599453f;
    const uint32_t o_smem = q_smem + t * C::kTileBytes;
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
        st_shared_v4(o_smem + panel * kPanelBytes + row * 128 + ((chunk ^ swz) << 4), w[0], w[1], w[2], w[3]);
      }
    }
    fence_proxy_async_smem();
    named_bar_sync(1 + t, kBM);
    if ((warp & 3) == 0 && lane == 0) {
      const int row0 = q_row0 + t * kBM;
      if (row0 < prm.S) {
        if (prm.n_push > 0) {
          // Output all-to-all in the epilogue (Alg. 1 line 21 between real ranks): the tile's rows belong to
          // one or two destination ranks.  Every destination has kBM pad rows in front of its row 0 (a TMA store with a
          // negative start coordinate faults on sm_100: measured), so the second rank of a straddling tile receives the
          // tile's leading rows in its pad; rows past a rank's end (and rows >= S) are clipped by the tensor map.
          const int r_lo = row0 / prm.push_rows;
          int r_hi = (row0 + kBM - 1) / prm.push_rows;
          r_hi = r_hi < prm.n_push ? r_hi : prm.n_push - 1;
          for (int r = r_lo; r <= r_hi; ++r)
#pragma unroll
            for (int pn = 0; pn < C::kPanels; ++pn)
              tma_store_3d(&maps.op[r], o_smem + pn * kPanelBytes, pn * 64, prm.push_head0 + hj, row0 - r * prm.push_rows + kBM);
        } else {
#pragma unroll
          for (int pn = 0; pn < C::kPanels; ++pn)
            tma_store_4d(&maps.o, o_smem + pn * kPanelBytes, pn * 64, hj, row0, rank);
        }
        bulk_commit();
        bulk_wait<0>();
      }
    }
  }

  tc_fence_before();
  if (kPair) {       // neither CTA may exit while the pair's MMAs can still read its shared memory or signal its barriers
    cluster_sync();
    if (warp == 2) tmem_dealloc_2sm(tmem_base, kTmemCols);
  } else {
    __syncthreads();
    if (warp == 2) tmem_dealloc(tmem_base, kTmemCols);
  }
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
    cudaError_t e = encode_tensor_map(a.cache, outs[i], CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, ptrs[i], dims, strides, box,
                                      CU_TENSOR_MAP_SWIZZLE_128B);
    if (e != cudaSuccess) return e;
  }
  for (int r = 0; r < kMaxPeers; ++r) m->op[r] = m->o;
  if (a.o_push) {
    if (a.P != 1 || a.n_push < 1 || a.n_push > kMaxPeers || a.push_rows < 1) return cudaErrorInvalidValue;
    const uint64_t pdims[3] = {static_cast<uint64_t>(a.D), static_cast<uint64_t>(a.push_heads),
                               static_cast<uint64_t>(a.push_rows) + kBM};     // o_push[r] points at kBM pad rows before row 0
    const uint64_t pstrides[2] = {static_cast<uint64_t>(a.D) * 2, static_cast<uint64_t>(a.push_heads) * a.D * 2};
    const uint32_t pbox[3] = {64, 1, 128};
    for (int r = 0; r < a.n_push; ++r) {
      cudaError_t e = encode_tensor_map(a.cache, &m->op[r], CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, a.o_push[r], pdims, pstrides, pbox,
                                        CU_TENSOR_MAP_SWIZZLE_128B);
      if (e != cudaSuccess) return e;
    }
  }
  if (!a.pair) {        // only the CTA-pair kernel reads the half-tile map
    m->kh = m->k;
    return cudaSuccess;
  }
  const uint32_t box_half[4] = {64, 1, 64, 1};
  return encode_tensor_map(a.cache, &m->kh, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, a.k, dims, strides, box_half,
                           CU_TENSOR_MAP_SWIZZLE_128B);
}

// Of every 8 column pairs, kPolyPairs take their exponential on the FMA pipe (swept on B200 with this kernel, 40-step
// sustained runs at cfg 3: 0 / 1 / 2 / 3 / 4 -> 16.79 / 16.75 / 16.52 / 16.91 / 17.36 ms; at D = 64, cfg 2: 2 / 3 / 4 / 5 / 6 ->
// 0.294 / 0.294 / 0.306 / 0.334 / 0.362 ms: that shape is bound by the softmax warps' issue slots, not by MUFU;
// profiles/r2d_experiments.md)
constexpr int kPolyPairs = 2;

cudaError_t set_attributes() {
  cudaError_t e = cudaFuncSetAttribute(attention_fwd_kernel<128, kPolyPairs, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       Cfg<128>::kSmemBytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(attention_fwd_kernel<64, kPolyPairs, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           Cfg<64>::kSmemBytes);
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(attention_fwd_kernel<128, kPolyPairs, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              Cfg<128, true>::kSmemBytes);
}

}  // namespace

cudaError_t attention_init() {
  static PerDeviceOnce once;
  return once_per_device(&once, set_attributes);
}

cudaError_t launch_attention(const AttnArgs& a0, cudaStream_t stream) {
  AttnArgs a = a0;
  a.pair = a0.pair && a0.D == 128;
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
  prm.lse = a.lse;
  prm.n_push = a.o_push ? a.n_push : 0;
  prm.push_rows = static_cast<int>(a.push_rows);
  prm.push_head0 = a.push_head0;
  dim3 grid(static_cast<unsigned>((a.S + kQTiles * kBM - 1) / (kQTiles * kBM)), static_cast<unsigned>(a.P * a.h_c));
  if (a.pair) {
    // CTA pairs: a cluster of 2 consecutive CTAs (512 query rows) per launch unit; an odd block count is padded by
    // one CTA whose query rows do not exist (its loads are zero fill, its stores are skipped)
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((grid.x + 1) / 2 * 2, grid.y);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = Cfg<128, true>::kSmemBytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr{};
    attr.id = cudaLaunchAttributeClusterDimension;
    attr.val.clusterDim.x = 2;
    attr.val.clusterDim.y = 1;
    attr.val.clusterDim.z = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, attention_fwd_kernel<128, kPolyPairs, true>, maps, prm);
  }
  if (a.D == 128)
    attention_fwd_kernel<128, kPolyPairs, false><<<grid, kThreads, Cfg<128>::kSmemBytes, stream>>>(maps, prm);
  else if (a.D == 64)
    attention_fwd_kernel<64, kPolyPairs, false><<<grid, kThreads, Cfg<64>::kSmemBytes, stream>>>(maps, prm);
  else
    return cudaErrorInvalidValue;
  return cudaGetLastError();
}

}  // namespace hcms
