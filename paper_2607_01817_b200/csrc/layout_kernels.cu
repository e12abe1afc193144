// All-to-all layout kernels: the on-device stand-in for Ulysses' input / output all-to-all
// (Algorithm 1 lines 8 and 21) for ONE head chunk.
//
//   scatter:  dense[p][s][j][d] = strided[s][p*Hl + o_c + j][d]      (input all-to-all)
//   gather :  strided[s][p*Hl + o_c + j][d] = dense[p][s][j][d]      (output all-to-all + Concat)
//
// "strided" is the global [S,H,D] tensor (the P ranks' shards back to back), "dense" the
// head-sharded chunk buffer [P][S][h_c][D].  Pure byte movement: every element is read once
// and written once, so the roofline is HBM bandwidth (2*P*S*h_c*D*es bytes per tensor).
//
// Two variants, same bits out:
//   * vec: 256-bit ld.global.nc / st.global (LDG.256 / STG.256; 128-bit if a pointer is only 16-byte
//          aligned), four independent requests per thread, one launch for Q,K,V (grid.z), thread order
//          following the contiguous side; no shared memory, so its CTAs fit beside a resident attention CTA;
//   * tma: one elected thread per CTA drives a ring of shared-memory stages: a TMA bulk-tensor
//          load of a [rows][h_c][D] box per (rank, head-chunk) tile, then a bulk store of the
//          now contiguous tile (scatter), or the reverse (gather).  Few registers, no LSU work.
#include "hcms_internal.h"
#include "ptx.cuh"

namespace hcms {
using namespace ptx;

// ------------------------------------------------------------------------------------------
// vec variant
// ------------------------------------------------------------------------------------------
struct LayoutVecParams {
  const uint8_t* src[3];
  uint8_t* dst[3];
  uint32_t n_per_rank;       // S * run_vecs  (vectors of one rank's dense block)
  uint32_t run_vecs;         // h_c*D*es / vector bytes  (contiguous run in the strided tensor)
  uint32_t row_stride_vecs;  // H*D*es / vector bytes
  uint32_t rank_stride_vecs; // Hl*D*es / vector bytes
  uint32_t chunk_off_vecs;   // o_c*D*es / vector bytes
  uint32_t step_rows;        // kVecThreads / run_vecs : how far a thread's next vector lies, in rows ...
  uint32_t step_cols;        // kVecThreads % run_vecs : ... and in vectors inside the run
};

// Distributed form (hcms_dist.cu, Alg. 1 lines 8 and 21 between P real ranks): the dense block
// of logical rank p is the address peer[t][p] -- a row range of rank p's own chunk buffer, reached through a
// CUDA-IPC / peer mapping -- instead of dense base + p * n_per_rank.  Scatter = PUSH (local strided shard -> stores
// into every peer's chunk buffer), gather = PULL (loads from every peer's O'_c -> local strided shard).
struct LayoutPeerTable {
  uint8_t* peer[3][kMaxPeers];   // kMaxPeers: hcms_internal.h
};

// 128-bit and 256-bit (sm_100: LDG.256 / STG.256) streaming accesses that stay out of L1
struct alignas(16) Vec16 {
  uint32_t v[4];
};
struct alignas(32) Vec32 {
  uint32_t v[8];
};
__device__ __forceinline__ void ld_stream(const uint8_t* p, Vec16& r) {
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.v[0]), "=r"(r.v[1]), "=r"(r.v[2]), "=r"(r.v[3])
               : "l"(p));
}
__device__ __forceinline__ void st_stream(uint8_t* p, const Vec16& r) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(r.v[0]), "r"(r.v[1]), "r"(r.v[2]),
               "r"(r.v[3])
               : "memory");
}
__device__ __forceinline__ void ld_stream(const uint8_t* p, Vec32& r) {
  asm volatile("ld.global.nc.L1::no_allocate.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r.v[0]), "=r"(r.v[1]), "=r"(r.v[2]), "=r"(r.v[3]), "=r"(r.v[4]), "=r"(r.v[5]), "=r"(r.v[6]),
                 "=r"(r.v[7])
               : "l"(p));
}
__device__ __forceinline__ void st_stream(uint8_t* p, const Vec32& r) {
  asm volatile("st.global.L1::no_allocate.v8.u32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(r.v[0]), "r"(r.v[1]),
               "r"(r.v[2]), "r"(r.v[3]), "r"(r.v[4]), "r"(r.v[5]), "r"(r.v[6]), "r"(r.v[7])
               : "memory");
}

constexpr int kVecThreads = 256;
constexpr int kVecUnroll = 4;

// Thread order follows the dense (contiguous) side: vector i of a rank's dense block is row s = i / run_vecs,
// column w = i % run_vecs of the run.  One division per thread; the thread's next vectors lie kVecThreads
// further, i.e. (step_rows, step_cols) further with a carry.  All loads are issued before the first store.
template <bool kGather, typename Vec, bool kPeer>
__device__ __forceinline__ void layout_vec_body(const LayoutVecParams& p, const LayoutPeerTable* tab) {
  const uint32_t rank = blockIdx.y;
  // selects, not p.src[blockIdx.z]: a dynamically indexed kernel parameter is copied to the stack
  const uint32_t z = blockIdx.z;
  const uint8_t* __restrict__ src = z == 0 ? p.src[0] : (z == 1 ? p.src[1] : p.src[2]);
  uint8_t* __restrict__ dst = z == 0 ? p.dst[0] : (z == 1 ? p.dst[1] : p.dst[2]);
  if (kPeer) {   // the dense side is rank `rank`'s buffer: one indexed constant-bank load of its address
    uint8_t* dense = tab->peer[z][rank];
    if (kGather) src = dense; else dst = dense;
  }
  // Programmatic dependent launch: a layout kernel that directly follows another kernel in its stream may be placed on
  // the SMs while that kernel drains (its blocks compute their addresses, then wait here until the predecessor has
  // completed and its writes are visible).  One chunk's copy is a 30-90 us kernel, so the launch gap and the ramp that
  // this hides are 5-8 % of it.  Without the launch attribute, or behind an event wait or a copy, both are no-ops.
  asm volatile("griddepcontrol.launch_dependents;");
  const uint32_t i0 = blockIdx.x * (kVecThreads * kVecUnroll) + threadIdx.x;
  const size_t dense_base = kPeer ? 0 : static_cast<size_t>(rank) * p.n_per_rank;
  const size_t strided_base = static_cast<size_t>(rank) * p.rank_stride_vecs + p.chunk_off_vecs;
  uint32_t s = i0 / p.run_vecs;
  uint32_t w = i0 - s * p.run_vecs;

  Vec val[kVecUnroll];
  size_t out_idx[kVecUnroll];
  asm volatile("griddepcontrol.wait;" ::: "memory");
#pragma unroll
  for (int u = 0; u < kVecUnroll; ++u) {
    const uint32_t i = i0 + u * kVecThreads;
    if (i < p.n_per_rank) {
      const size_t strided = static_cast<size_t>(s) * p.row_stride_vecs + strided_base + w;
      const size_t dense = dense_base + i;
      ld_stream(src + (kGather ? dense : strided) * sizeof(Vec), val[u]);
      out_idx[u] = kGather ? strided : dense;
    }
    s += p.step_rows;
    w += p.step_cols;
    if (w >= p.run_vecs) {
      w -= p.run_vecs;
      s += 1;
    }
  }
#pragma unroll
  for (int u = 0; u < kVecUnroll; ++u) {
    const uint32_t i = i0 + u * kVecThreads;
    if (i < p.n_per_rank) st_stream(dst + out_idx[u] * sizeof(Vec), val[u]);
  }
}

template <bool kGather, typename Vec>
__global__ void __launch_bounds__(kVecThreads) layout_vec_kernel(const LayoutVecParams p) {
  layout_vec_body<kGather, Vec, false>(p, nullptr);
}
template <bool kGather, typename Vec>
__global__ void __launch_bounds__(kVecThreads)
layout_vec_peer_kernel(const LayoutVecParams p, const __grid_constant__ LayoutPeerTable tab) {
  layout_vec_body<kGather, Vec, true>(p, &tab);
}

cudaError_t launch_layout_vec(const LayoutArgs& a, cudaStream_t stream) {
  LayoutVecParams p{};
  const size_t run_bytes = static_cast<size_t>(a.h_c) * a.D * a.es;
  // 256-bit accesses when every address is 32-byte aligned (runs are multiples of 128 B for D >= 64), else 128-bit
  bool wide = run_bytes % 32 == 0 && (static_cast<size_t>(a.D) * a.es) % 32 == 0;
  const bool peer = a.peer[0] != nullptr;
  if (peer && a.P > kMaxPeers) return cudaErrorInvalidValue;
  LayoutPeerTable tab{};
  for (int t = 0; t < a.n_tensors; ++t) {
    // peer form: the strided side is src (scatter) / dst (gather); the dense side comes from the table
    const void* strided = a.gather ? a.dst[t] : a.src[t];
    if (peer) {
      wide = wide && reinterpret_cast<uintptr_t>(strided) % 32 == 0;
      for (int r = 0; r < a.P; ++r) {
        tab.peer[t][r] = static_cast<uint8_t*>(a.peer[t][r]);
        wide = wide && reinterpret_cast<uintptr_t>(a.peer[t][r]) % 32 == 0;
      }
    } else {
      wide = wide && reinterpret_cast<uintptr_t>(a.src[t]) % 32 == 0 && reinterpret_cast<uintptr_t>(a.dst[t]) % 32 == 0;
    }
  }
  const size_t vb = wide ? 32 : 16;
  const size_t n_per_rank = static_cast<size_t>(a.S) * (run_bytes / vb);
  if (run_bytes % vb || n_per_rank >= (1ull << 31)) return cudaErrorInvalidValue;
  for (int t = 0; t < a.n_tensors; ++t) {
    p.src[t] = static_cast<const uint8_t*>(a.src[t]);
    p.dst[t] = static_cast<uint8_t*>(a.dst[t]);
  }
  p.n_per_rank = static_cast<uint32_t>(n_per_rank);
  p.run_vecs = static_cast<uint32_t>(run_bytes / vb);
  p.row_stride_vecs = static_cast<uint32_t>(static_cast<size_t>(a.H) * a.D * a.es / vb);
  p.rank_stride_vecs = static_cast<uint32_t>(static_cast<size_t>(a.Hl) * a.D * a.es / vb);
  p.chunk_off_vecs = static_cast<uint32_t>(static_cast<size_t>(a.o_c) * a.D * a.es / vb);
  p.step_rows = kVecThreads / p.run_vecs;
  p.step_cols = kVecThreads % p.run_vecs;
  const uint32_t per_block = kVecThreads * kVecUnroll;
  dim3 grid((p.n_per_rank + per_block - 1) / per_block, a.P, a.n_tensors);
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = dim3(kVecThreads);
  cfg.stream = stream;
  cudaLaunchAttribute attr{};
  attr.id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr.val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = &attr;
  cfg.numAttrs = 1;
  if (peer) {
    if (a.gather)
      return wide ? cudaLaunchKernelEx(&cfg, layout_vec_peer_kernel<true, Vec32>, p, tab)
                  : cudaLaunchKernelEx(&cfg, layout_vec_peer_kernel<true, Vec16>, p, tab);
    return wide ? cudaLaunchKernelEx(&cfg, layout_vec_peer_kernel<false, Vec32>, p, tab)
                : cudaLaunchKernelEx(&cfg, layout_vec_peer_kernel<false, Vec16>, p, tab);
  }
  if (a.gather)
    return wide ? cudaLaunchKernelEx(&cfg, layout_vec_kernel<true, Vec32>, p) : cudaLaunchKernelEx(&cfg, layout_vec_kernel<true, Vec16>, p);
  return wide ? cudaLaunchKernelEx(&cfg, layout_vec_kernel<false, Vec32>, p) : cudaLaunchKernelEx(&cfg, layout_vec_kernel<false, Vec16>, p);
}

// ------------------------------------------------------------------------------------------
// tma variant
// ------------------------------------------------------------------------------------------
struct alignas(64) LayoutTmaMaps {
  CUtensorMap strided[3];   // rank-3 maps over the global [S][H][D] tensors, box [rows][h_c][D]
};

struct LayoutTmaParams {
  const uint8_t* dense_src[3];  // gather: dense buffers read with cp.async.bulk
  uint8_t* dense_dst[3];        // scatter: dense buffers written with cp.async.bulk
  int64_t S;
  int P, Hl, o_c, n_tensors;
  int rows;                     // rows per tile (box dim 2)
  uint32_t row_bytes;           // h_c*D*es
  uint32_t tiles_per_rank;      // ceil(S/rows)
  uint32_t n_tiles;             // n_tensors*P*tiles_per_rank
};

constexpr int kTmaStages = 4;

template <bool kGather>
__global__ void __launch_bounds__(32) layout_tma_kernel(const __grid_constant__ LayoutTmaMaps maps,
                                                         const LayoutTmaParams p) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t full_bar[kTmaStages];
  if (threadIdx.x != 0) return;

  const uint32_t tile_bytes = static_cast<uint32_t>(p.rows) * p.row_bytes;
  const uint32_t smem_base = (smem_u32(smem_raw) + 127u) & ~127u;
  for (int s = 0; s < kTmaStages; ++s) mbar_init(smem_u32(&full_bar[s]), 1);
  fence_mbar_init();
  fence_proxy_async_smem();

  const uint32_t first = blockIdx.x, step = gridDim.x;
  const uint32_t my_tiles = first < p.n_tiles ? (p.n_tiles - first + step - 1) / step : 0;

  auto issue_load = [&](uint32_t k) {
    const uint32_t tile = first + k * step;
    const uint32_t stage = k % kTmaStages;
    const uint32_t t = tile / (p.P * p.tiles_per_rank);
    const uint32_t rem = tile - t * (p.P * p.tiles_per_rank);
    const uint32_t rank = rem / p.tiles_per_rank;
    const uint32_t rt = rem - rank * p.tiles_per_rank;
    const int64_t s0 = static_cast<int64_t>(rt) * p.rows;
    const uint32_t dst = smem_base + stage * tile_bytes;
    const uint32_t bar = smem_u32(&full_bar[stage]);
    if (!kGather) {
      mbar_expect_tx(bar, tile_bytes);  // OOB rows are zero-filled and still counted
      tma_load_3d(dst, &maps.strided[t], bar, 0, static_cast<int>(rank * p.Hl + p.o_c), static_cast<int>(s0));
    } else {
      const int64_t rows_valid = (p.S - s0) < p.rows ? (p.S - s0) : p.rows;
      const uint32_t bytes = static_cast<uint32_t>(rows_valid) * p.row_bytes;
      const uint8_t* src = p.dense_src[t] + (static_cast<size_t>(rank) * p.S + s0) * p.row_bytes;
      mbar_expect_tx(bar, bytes);
      bulk_load(dst, src, bytes, bar);
    }
  };

  const uint32_t prologue = my_tiles < kTmaStages ? my_tiles : kTmaStages;
  for (uint32_t k = 0; k < prologue; ++k) issue_load(k);

  for (uint32_t k = 0; k < my_tiles; ++k) {
    const uint32_t tile = first + k * step;
    const uint32_t stage = k % kTmaStages;
    const uint32_t t = tile / (p.P * p.tiles_per_rank);
    const uint32_t rem = tile - t * (p.P * p.tiles_per_rank);
    const uint32_t rank = rem / p.tiles_per_rank;
    const uint32_t rt = rem - rank * p.tiles_per_rank;
    const int64_t s0 = static_cast<int64_t>(rt) * p.rows;
    const uint32_t src = smem_base + stage * tile_bytes;
    mbar_wait(smem_u32(&full_bar[stage]), (k / kTmaStages) & 1);
    if (!kGather) {
      const int64_t rows_valid = (p.S - s0) < p.rows ? (p.S - s0) : p.rows;
      const uint32_t bytes = static_cast<uint32_t>(rows_valid) * p.row_bytes;
      uint8_t* dst = p.dense_dst[t] + (static_cast<size_t>(rank) * p.S + s0) * p.row_bytes;
      bulk_store(dst, src, bytes);
    } else {
      tma_store_3d(&maps.strided[t], src, 0, static_cast<int>(rank * p.Hl + p.o_c), static_cast<int>(s0));
    }
    bulk_commit();
    // stage (k-1)%N is free once the store issued in iteration k-1 has finished reading it
    if (k >= 1 && (k - 1 + kTmaStages) < my_tiles) {
      bulk_wait_read<1>();
      issue_load(k - 1 + kTmaStages);
    }
  }
  bulk_wait<0>();
}

cudaError_t launch_layout_tma(const LayoutArgs& a, cudaStream_t stream, int num_sms) {
  const uint32_t row_bytes = static_cast<uint32_t>(a.h_c) * a.D * a.es;
  if (row_bytes % 16 || a.D > 256) return cudaErrorInvalidValue;
  // ~16 KB tiles: 4 stages x 16 KB x 3 CTAs/SM = 192 KB in flight per SM
  int rows = static_cast<int>(16384 / row_bytes);
  if (rows < 1) rows = 1;
  if (rows > 256) rows = 256;
  LayoutTmaMaps maps;
  LayoutTmaParams p{};
  const CUtensorMapDataType dt = a.es == 2 ? CU_TENSOR_MAP_DATA_TYPE_UINT16 : CU_TENSOR_MAP_DATA_TYPE_UINT32;
  for (int t = 0; t < a.n_tensors; ++t) {
    const void* strided = a.gather ? a.dst[t] : a.src[t];
    const uint64_t dims[3] = {static_cast<uint64_t>(a.D), static_cast<uint64_t>(a.H), static_cast<uint64_t>(a.S)};
    const uint64_t strides[2] = {static_cast<uint64_t>(a.D) * a.es, static_cast<uint64_t>(a.H) * a.D * a.es};
    const uint32_t box[3] = {static_cast<uint32_t>(a.D), static_cast<uint32_t>(a.h_c), static_cast<uint32_t>(rows)};
    cudaError_t e = encode_tensor_map(a.cache, &maps.strided[t], dt, 3, strided, dims, strides, box, CU_TENSOR_MAP_SWIZZLE_NONE);
    if (e != cudaSuccess) return e;
    p.dense_src[t] = static_cast<const uint8_t*>(a.src[t]);
    p.dense_dst[t] = static_cast<uint8_t*>(a.dst[t]);
  }
  for (int t = a.n_tensors; t < 3; ++t) maps.strided[t] = maps.strided[0];
  p.S = a.S;
  p.P = a.P;
  p.Hl = a.Hl;
  p.o_c = a.o_c;
  p.n_tensors = a.n_tensors;
  p.rows = rows;
  p.row_bytes = row_bytes;
  p.tiles_per_rank = static_cast<uint32_t>((a.S + rows - 1) / rows);
  p.n_tiles = static_cast<uint32_t>(a.n_tensors) * a.P * p.tiles_per_rank;
  const size_t smem = static_cast<size_t>(kTmaStages) * rows * row_bytes + 128;
  static PerDeviceOnce once;
  cudaError_t ea = once_per_device(&once, [] {
    cudaError_t e = cudaFuncSetAttribute(layout_tma_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(layout_tma_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
  });
  if (ea != cudaSuccess) return ea;
  uint32_t grid = static_cast<uint32_t>(num_sms) * 3;
  if (grid > p.n_tiles) grid = p.n_tiles;
  if (a.gather)
    layout_tma_kernel<true><<<grid, 32, smem, stream>>>(maps, p);
  else
    layout_tma_kernel<false><<<grid, 32, smem, stream>>>(maps, p);
  return cudaGetLastError();
}

}  // namespace hcms
