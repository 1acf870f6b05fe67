// TMA / mbarrier helpers (inline PTX, sm_100a) and the per-warp row-tile ring used by the
// aprod kernels.
//
// Row tile = 32 consecutive rows.  Its 24-coefficient records (32 x 192 B, contiguous in HBM) are
// fetched by ONE tensor-map TMA load whose box is 26 x 32 doubles on a tensor of extent 24 x M:
// columns 24,25 are out of bounds and zero-filled, so every row lands in shared memory with a
// 208-byte stride.  208 = 13 * 16, an odd number of 16-byte chunks, which makes the lane-per-row
// LDS.128 pattern (lane l reads chunk c of row l) bank-conflict free; a dense 192-byte stride
// would be a 4-way conflict.  Rows past M are zero-filled the same way (ragged tail).
// The 32 index records (32 x 32 B) follow with one 1-D bulk copy.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace gsr {

constexpr int TILE_ROWS = 32;
constexpr int ROW_STRIDE_D = 26;                               // doubles per staged row (24 + 2 zero pad)
constexpr int COEF_TILE_BYTES = TILE_ROWS * ROW_STRIDE_D * 8;  // 6656
constexpr int IDX_TILE_BYTES = TILE_ROWS * 32;                 // 1024
constexpr int STAGE_BYTES = COEF_TILE_BYTES + IDX_TILE_BYTES;  // 7680 (multiple of 128)

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
// 2-D tensor-map load global -> shared, completion on an mbarrier, L2 evict-first (streamed once)
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar,
                                            uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%2, %3}], [%4], %5;" ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}
// 1-D bulk copy global -> shared (bytes multiple of 16, both addresses 16-byte aligned)
__device__ __forceinline__ void bulk_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
          smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
      : "memory");
}

// Per-warp ring of `nstages` row tiles.  All 32 lanes call every method; lane 0 talks to the TMA.
struct TileRing {
  char* base;       // this warp's STAGES * STAGE_BYTES of shared memory (128-byte aligned)
  uint64_t* bars;   // this warp's STAGES mbarriers
  const CUtensorMap* map;
  const int32_t* idx;
  int64_t M, n_tiles, stride;   // stride = number of warps sharing the tile sequence
  int64_t next_issue;           // next tile this warp will request
  uint64_t policy;
  int stage;                    // stage of the next tile to consume
  int nstages;
  uint32_t phase;

  __device__ __forceinline__ void issue(int s, int64_t tile) {
    const int64_t row0 = tile * TILE_ROWS;
    const int64_t left = M - row0;
    const uint32_t idx_bytes = static_cast<uint32_t>((left < TILE_ROWS ? left : TILE_ROWS) * 32);
    char* dst = base + s * STAGE_BYTES;
    mbar_expect_tx(bars + s, COEF_TILE_BYTES + idx_bytes);
    tma_load_2d(dst, map, 0, static_cast<int>(row0), bars + s, policy);
    bulk_load_1d(dst + COEF_TILE_BYTES, idx + row0 * 8, idx_bytes, bars + s, policy);
  }

  __device__ __forceinline__ void init(char* smem_base, uint64_t* bar_base, const CUtensorMap* m, const int32_t* idx_,
                                       int64_t M_, int64_t first_tile, int64_t stride_, int lane, int nstages_) {
    base = smem_base; bars = bar_base; map = m; idx = idx_; M = M_; nstages = nstages_;
    n_tiles = (M_ + TILE_ROWS - 1) / TILE_ROWS;
    stride = stride_; next_issue = first_tile; stage = 0; phase = 0;
    policy = l2_policy_evict_first();
    // index areas start as all-zero records, so that the rows of a ragged last tile that the copy does
    // not cover always hold in-range indices (zeros or an earlier tile's records)
    for (int s = 0; s < nstages; s++)
      reinterpret_cast<int4*>(base + s * STAGE_BYTES + COEF_TILE_BYTES)[lane] = make_int4(0, 0, 0, 0),
      reinterpret_cast<int4*>(base + s * STAGE_BYTES + COEF_TILE_BYTES)[32 + lane] = make_int4(0, 0, 0, 0);
    if (lane == 0) {
      for (int s = 0; s < nstages; s++) mbar_init(bars + s, 1);
      mbar_fence_init();
    }
    __syncwarp();
    if (lane == 0) {
      fence_proxy_async();
      for (int s = 0; s < nstages; s++) {
        if (next_issue < n_tiles) issue(s, next_issue);
        next_issue += stride;
      }
    }
    next_issue = __shfl_sync(0xffffffffu, next_issue, 0);
  }

  // wait until the current tile has landed; returns its shared-memory address
  __device__ __forceinline__ char* acquire() {
    mbar_wait(bars + stage, phase);
    return base + stage * STAGE_BYTES;
  }
  // the warp is done with the current tile (it may have written into it: exchange runs, aprod_device.cuh):
  // order those generic-proxy accesses before the async-proxy refill, then request the next tile
  __device__ __forceinline__ void release(int lane) {
    __syncwarp();
    if (lane == 0 && next_issue < n_tiles) {
      fence_proxy_async();
      issue(stage, next_issue);
    }
    next_issue += stride;
    if (++stage == nstages) { stage = 0; phase ^= 1; }
  }
};

}  // namespace gsr
