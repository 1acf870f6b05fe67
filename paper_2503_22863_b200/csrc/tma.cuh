// TMA / mbarrier helpers (inline PTX, sm_100a) and the per-warp row-tile ring used by the
// aprod kernels.
//
// Row tile = 32 consecutive rows.  Its 24-coefficient records (32 x 192 B, contiguous in HBM) are
// fetched by ONE tensor-map TMA load.  The tensor view pairs the rows: extent 48 x floor(M/2) doubles,
// i.e. one tensor row = two matrix rows = 384 B = three whole 128-byte lines, so the stream costs 1.5 L2
// requests per matrix row (a 24 x M view with 192-byte tensor rows costs 2-3).  The box is 50 x 16:
// columns 48,49 are out of bounds and zero-filled, so every PAIR lands in shared memory with a 400-byte
// stride and the rows of a pair 192 B apart.  400 = 25 * 16 and 192 = 12 * 16 make the lane-per-row
// LDS.128 pattern (lane l reads chunk c of row l) bank-conflict free: the 16-byte chunk positions
// (25 * (l >> 1) + 12 * (l & 1) + c) mod 8 take each value exactly four times over a warp.  Pairs past
// floor(M/2) are zero-filled the same way (ragged tail); the last row of an odd M is copied by the warp
// itself (TileRing::acquire).  The 32 index records (32 x 32 B) follow with one 1-D bulk copy.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace gsr {

constexpr int TILE_ROWS = 32;
constexpr int COEF_TILE_BYTES = 6400;                          // staged coefficients of a tile, either record format
constexpr int IDX_TILE_BYTES = TILE_ROWS * 32;                 // 1024
constexpr int STAGE_BYTES = COEF_TILE_BYTES + IDX_TILE_BYTES;  // 7424 (multiple of 128)

// How the records of a tile lie in shared memory, per record format.  A GROUP of consecutive rows is one row of the
// tensor view (a whole number of 16-byte units in HBM, which cuTensorMapEncodeTiled needs for its pitch); the box is a
// few columns wider than the group, the out-of-bounds columns are zero-filled, and that pad (i) sets the group stride in
// shared memory so that the lane-per-row loads are bank-conflict free and (ii) holds the group's y values (y_off).
//   Rec24: 24 doubles per row (192 B).  Group = 2 rows = 384 B = three whole 128-byte lines; box 50 x 16; group stride
//          400 B, rows 192 B apart: every row is 16-byte aligned, LDS.128 per lane, the chunk positions
//          (25 * (l >> 1) + 12 * (l & 1) + c) mod 8 take each value exactly four times over a warp.
//   Rec23: 23 doubles per row (184 B, the production record without the global slot).  184 B is 8-byte
//          aligned only and 2 rows (368 B) are no whole number of 16-byte units, but 4 rows are: group = 4 rows = 736 B,
//          view 92 x floor(M/4), box 100 x 8; group stride 800 B, rows 184 B apart.  Odd rows of a group are 8-byte
//          aligned only, so the lanes use LDS.64: in 8-byte units lane l reads (100 * (l >> 2) + 23 * (l & 3) + c), and
//          {4 g + 7 i mod 16 : g, i < 4} are 16 different values, i.e. each half-warp (one 128-byte wavefront of 8-byte
//          accesses) touches 16 different bank pairs: conflict free.
struct Rec24 {
  static constexpr int CPR = 24, GROUP = 2, GROUP_SHIFT = 1, GROUP_BYTES = 400, BOX_COLS = 50, VIEW_COLS = 48;
  static constexpr bool VEC16 = true;
  __host__ __device__ static constexpr int row_off(int r) { return (r >> 1) * GROUP_BYTES + (r & 1) * 192; }
  __host__ __device__ static constexpr int y_off(int r) { return (r >> 1) * GROUP_BYTES + 384 + (r & 1) * 8; }
  // row 2 * it + h (h = 0, 1), the row a half-warp serves in pass `it` of the cooperative attitude routines
  __host__ __device__ static constexpr int coop_off(int it, int h) { return it * GROUP_BYTES + h * 192; }
};
struct Rec23 {
  static constexpr int CPR = 23, GROUP = 4, GROUP_SHIFT = 2, GROUP_BYTES = 800, BOX_COLS = 100, VIEW_COLS = 92;
  static constexpr bool VEC16 = false;
  __host__ __device__ static constexpr int row_off(int r) { return (r >> 2) * GROUP_BYTES + (r & 3) * 184; }
  __host__ __device__ static constexpr int y_off(int r) { return (r >> 2) * GROUP_BYTES + 736 + (r & 3) * 8; }
  __host__ __device__ static constexpr int coop_off(int it, int h) { return (it >> 1) * GROUP_BYTES + ((it & 1) * 2 + h) * 184; }
};
static_assert((TILE_ROWS / Rec24::GROUP) * Rec24::GROUP_BYTES == COEF_TILE_BYTES, "Rec24 tile");
static_assert((TILE_ROWS / Rec23::GROUP) * Rec23::GROUP_BYTES == COEF_TILE_BYTES, "Rec23 tile");

#ifdef GSR_HOST_EMULATION
// tests/emu: the same helpers for the host build of the kernels (test infrastructure; never part of libgsr.so).
// The copies complete at issue time, so the mbarrier calls reduce to a warp barrier on the waiting side.
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return static_cast<uint32_t>(reinterpret_cast<uintptr_t>(p)); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int) { *bar = 0; }
__device__ __forceinline__ void mbar_fence_init() {}
__device__ __forceinline__ void mbar_expect_tx(uint64_t*, uint32_t) {}
__device__ __forceinline__ void mbar_wait(uint64_t*, uint32_t) { __syncwarp(); }
__device__ __forceinline__ void fence_proxy_async() {}
__device__ __forceinline__ uint64_t l2_policy_evict_first() { return 0; }
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int c0, int c1, uint64_t*, uint64_t) {
  emu::tensor_load_2d(dst, map, c0, c1);
}
__device__ __forceinline__ void bulk_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t*, uint64_t) {
  emu::bulk_copy(dst, src, bytes);
}
#else
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
#endif  // GSR_HOST_EMULATION

// Per-warp ring of `nstages` row tiles.  All 32 lanes call every method; lane 0 talks to the TMA.
template <class REC>
struct TileRing {
  char* base;       // this warp's STAGES * STAGE_BYTES of shared memory (128-byte aligned)
  uint64_t* bars;   // this warp's STAGES mbarriers
  const CUtensorMap* map;
  const double* vals;
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
    const bool pairs = row0 + (REC::GROUP - 1) < M;   // the tile holds at least one whole group (else: only rows the warp copies)
    mbar_expect_tx(bars + s, (pairs ? COEF_TILE_BYTES : 0) + idx_bytes);
    if (pairs) tma_load_2d(dst, map, 0, static_cast<int>(row0 >> REC::GROUP_SHIFT), bars + s, policy);
    bulk_load_1d(dst + COEF_TILE_BYTES, idx + row0 * 8, idx_bytes, bars + s, policy);
  }

  __device__ __forceinline__ void init(char* smem_base, uint64_t* bar_base, const CUtensorMap* m, const double* vals_,
                                       const int32_t* idx_, int64_t M_, int64_t first_tile, int64_t stride_, int lane,
                                       int nstages_) {
    base = smem_base; bars = bar_base; map = m; vals = vals_; idx = idx_; M = M_; nstages = nstages_;
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

  // wait until tile t (the current one) has landed; returns its shared-memory address
  __device__ __forceinline__ char* acquire(int64_t t, int lane) {
    mbar_wait(bars + stage, phase);
    char* tile = base + stage * STAGE_BYTES;
    if (REC::GROUP == 2) {
      if ((M & 1) && t == n_tiles - 1) {
        // odd M: the last row has no partner, so the pair view does not cover it.  The warp copies it
        // (and clears the coefficient area first when the tile is that single row and no TMA load ran).
        const int last = static_cast<int>(M - 1 - t * TILE_ROWS);
        if (last == 0)
          for (int i = lane; i < COEF_TILE_BYTES / 16; i += 32) reinterpret_cast<int4*>(tile)[i] = make_int4(0, 0, 0, 0);
        __syncwarp();
        if (lane < 24) reinterpret_cast<double*>(tile + REC::row_off(last))[lane] = vals[(M - 1) * 24 + lane];
        __syncwarp();
      }
    } else if ((M & (REC::GROUP - 1)) && t == n_tiles - 1) {
      // the last M mod GROUP rows have no whole group, so the tensor view does not cover them.  The warp copies
      // them (and clears the coefficient area first when the tile holds nothing else and no TMA load ran).
      const int64_t tail0 = M & ~static_cast<int64_t>(REC::GROUP - 1);   // first row of the tail; it lies in this, the last, tile
      const int first = static_cast<int>(tail0 - t * TILE_ROWS);
      if (first == 0)
        for (int i = lane; i < COEF_TILE_BYTES / 16; i += 32) reinterpret_cast<int4*>(tile)[i] = make_int4(0, 0, 0, 0);
      __syncwarp();
      for (int64_t r = tail0; r < M; r++)
        if (lane < REC::CPR)
          reinterpret_cast<double*>(tile + REC::row_off(first + static_cast<int>(r - tail0)))[lane] = vals[r * REC::CPR + lane];
      __syncwarp();
    }
    return tile;
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
