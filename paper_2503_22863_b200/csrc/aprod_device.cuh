// Per-tile device routines shared by the aprod1, aprod2 and fused LSQR kernels.
// A tile is 32 rows staged in shared memory by TMA (tma.cuh): coefficients with a 208-byte row
// stride, then the 32 index records.
//
// What bounds these kernels on B200 is the number of L2 requests per row (each SM can send one
// request per cycle to the crossbar, each of the 184 L2 slices looks up one tag per cycle; ncu:
// l1tex__m_l1tex2xbar_req_cycles_active and lts__t_tag_requests both ~82 % with the previous
// design), not DRAM bytes.  So every block of a row is handled in the way that needs the fewest
// requests:
//   astro  : lanes of a warp share 1-2 stars -> L1 hits / a segmented warp reduction
//   att    : INTERLEAVED attitude layout  il[3*t + ax] = x_att[ax*K + t]: the 12 values a row needs
//            (3 axes x 4 knots from one start t) are ONE contiguous 96-byte run, fetched / reduced
//            by 12 consecutive lanes in one instruction (1-2 requests instead of 3-6)
//   instr  : shared memory when the slice fits, else L1/L2 gathers and L2 reductions
#pragma once
#include "gsr_internal.cuh"
#include "tma.cuh"

namespace gsr {

constexpr unsigned FULL = 0xffffffffu;

// streaming (single-use) 8-byte gather: do not allocate in L1 (keeps L1 for the instrumental slice)
#ifndef ATT_LD_MODE
#define ATT_LD_MODE 1
#endif
__device__ __forceinline__ double ld_nc_na(const double* p) {
#if ATT_LD_MODE == 0
  double v;
  asm("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
  return v;
#elif ATT_LD_MODE == 1
  return __ldg(p);
#elif ATT_LD_MODE == 2
  return *p;
#else
  return 1.0 + (double)(reinterpret_cast<uintptr_t>(p) & 8);   // experiment: no load at all
#endif
}

// What a kernel needs to gather from x (aprod 1 side).
struct GatherCtx {
  const double* x;          // the n-vector being multiplied (astro block at x, 5 per star)
  const double* att_il;     // attitude block of x in the interleaved layout, 3K doubles
  const double* xi_s;       // shared-memory copy of the instrumental slice, or nullptr
  const double* xi_g;       // x + oI
  double xg;                // x[oG] (0 when G = 0)
};

// The lane-per-row part of a staged tile in registers: astro, instrumental, global slots + indices.
struct RowRegs {
  double as[5];   // slots 0-4
  double ai[6];   // slots 17-22
  double ag;      // slot 23
  int4 i0, i1;    // {star, att_start, instr0, instr1}, {instr2..5}
};

// Lane l reads row l of the tile: conflict-free LDS.128 (208-byte stride), and the 32-byte index
// record as two LDS.128 issued in swizzled order (lanes 4-7, 12-15, ... read the second half
// first), which makes the 32-byte-stride pattern bank-conflict free.
// Tail lanes (row >= M) get zero coefficients (TMA zero fill) and an all-zero index record.
__device__ __forceinline__ void load_row(const char* tile, int lane, bool valid, RowRegs& r) {
  const double2* ap = reinterpret_cast<const double2*>(tile + lane * (ROW_STRIDE_D * 8));
  const double2 c0 = ap[0], c1 = ap[1], c2 = ap[2], c8 = ap[8], c9 = ap[9], c10 = ap[10], c11 = ap[11];
  r.as[0] = c0.x; r.as[1] = c0.y; r.as[2] = c1.x; r.as[3] = c1.y; r.as[4] = c2.x;
  r.ai[0] = c8.y; r.ai[1] = c9.x; r.ai[2] = c9.y; r.ai[3] = c10.x; r.ai[4] = c10.y; r.ai[5] = c11.x;
  r.ag = c11.y;
  const int4* ip = reinterpret_cast<const int4*>(tile + COEF_TILE_BYTES + lane * 32);
  const int sw = (lane >> 2) & 1;
  const int4 first = ip[sw], second = ip[sw ^ 1];
  r.i0 = sw ? second : first;
  r.i1 = sw ? first : second;
  if (!valid) { r.i0 = make_int4(0, 0, 0, 0); r.i1 = r.i0; }
}

// ---- attitude block, cooperative: half-warp h handles row 2*it + h in pass it (16 passes per tile);
// lane p = lane & 15 < 12 owns position p = 3*j + ax of the row's 96-byte run, i.e. coefficient slot
// 5 + 4*ax + j.  The LDS.64 of a pass is conflict free (each half-warp reads 12 distinct words-pairs
// of one row; the two halves are separate wavefronts).
struct AttLane {
  int h, p, slot;
  bool act;
  __device__ __forceinline__ explicit AttLane(int lane) {
    h = lane >> 4; p = lane & 15; act = p < 12;
    const int ax = p % 3, j = p / 3;
    slot = 5 + 4 * ax + j;
  }
};

// c[it] = the lane's attitude coefficient of pass it (0 for idle lanes and rows past the tile's end)
__device__ __forceinline__ void att_load_coefs(const char* tile, const AttLane& L, int nvalid, double (&c)[16]) {
  const double* td = reinterpret_cast<const double*>(tile);
#pragma unroll
  for (int it = 0; it < 16; it++) {
    const int row = 2 * it + L.h;
    c[it] = (L.act && row < nvalid) ? td[row * ROW_STRIDE_D + L.slot] : 0.0;
  }
}

// Attitude part of (A x)[row of this lane]: sum_{ax,j} a[r][5+4ax+j] * x_att[ax*K + t_r + j].
// 16 independent 8-byte gathers per lane are in flight at once; the 16 x 16 products of a half-warp
// are summed by a transposing butterfly (15 shuffle-adds instead of 16 x 4), after which lane p of
// half h holds the sum of row 2p + h; one more shuffle hands it to the lane that owns the row.
__device__ __forceinline__ double att_dot(const AttLane& L, int lane, int nvalid, int att_start,
                                          const double* __restrict__ att_il, const double (&c)[16]) {
  double v[16];
#pragma unroll
  for (int it = 0; it < 16; it++) {
    const int row = 2 * it + L.h;
    const int t = __shfl_sync(FULL, att_start, row);
    // unconditional load from a clamped address (a predicated load + select makes ptxas wait for each
    // load in turn: 16 serialised L2 round trips per tile); idle lanes read element 0 and are masked
    const bool ok = L.act && row < nvalid;
    const double xv = ld_nc_na(att_il + (ok ? 3 * (int64_t)t + L.p : 0));
    v[it] = ok ? c[it] * xv : 0.0;
  }
#pragma unroll
  for (int w = 8; w >= 1; w >>= 1) {
    const bool up = (lane & w) != 0;
#pragma unroll
    for (int i = 0; i < w; i++) {
      const double keep = up ? v[i + w] : v[i];
      const double send = up ? v[i] : v[i + w];
      v[i] = keep + __shfl_xor_sync(FULL, send, w);
    }
  }
  return __shfl_sync(FULL, v[0], (lane >> 1) | ((lane & 1) << 4));
}

// g_att(il)[3*t_r + p] += a[r][slot(p)] * y[r]  -- PAPER.md:49, Eq. (3), attitude block: per pass one
// red.global.add.f64 instruction whose 12 active lanes of each half-warp cover one contiguous run.
__device__ __forceinline__ void att_scatter(const AttLane& L, int nvalid, double yv, int att_start,
                                            double* __restrict__ gatt_il, const double (&c)[16]) {
#pragma unroll
  for (int it = 0; it < 16; it++) {
    const int row = 2 * it + L.h;
    const double yy = __shfl_sync(FULL, yv, row);
    const int t = __shfl_sync(FULL, att_start, row);
    if (L.act && row < nvalid) atomicAdd(gatt_il + 3 * (int64_t)t + L.p, c[it] * yy);
  }
}

// Astrometric + instrumental + global part of (A x)[row of this lane]   -- PAPER.md:45, Eq. (2).
template <bool INSTR_SMEM>
__device__ __forceinline__ double row_dot_rest(const RowRegs& r, const GatherCtx& c) {
  const double* xa = c.x + 5 * (int64_t)r.i0.x;
  double g[11];
#pragma unroll
  for (int k = 0; k < 5; k++) g[k] = __ldg(xa + k);
  {
    const int col[6] = {r.i0.z, r.i0.w, r.i1.x, r.i1.y, r.i1.z, r.i1.w};
#pragma unroll
    for (int q = 0; q < 6; q++) g[5 + q] = INSTR_SMEM ? c.xi_s[col[q]] : __ldg(c.xi_g + col[q]);
  }
  double acc0 = r.ag * c.xg, acc1 = 0.0;
  acc0 = fma(r.as[0], g[0], acc0); acc1 = fma(r.as[1], g[1], acc1);
  acc0 = fma(r.as[2], g[2], acc0); acc1 = fma(r.as[3], g[3], acc1);
  acc0 = fma(r.as[4], g[4], acc0);
  acc1 = fma(r.ai[0], g[5], acc1); acc0 = fma(r.ai[1], g[6], acc0);
  acc1 = fma(r.ai[2], g[7], acc1); acc0 = fma(r.ai[3], g[8], acc0);
  acc1 = fma(r.ai[4], g[9], acc1); acc0 = fma(r.ai[5], g[10], acc0);
  return acc0 + acc1;
}

// Where a kernel scatters to (aprod 2 side).
struct ScatterCtx {
  double* x;        // the n-vector being accumulated into (astro and global parts)
  double* gatt_il;  // attitude accumulator, interleaved layout, 3K doubles
  double* xins;     // instrumental accumulator in global memory: x + oI, or this CTA's private copy
  double* acc_s;    // shared-memory instrumental accumulator, or nullptr
};

// Astrometric, instrumental and global slots of the lane's own row, from registers.
//  astro  (slots 0-4)  : rows are sorted by star, so the lanes of a warp hold runs of equal star; a
//                        segmented warp scan (shuffles) sums each run, the run head issues 5 adds.
//  instr  (slots 17-22): block-privatised accumulators in shared memory when the slice fits (flushed
//                        once per CTA), else reductions at L2.
//  global (slot 23)    : returned as the lane's contribution, reduced once per CTA by the caller.
template <bool INSTR_SMEM>
__device__ __forceinline__ double scatter_row(const RowRegs& r, int lane, bool valid, double yv, const ScatterCtx& c) {
  const int star = valid ? r.i0.x : (-1 - lane);
  double p0 = r.as[0] * yv, p1 = r.as[1] * yv, p2 = r.as[2] * yv, p3 = r.as[3] * yv, p4 = r.as[4] * yv;
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const int so = __shfl_down_sync(FULL, star, off);
    const double q0 = __shfl_down_sync(FULL, p0, off), q1 = __shfl_down_sync(FULL, p1, off),
                 q2 = __shfl_down_sync(FULL, p2, off), q3 = __shfl_down_sync(FULL, p3, off),
                 q4 = __shfl_down_sync(FULL, p4, off);
    if (lane + off < 32 && so == star) { p0 += q0; p1 += q1; p2 += q2; p3 += q3; p4 += q4; }
  }
  const int sprev = __shfl_up_sync(FULL, star, 1);
  if (valid && (lane == 0 || sprev != star)) {   // head of a run of equal star
    double* xa = c.x + 5 * (int64_t)star;
    atomicAdd(xa, p0); atomicAdd(xa + 1, p1); atomicAdd(xa + 2, p2); atomicAdd(xa + 3, p3); atomicAdd(xa + 4, p4);
  }
  double gl = 0.0;
  if (valid) {
    double* t = INSTR_SMEM ? c.acc_s : c.xins;
    atomicAdd(t + r.i0.z, r.ai[0] * yv); atomicAdd(t + r.i0.w, r.ai[1] * yv); atomicAdd(t + r.i1.x, r.ai[2] * yv);
    atomicAdd(t + r.i1.y, r.ai[3] * yv); atomicAdd(t + r.i1.z, r.ai[4] * yv); atomicAdd(t + r.i1.w, r.ai[5] * yv);
    gl = r.ag * yv;
  }
  return gl;
}

// Shared-memory plan of the TMA kernels.
struct SmemPlan {
  int warps, stages;
  bool gather_smem;   // instrumental slice of x staged in shared memory (aprod 1 side)
  bool acc_smem;      // instrumental accumulators privatised in shared memory (aprod 2 side)
  size_t bytes;       // dynamic shared memory to request
};
enum { PLAN_APROD1 = 1, PLAN_APROD2 = 2, PLAN_FUSED = 3 };
SmemPlan plan_smem(const SysView& s, const Tuning& t, int what);

__device__ __forceinline__ char* smem_align128(char* p) { return p + ((128u - (smem_u32(p) & 127u)) & 127u); }

}  // namespace gsr
