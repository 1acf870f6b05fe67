// Per-tile device routines shared by the aprod1, aprod2 and fused LSQR kernels.
// A tile is 32 rows staged in shared memory by TMA (tma.cuh): coefficients with a 208-byte row
// stride, then the 32 index records.
#pragma once
#include "gsr_internal.cuh"
#include "tma.cuh"

namespace gsr {

enum { ATT_FULL = 1, ATT_HALF = 2 };

__device__ __forceinline__ void ld_nc_v4(const double* p, double& a, double& b, double& c, double& d) {
  asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}

// What a kernel needs to gather from x (aprod 1 side).
struct GatherCtx {
  const double* x;          // the n-vector being multiplied
  const double* xw;         // expanded attitude windows built from x (k_expand_att)
  int64_t xw_axis_stride;   // doubles between axes in xw
  const double* xi_s;       // shared-memory copy of the instrumental slice, or nullptr
  const double* xi_g;       // x + oI
  double xg;                // x[oG] (0 when G = 0)
};

// One row of a staged tile in registers (lane-per-row).
struct RowRegs {
  double a[NSLOT];
  int4 i0, i1;   // {star, att_start, instr0, instr1}, {instr2..5}
};

// Lane l reads row l of the tile: 12 conflict-free LDS.128 for the coefficients (208-byte stride), and
// the 32-byte index record as two LDS.128 issued in swizzled order (lanes 4-7, 12-15, ... read the
// second half first), which makes the 32-byte-stride pattern bank-conflict free.
// Tail lanes (row >= M) get zero coefficients (TMA zero fill) and an all-zero index record.
__device__ __forceinline__ void load_row(const char* tile, int lane, bool valid, RowRegs& r) {
  const double2* ap = reinterpret_cast<const double2*>(tile + lane * (ROW_STRIDE_D * 8));
#pragma unroll
  for (int q = 0; q < NSLOT / 2; q++) {
    const double2 v = ap[q];
    r.a[2 * q] = v.x;
    r.a[2 * q + 1] = v.y;
  }
  const int4* ip = reinterpret_cast<const int4*>(tile + COEF_TILE_BYTES + lane * 32);
  const int sw = (lane >> 2) & 1;
  const int4 first = ip[sw], second = ip[sw ^ 1];
  r.i0 = sw ? second : first;
  r.i1 = sw ? first : second;
  if (!valid) { r.i0 = make_int4(0, 0, 0, 0); r.i1 = r.i0; }
}

// (A x)[row of this lane]   -- PAPER.md:45, Eq. (2).
// Gathers (the L1 tag stage serves ~1 random line per cycle per SM, measured 284 G gathers/s
// chip-wide whatever the access width, so the number of gather instructions per row is what counts):
//   astro  : x[5*star .. +4]   (rows are sorted by star: the lanes of a warp share 1-2 stars)
//   att    : 32-byte loads from the expanded window table:
//              ATT_FULL : xw[ax][t] = x[t..t+3] for every start t        -> 1 load per axis
//              ATT_HALF : xw[ax][j] = x[2j..2j+3] (even starts only)     -> 1 load (even start) or 2
//                         (odd start); half the footprint, for tables that would not stay L2-resident
//                         at full expansion (96 MB at K = 1e6 thrashed L2: +96 B/row of DRAM reads)
//   instr  : shared-memory copy of the instrumental slice when it fits, else L2 gathers
//   global : one register.
template <int ATT, bool INSTR_SMEM>
__device__ __forceinline__ double row_dot(const RowRegs& r, const GatherCtx& c) {
  const double* a = r.a;
  const double* xa = c.x + 5 * (int64_t)r.i0.x;
  double g[NSLOT - 1];
#pragma unroll
  for (int k = 0; k < 5; k++) g[k] = __ldg(xa + k);
  if (ATT == ATT_FULL) {
    const double* w0 = c.xw + (int64_t)r.i0.y * 4;
    ld_nc_v4(w0, g[5], g[6], g[7], g[8]);
    ld_nc_v4(w0 + c.xw_axis_stride, g[9], g[10], g[11], g[12]);
    ld_nc_v4(w0 + 2 * c.xw_axis_stride, g[13], g[14], g[15], g[16]);
  } else {
    const bool odd = r.i0.y & 1;
    const double* w0 = c.xw + (int64_t)(r.i0.y >> 1) * 4;
#pragma unroll
    for (int ax = 0; ax < 3; ax++) {
      double e0, e1, e2, e3, f0 = 0.0, f1 = 0.0, f2 = 0.0, f3 = 0.0;
      ld_nc_v4(w0 + ax * c.xw_axis_stride, e0, e1, e2, e3);               // x[2j .. 2j+3]
      if (odd) ld_nc_v4(w0 + ax * c.xw_axis_stride + 4, f0, f1, f2, f3);  // x[2j+2 .. 2j+5]
      g[5 + 4 * ax] = odd ? e1 : e0;
      g[6 + 4 * ax] = odd ? e2 : e1;
      g[7 + 4 * ax] = odd ? e3 : e2;
      g[8 + 4 * ax] = odd ? f2 : e3;
    }
  }
  {
    const int col[6] = {r.i0.z, r.i0.w, r.i1.x, r.i1.y, r.i1.z, r.i1.w};
#pragma unroll
    for (int q = 0; q < 6; q++) g[17 + q] = INSTR_SMEM ? c.xi_s[col[q]] : __ldg(c.xi_g + col[q]);
  }
  double acc0 = a[23] * c.xg, acc1 = 0.0, acc2 = 0.0;
#pragma unroll
  for (int k = 0; k < 21; k += 3) {
    acc0 = fma(a[k], g[k], acc0);
    acc1 = fma(a[k + 1], g[k + 1], acc1);
    acc2 = fma(a[k + 2], g[k + 2], acc2);
  }
  acc0 = fma(a[21], g[21], acc0);
  acc1 = fma(a[22], g[22], acc1);
  return (acc0 + acc1) + acc2;
}

// Where a kernel scatters to (aprod 2 side).
struct ScatterCtx {
  double* x;        // the n-vector being accumulated into (astro and global parts)
  double* xatt;     // x + oA
  double* xins;     // instrumental accumulator in global memory: x + oI, or this CTA's private copy
  double* acc_s;    // shared-memory instrumental accumulator, or nullptr
  int64_t K;
};

// x[col(r,k)] += a[r][k] * yv  for the 32 rows of a tile  -- PAPER.md:49, Eq. (3).
// yv = the lane's (scaled) y value, 0 for tail lanes; nvalid = rows of the tile that exist.
//
// Attitude (slots 5-16): the 12 x 32 products are walked so that 4 consecutive lanes cover one
// 4-knot run: its fp64 reductions then travel to L2 as one request (measured 2.2x the add rate of
// lane-per-row issue).  Pass `it` handles axis it%3 of rows 8*(it/3) .. +7; each half-warp takes the
// rows of one parity (r, r+2, r+4, r+6): with the 208-byte row stride their 32-byte runs fall in
// disjoint banks, so the LDS.64 is conflict free.  att_start and y come by shuffle from the lane that
// owns the row.
__device__ __forceinline__ void scatter_att(const char* tile, int lane, int nvalid, double yv, int att_start,
                                            const ScatterCtx& c) {
  const double* td = reinterpret_cast<const double*>(tile);
  const int sub = 2 * ((lane >> 2) & 3) + (lane >> 4);   // row within the group of 8
  const int j = lane & 3;
#pragma unroll
  for (int it = 0; it < 12; it++) {
    const int ax = it % 3, row = 8 * (it / 3) + sub;
    const double yy = __shfl_sync(0xffffffffu, yv, row);
    const int att = __shfl_sync(0xffffffffu, att_start, row);
    if (row < nvalid) {
      const double a = td[row * ROW_STRIDE_D + 5 + 4 * ax + j];
      atomicAdd(c.xatt + (int64_t)ax * c.K + att + j, a * yy);
    }
  }
}

// Astrometric, instrumental and global slots of the lane's own row, from registers.
//  astro  (slots 0-4)  : rows are sorted by star, so the lanes of a warp hold runs of equal star; a
//                        segmented warp scan (shuffles) sums each run, the run head issues 5 adds.
//  instr  (slots 17-22): block-privatised accumulators in shared memory when the slice fits (flushed
//                        once per CTA), else reductions at L2.
//  global (slot 23)    : returned as the lane's contribution, reduced once per CTA by the caller.
template <bool INSTR_SMEM>
__device__ __forceinline__ double scatter_row(const RowRegs& r, int lane, bool valid, double yv, const ScatterCtx& c) {
  const int star = valid ? r.i0.x : (-1 - lane);
  double p0 = r.a[0] * yv, p1 = r.a[1] * yv, p2 = r.a[2] * yv, p3 = r.a[3] * yv, p4 = r.a[4] * yv;
#pragma unroll
  for (int off = 1; off < 32; off <<= 1) {
    const int so = __shfl_down_sync(0xffffffffu, star, off);
    const double q0 = __shfl_down_sync(0xffffffffu, p0, off), q1 = __shfl_down_sync(0xffffffffu, p1, off),
                 q2 = __shfl_down_sync(0xffffffffu, p2, off), q3 = __shfl_down_sync(0xffffffffu, p3, off),
                 q4 = __shfl_down_sync(0xffffffffu, p4, off);
    if (lane + off < 32 && so == star) { p0 += q0; p1 += q1; p2 += q2; p3 += q3; p4 += q4; }
  }
  const int sprev = __shfl_up_sync(0xffffffffu, star, 1);
  if (valid && (lane == 0 || sprev != star)) {   // head of a run of equal star
    double* xa = c.x + 5 * (int64_t)star;
    atomicAdd(xa, p0); atomicAdd(xa + 1, p1); atomicAdd(xa + 2, p2); atomicAdd(xa + 3, p3); atomicAdd(xa + 4, p4);
  }
  double gl = 0.0;
  if (valid) {
    double* t = INSTR_SMEM ? c.acc_s : c.xins;
    atomicAdd(t + r.i0.z, r.a[17] * yv); atomicAdd(t + r.i0.w, r.a[18] * yv); atomicAdd(t + r.i1.x, r.a[19] * yv);
    atomicAdd(t + r.i1.y, r.a[20] * yv); atomicAdd(t + r.i1.z, r.a[21] * yv); atomicAdd(t + r.i1.w, r.a[22] * yv);
    gl = r.a[23] * yv;
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
