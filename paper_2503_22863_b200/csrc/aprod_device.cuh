// Per-tile device routines shared by the aprod1, aprod2 and fused LSQR kernels.
// A tile is 32 rows staged in shared memory by TMA (tma.cuh): coefficients in groups of rows (REC = Rec24: 16 pairs
// with a 400-byte stride; REC = Rec23: 8 groups of four 184-byte rows with an 800-byte stride), then the 32 index
// records.  Every routine that touches the staged tile is a template on REC.
//
// What bounds these kernels on B200 at C4 is the number of requests that leave the SM per row (one per clock
// into the crossbar, an fp64 reduction counting ~1.65), not DRAM bytes and not shared-memory
// wavefronts (taking 27 of a tile's 267 away changed the fused pass by 0.4 %: shared-memory work runs in the
// shadow of the requests).  So every block of a row is handled in the way that needs the fewest requests, and
// whatever can stay in shared memory does:
//   astro  : lanes of a warp share 1-2 stars -> L1 hits on the gather side; on the scatter side the
//            per-star sums of a tile are ONE small matrix product (star indicator x coefficients) done
//            with eight fp64 DMMA.8x8x4, so no shuffles and 2 reduction instructions per tile
//   att    : INTERLEAVED attitude layout  il[3*t + ax] = x_att[ax*K + t]: the 12 values a row needs
//            (3 axes x 4 knots from one start t) are ONE contiguous 96-byte run, fetched / reduced
//            by 12 consecutive lanes in one instruction (1-2 requests instead of 3-6).  The run is
//            handed between those 12 lanes and the lane that owns the row through the row's own
//            staged record in shared memory (the "exchange run"), not through shuffles
//   instr  : shared memory when the slice fits, else L1/L2 gathers and L2 reductions
#pragma once
#include "gsr_internal.cuh"
#include "tma.cuh"

namespace gsr {

constexpr unsigned FULL = 0xffffffffu;

// 8-byte gather through the read-only path (measured the same with L1::no_allocate, with plain ld.global and
// with an L2 evict-last policy on the attitude table: profiles/r01_summary.md section 3)
__device__ __forceinline__ double ld_nc_na(const double* p) { return __ldg(p); }

#ifdef GSR_HOST_EMULATION
// (tests/emu: host build of the kernels; an atomic add stands in for the L2 reduction)
__device__ __forceinline__ void red_add(double* p, double v, const std::source_location loc = std::source_location::current()) {
  atomicAdd(p, v, loc);
}
__device__ __forceinline__ void red_add_if_ge(double* p, double v, int a, int b,
                                              const std::source_location loc = std::source_location::current()) {
  if (a >= b) atomicAdd(p, v, loc);
}
#else
// fp64 reduction at L2, fire and forget.  Explicitly .global: a pointer that was read from a table in
// shared memory would otherwise compile to a GENERIC atomic (no RED, address-space check per lane).
__device__ __forceinline__ void red_add(double* p, double v) {
  asm volatile("red.global.add.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory");
}

// the same, predicated on a >= b (no branch: keeps a run of reductions back to back in the instruction stream)
__device__ __forceinline__ void red_add_if_ge(double* p, double v, int a, int b) {
  asm volatile("{\n.reg .pred q;\nsetp.ge.s32 q, %2, %3;\n@q red.global.add.f64 [%0], %1;\n}" ::"l"(p), "d"(v), "r"(a), "r"(b) : "memory");
}
#endif

// What a kernel needs to gather from x (aprod 1 side).
struct GatherCtx {
  const double* x;          // the n-vector being multiplied (astro block at x, 5 per star)
  const double* att_il;     // attitude block of x in the interleaved layout, 3K doubles
  const double* xi_s;       // shared-memory copy of the instrumental slice, or nullptr
  const double* xi_g;       // x + oI
  double xg;                // x[oG] (0 when G = 0)
};

// A staged row: its coefficients at REC::row_off(r) of the tile (tma.cuh).  Once the owning lane holds the row
// in registers, bytes [XOFF, XOFF+96) of the record (attitude slots 1-11 + instrumental slot 0) are
// reused as the row's EXCHANGE RUN: 12 doubles in run order p = 3*j + ax (coefficient slot 5 + 4*ax + j).
// Rec24: 16-byte aligned, so the owner moves it with 6 conflict-free LDS.128 / STS.128; Rec23: 8-byte aligned (12
// LDS.64 / STS.64).  The cooperative lanes use one LDS.64 / STS.64 per row either way.  The 8 bytes at REC::y_off(r)
// (zero pad of the TMA box) carry the row's y value for the astrometric matrix product.  Bytes [0, 40) (astro
// slots) stay intact.
constexpr int XOFF = 48;

// The lane-per-row view of a staged tile in registers: all 24 coefficients + the index record.
struct RowRegs {
  double a[NSLOT];
  int4 i0, i1;    // {star, att_start, instr0, instr1}, {instr2..5}
};

// Lane l reads row l of the tile: conflict-free LDS.128 (Rec24) or LDS.64 (Rec23; slot 23 reads as 0), and the
// 32-byte index record as two LDS.128 issued in swizzled order (lanes 4-7, 12-15, ... read the second half
// first), which makes the 32-byte-stride pattern bank-conflict free.
// Tail lanes (row >= M) get zero coefficients (TMA zero fill) and an all-zero index record.
template <class REC>
__device__ __forceinline__ void load_row(const char* tile, int lane, bool valid, RowRegs& r) {
  if (REC::VEC16) {
    const double2* ap = reinterpret_cast<const double2*>(tile + REC::row_off(lane));
#pragma unroll
    for (int q = 0; q < NSLOT / 2; q++) {
      const double2 c = ap[q];
      r.a[2 * q] = c.x;
      r.a[2 * q + 1] = c.y;
    }
  } else {
    const double* ap = reinterpret_cast<const double*>(tile + REC::row_off(lane));
#pragma unroll
    for (int k = 0; k < REC::CPR; k++) r.a[k] = ap[k];
#pragma unroll
    for (int k = REC::CPR; k < NSLOT; k++) r.a[k] = 0.0;
  }
  const int4* ip = reinterpret_cast<const int4*>(tile + COEF_TILE_BYTES + lane * 32);
  const int sw = (lane >> 2) & 1;
  const int4 first = ip[sw], second = ip[sw ^ 1];
  r.i0 = sw ? second : first;
  r.i1 = sw ? first : second;
  if (!valid) { r.i0 = make_int4(0, 0, 0, 0); r.i1 = r.i0; }
}

// ---- attitude block, cooperative side: half-warp h handles row 2*it + h in pass it (16 passes per
// tile); lane p = lane & 15 < 12 owns position p of the row's 96-byte run.
struct AttLane {
  int h, p;
  bool act;
  __device__ __forceinline__ explicit AttLane(int lane) { h = lane >> 4; p = lane & 15; act = p < 12; }
};

// t[it] = att_start of the row this lane serves in pass it, read from the staged index records (a
// half-warp broadcast), which nothing overwrites.  Rows past the end of the matrix (ragged last tile)
// carry zero coefficients (TMA zero fill) and whatever VALID index record the stage held before (the
// index areas are zeroed at kernel start, TileRing::init): they gather in range and scatter zeros.
__device__ __forceinline__ void att_starts(const char* tile, const AttLane& L, int (&t)[16]) {
#pragma unroll
  for (int it = 0; it < 16; it++)
    t[it] = *reinterpret_cast<const int*>(tile + COEF_TILE_BYTES + (2 * it + L.h) * 32 + 4);
}

// Gather side: exchange run of row <- x_att(il)[3*t_row .. +12).  16 independent 8-byte loads per lane
// in flight at once.  Call after every lane has loaded its row (a __syncwarp()).
template <class REC>
__device__ __forceinline__ void att_gather(char* tile, const AttLane& L, const int (&t)[16],
                                           const double* __restrict__ att_il) {
  if (L.act) {
    double v[16];
#pragma unroll
    for (int it = 0; it < 16; it++) v[it] = ld_nc_na(att_il + 3 * (int64_t)t[it] + L.p);
#pragma unroll
    for (int it = 0; it < 16; it++)
      *reinterpret_cast<double*>(tile + REC::coop_off(it, L.h) + XOFF + 8 * L.p) = v[it];
  }
}

// Owner side: sum_{ax,j} a[r][5+4ax+j] * x_att[ax*K + t_r + j] from the row's exchange run.
template <class REC>
__device__ __forceinline__ double att_dot_row(const char* tile, int lane, const RowRegs& r) {
  double xv[12];
  if (REC::VEC16) {
    const double2* xr = reinterpret_cast<const double2*>(tile + REC::row_off(lane) + XOFF);
#pragma unroll
    for (int q = 0; q < 6; q++) {
      const double2 c = xr[q];
      xv[2 * q] = c.x;
      xv[2 * q + 1] = c.y;
    }
  } else {
    const double* xr = reinterpret_cast<const double*>(tile + REC::row_off(lane) + XOFF);
#pragma unroll
    for (int q = 0; q < 12; q++) xv[q] = xr[q];
  }
  double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0;
#pragma unroll
  for (int j = 0; j < 4; j++) {   // run positions 3j, 3j+1, 3j+2 = axes 0, 1, 2 of knot j
    acc0 = fma(r.a[5 + j], xv[3 * j], acc0);
    acc1 = fma(r.a[9 + j], xv[3 * j + 1], acc1);
    acc2 = fma(r.a[13 + j], xv[3 * j + 2], acc2);
  }
  return (acc0 + acc1) + acc2;
}

// Owner side of the scatter: exchange run of the lane's row <- a[r][slot(p)] * y[r]; pad <- y[r].
// (The lane only overwrites what it alone reads, so no barrier is needed after att_dot_row.)
template <class REC>
__device__ __forceinline__ void att_products(char* tile, int lane, const RowRegs& r, double yv) {
  double pr[12];
#pragma unroll
  for (int j = 0; j < 4; j++) {
    pr[3 * j] = r.a[5 + j] * yv;
    pr[3 * j + 1] = r.a[9 + j] * yv;
    pr[3 * j + 2] = r.a[13 + j] * yv;
  }
  if (REC::VEC16) {
    double2* xr = reinterpret_cast<double2*>(tile + REC::row_off(lane) + XOFF);
#pragma unroll
    for (int q = 0; q < 6; q++) xr[q] = make_double2(pr[2 * q], pr[2 * q + 1]);
  } else {
    double* xr = reinterpret_cast<double*>(tile + REC::row_off(lane) + XOFF);
#pragma unroll
    for (int q = 0; q < 12; q++) xr[q] = pr[q];
  }
  *reinterpret_cast<double*>(tile + REC::y_off(lane)) = yv;
}

// g_att(il)[3*t_r + p] += a[r][slot(p)] * y[r]  -- PAPER.md:49, Eq. (3), attitude block: per pass one
// red.global.add.f64 instruction whose 12 active lanes of each half-warp cover one contiguous run.
// Call after a __syncwarp() that follows att_products.
template <class REC>
__device__ __forceinline__ void att_scatter(const char* tile, const AttLane& L, const int (&t)[16],
                                            double* __restrict__ gatt_il) {
  if (L.act) {
#pragma unroll
    for (int it = 0; it < 16; it++)
      red_add(gatt_il + 3 * (int64_t)t[it] + L.p,
              *reinterpret_cast<const double*>(tile + REC::coop_off(it, L.h) + XOFF + 8 * L.p));
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
  double acc0 = r.a[23] * c.xg, acc1 = 0.0;
  acc0 = fma(r.a[0], g[0], acc0); acc1 = fma(r.a[1], g[1], acc1);
  acc0 = fma(r.a[2], g[2], acc0); acc1 = fma(r.a[3], g[3], acc1);
  acc0 = fma(r.a[4], g[4], acc0);
  acc1 = fma(r.a[17], g[5], acc1); acc0 = fma(r.a[18], g[6], acc0);
  acc1 = fma(r.a[19], g[7], acc1); acc0 = fma(r.a[20], g[8], acc0);
  acc1 = fma(r.a[21], g[9], acc1); acc0 = fma(r.a[22], g[10], acc0);
  return acc0 + acc1;
}

// Where a kernel scatters to (aprod 2 side).
struct ScatterCtx {
  double* x;        // the n-vector being accumulated into (astro and global parts)
  double* gatt_il;  // attitude accumulator, interleaved layout, 3K doubles
  double* xins;     // instrumental accumulator in global memory when neither of the next two is used: x + oI
  double* acc_s;    // shared-memory instrumental accumulator, or nullptr
  const uint32_t* ins_tab;  // shared-memory table of this CTA's die-local 4 KB accumulator chunks, or nullptr:
                            //   chunk c of the slice starts at ins_base + ins_tab[(c << tab_shift) | (lane & tab_mask)] doubles
  double* ins_base;
  int tab_shift, tab_mask;  // 5, 31: every lane reads its own bank (32 copies of the table, no bank conflicts); 0, 0: one copy
  int acc_part;             // with ins_tab: columns [0, acc_part) are accumulated in acc_s instead (whatever shared memory is left)
};

#ifdef GSR_HOST_EMULATION
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) { emu::dmma884(c0, c1, a, b); }
#else
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
#endif

// x[5*s + k] += sum_{rows r of star s in this tile} a[r][k] * y[r], k < 5   -- Eq. (3), astrometric block.
// Rows are sorted by star, so a tile covers the consecutive star ids s0 .. s1.  When s1 - s0 < 8 the sums
// are the 8 x 8 matrix product  C[q][k] = sum_r [star_r == s0 + q] y[r] * a[r][k]  (k < 5), accumulated
// over the 32 rows by eight fp64 DMMA.8x8x4 whose operands every lane reads straight from the staged
// tile: A[q][r] = y[r] or 0 (y from the row's pad, star from the index record), B[r][k] = a[r][k]
// (astro slots, intact).  Lane (q = lane >> 2, i = lane & 3) then owns C[q][2i], C[q][2i+1] and issues
// at most 2 reductions.  Exact fp64 FMAs (the indicator multiplies by 1 or adds 0).
// Otherwise (stars with < 5 rows, or unused star ids inside the tile): 5 reductions per row.
// Requires: att_products(yv) stored (yv = 0 for rows past the end) and a __syncwarp() since.
// square: the staged coefficients are squared on the fly (column-norm pass; r.a is squared by the caller).
template <class REC>
__device__ __forceinline__ void astro_scatter(const char* tile, int lane, int nvalid, bool valid, const RowRegs& r,
                                              double yv, double* __restrict__ x, bool square = false) {
  const int s0 = __shfl_sync(FULL, r.i0.x, 0), s1 = __shfl_sync(FULL, r.i0.x, nvalid - 1);
  if (s1 - s0 < 8) {
    const int q = lane >> 2, i = lane & 3;
    double c0 = 0.0, c1 = 0.0, d0 = 0.0, d1 = 0.0;   // two independent accumulation chains
#pragma unroll
    for (int j = 0; j < 8; j++) {
      const int row = 4 * j + i;
      const int st = *reinterpret_cast<const int*>(tile + COEF_TILE_BYTES + row * 32);
      const double y = *reinterpret_cast<const double*>(tile + REC::y_off(row));
      double b = *reinterpret_cast<const double*>(tile + REC::row_off(row) + 8 * (q < 5 ? q : 0));
      if (square) b *= b;
      if (j & 1) dmma884(d0, d1, (st - s0 == q) ? y : 0.0, q < 5 ? b : 0.0);
      else dmma884(c0, c1, (st - s0 == q) ? y : 0.0, q < 5 ? b : 0.0);
    }
    c0 += d0;
    c1 += d1;
    if (q <= s1 - s0 && i < 3) {
      double* xa = x + 5 * (int64_t)(s0 + q) + 2 * i;
      red_add(xa, c0);
      if (i < 2) red_add(xa + 1, c1);
    }
  } else if (valid) {
    double* xa = x + 5 * (int64_t)r.i0.x;
#pragma unroll
    for (int k = 0; k < 5; k++) red_add(xa + k, r.a[k] * yv);
  }
}

// Instrumental and global slots of the lane's own row, from registers.
//  instr  (slots 17-22): block-privatised accumulators in shared memory when the slice fits (flushed
//                        once per CTA), else reductions at L2.
//  global (slot 23)    : returned as the lane's contribution, reduced once per CTA by the caller.
//  (Shared memory has no native fp64 add: atomicAdd is an LDS / DADD / ATOMS.CAST.SPIN loop.  Running the
//  six chains of a row side by side with plain atomicCAS was measured SLOWER: aprod 2 at C2 0.72 vs 0.52 ms.)
template <bool INSTR_SMEM, bool PART>
__device__ __forceinline__ double scatter_rest(const RowRegs& r, int lane, bool valid, double yv, const ScatterCtx& c) {
  double gl = 0.0;
  if (valid) {
    const int col[6] = {r.i0.z, r.i0.w, r.i1.x, r.i1.y, r.i1.z, r.i1.w};
    double inc[6];
#pragma unroll
    for (int q = 0; q < 6; q++) inc[q] = r.a[17 + q] * yv;
    if (!INSTR_SMEM && c.ins_tab) {
      const int lsel = lane & c.tab_mask;
      double* dst[6];
#pragma unroll
      for (int q = 0; q < 6; q++)
        dst[q] = c.ins_base + c.ins_tab[((col[q] >> INS_CHUNK_SHIFT) << c.tab_shift) | lsel] + (col[q] & (INS_CHUNK - 1));
      if (PART) {
        // what bounds the pass at C4 is L2 requests (an fp64 reduction costs ~1.65 of them), and shared-memory work
        // runs in their shadow: every column that still fits shared memory is accumulated there.  The six L2
        // reductions stay back to back as predicated instructions (a branch per slot serialised them: +15 %).
        // PART is a template parameter so that kernels without the partial accumulators carry none of this code.
#pragma unroll
        for (int q = 0; q < 6; q++) red_add_if_ge(dst[q], inc[q], col[q], c.acc_part);
#pragma unroll
        for (int q = 0; q < 6; q++)
          if (col[q] < c.acc_part) atomicAdd(c.acc_s + col[q], inc[q]);
      } else {
#pragma unroll
        for (int q = 0; q < 6; q++) red_add(dst[q], inc[q]);
      }
    } else {
      if (INSTR_SMEM) {
#pragma unroll
        for (int q = 0; q < 6; q++) atomicAdd(c.acc_s + col[q], inc[q]);
      } else {
#pragma unroll
        for (int q = 0; q < 6; q++) red_add(c.xins + col[q], inc[q]);
      }
    }
    gl = r.a[23] * yv;
  }
  return gl;
}

// One thread reads one whole record from global memory (row-thread kernels): 24 doubles as 12 x 128-bit, or the
// 23 doubles of the production record (184-byte rows: 8-byte alignment only) one by one; slot 23 reads as 0 there.
__device__ __forceinline__ void load_record(const SysView& s, int64_t r, double (&a)[NSLOT]) {
  if (s.cpr == NSLOT) {
    const double2* ap = reinterpret_cast<const double2*>(s.vals + r * NSLOT);
#pragma unroll
    for (int q = 0; q < NSLOT / 2; q++) {
      const double2 t = __ldcs(ap + q);
      a[2 * q] = t.x;
      a[2 * q + 1] = t.y;
    }
  } else {
    const double* ap = s.vals + r * (NSLOT - 1);
#pragma unroll
    for (int k = 0; k < NSLOT - 1; k++) a[k] = __ldcs(ap + k);
    a[NSLOT - 1] = 0.0;
  }
}

// Shared-memory plan of the TMA kernels.
struct SmemPlan {
  int warps, stages;
  bool gather_smem;   // instrumental slice of x staged in shared memory (aprod 1 side)
  bool acc_smem;      // instrumental accumulators privatised in shared memory (aprod 2 side)
  bool ins_tab;       // else: room reserved for the table of die-local accumulator chunks (InstrAcc)
  int tab_shift;      // 5: the table is replicated 32 times, one copy per bank (LDS without bank conflicts); 0: one copy
  int acc_part;       // with ins_tab: leading columns whose accumulators are privatised in the shared memory left over
  size_t bytes;       // dynamic shared memory to request
};
enum { PLAN_APROD1 = 1, PLAN_APROD2 = 2, PLAN_FUSED = 3 };
SmemPlan plan_smem(const SysView& s, const Tuning& t, int what);

// This CTA's set of die-local accumulator chunks -> shared memory (n_chunks pointers).  Call before a
// __syncthreads().  The set is chosen by the die of the SM the CTA runs on.
// Entry (c << tab_shift) + j, j < 2^tab_shift, is the offset (in doubles, from ia.base) of chunk c: with tab_shift = 5
// lane l reads word 32 c + l, i.e. always its own bank (a single shared copy cost 5.5 wavefronts per LDS at C4).
__device__ __forceinline__ void load_ins_tab(uint32_t* tab_s, const InstrAcc& ia, int tab_shift) {
  unsigned smid;
#ifdef GSR_HOST_EMULATION
  smid = emu::smid();
#else
  asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
#endif
  int die = smid < (unsigned)SMID_SLOTS ? ia.sm_die[smid] : 0;
  if (die < 0 || !ia.two_dies) die = 0;
  const int set = die * ia.copies_per_die + (int)(blockIdx.x % (unsigned)ia.copies_per_die);
  for (int i = threadIdx.x; i < (ia.n_chunks << tab_shift); i += blockDim.x)
    tab_s[i] = (uint32_t)(ia.chunk_tab[(size_t)set * ia.n_chunks + (i >> tab_shift)] - ia.base);
}

__device__ __forceinline__ char* smem_align128(char* p) { return p + ((128u - (smem_u32(p) & 127u)) & 127u); }

}  // namespace gsr
