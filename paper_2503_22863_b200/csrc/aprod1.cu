// aprod1:  y[r] = sum_k a[r][k] * x[col(r,k)] + c0 * y[r]           (Eq. 2)
// with the LSQR u-update and ||u||^2 fused in.
#include "aprod_device.cuh"

namespace gsr {

// ---- variant 1 (default): TMA-staged row tiles, one warp per tile ---------------------------------
template <class REC, bool GSMEM>
__global__ void __launch_bounds__(MAX_TMA_WARPS * 32, 1)
k_aprod1_tma(const __grid_constant__ CUtensorMap map, SysView s, int nstages, const double* __restrict__ x,
             const double* __restrict__ att_il, double* __restrict__ y, const double* __restrict__ c0p, double* sumsq,
             int* done) {
  if (done) {
    const int d = *done;
    if (d) {  // LSQR already stopped: no-op (and latch "update pending" 2 -> 1, see k_step_scalars)
      if (d == 2 && blockIdx.x == 0 && threadIdx.x == 0) *done = 1;
      return;
    }
  }
  extern __shared__ char smem_raw[];
  char* smem = smem_align128(smem_raw);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  char* ring_mem = smem + (size_t)warp * nstages * STAGE_BYTES;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)nwarps * nstages * STAGE_BYTES);
  double* xi_s = reinterpret_cast<double*>(bars + nwarps * nstages + 2);

  TileRing<REC> ring;
  const int64_t gw = (int64_t)blockIdx.x * nwarps + warp, W = (int64_t)gridDim.x * nwarps;
  ring.init(ring_mem, bars + warp * nstages, &map, s.vals, s.idx, s.M, gw, W, lane, nstages);
  if (GSMEM) {
    for (int64_t i = threadIdx.x; i < s.I; i += blockDim.x) xi_s[i] = __ldg(x + s.oI + i);
    __syncthreads();
  }
  GatherCtx gc{x, att_il, xi_s, x + s.oI, s.G ? __ldg(x + s.oG) : 0.0};
  const AttLane al(lane);
  const double c0 = c0p ? *c0p : 1.0;
  double sq = 0.0;

  double ynext = (gw < ring.n_tiles && gw * TILE_ROWS + lane < s.M) ? y[gw * TILE_ROWS + lane] : 0.0;
  for (int64_t t = gw; t < ring.n_tiles; t += W) {
    const int64_t row0 = t * TILE_ROWS;
    const int64_t r = row0 + lane;
    const bool valid = r < s.M;
    const double yin = ynext;
    {  // prefetch the next tile's y (keeps a DRAM round trip off every tile's critical path)
      const int64_t rn = r + W * TILE_ROWS;
      ynext = rn < s.M ? y[rn] : 0.0;
    }
    char* tile = ring.acquire(t, lane);
    RowRegs row;
    load_row<REC>(tile, lane, valid, row);
    int ts[16];
    att_starts(tile, al, ts);
    __syncwarp();   // every lane holds its row: the exchange runs may be written
    att_gather<REC>(tile, al, ts, att_il);
    const double rest = row_dot_rest<GSMEM>(row, gc);
    __syncwarp();
    const double out = fma(c0, yin, att_dot_row<REC>(tile, lane, row) + rest);
    if (valid) {
      y[r] = out;
      sq = fma(out, out, sq);
    }
    ring.release(lane);
  }
  if (sumsq) {
    sq = block_sum(sq);
    if (threadIdx.x == 0) atomicAdd(sumsq, sq);
  }
}

// Attitude block between the API layout (axis-major: x[oA + ax*K + t]) and the interleaved layout the
// kernels gather from / scatter into (il[3*t + ax]); 3K elements, negligible next to the matrix.
__global__ void __launch_bounds__(256) k_att_to_il(const double* __restrict__ xatt, int64_t K, double* __restrict__ il,
                                                   const int* done) {
  if (done && *done) return;
  const int64_t total = 3 * K;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t t = i / 3, ax = i - 3 * t;
    il[i] = __ldg(xatt + ax * K + t);
  }
}
// x_att[ax*K + t] += il[3*t + ax] ; il <- 0   (folds the interleaved accumulator of a standalone aprod 2)
__global__ void __launch_bounds__(256) k_att_fold(double* __restrict__ xatt, int64_t K, double* __restrict__ il) {
  const int64_t total = 3 * K;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t ax = i / K, t = i - ax * K;
    xatt[i] += il[3 * t + ax];
  }
}
// dst[ax*K + t] = il[3*t + ax]   (export of an internal n-vector's attitude block)
__global__ void __launch_bounds__(256) k_att_from_il(const double* __restrict__ il, int64_t K, double* __restrict__ dst) {
  const int64_t total = 3 * K;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t ax = i / K, t = i - ax * K;
    dst[i] = il[3 * t + ax];
  }
}

static unsigned att_grid(int64_t K, int num_sms) {
  int64_t b = (3 * K + 255) / 256;
  if (b > (int64_t)num_sms * 8) b = (int64_t)num_sms * 8;
  return (unsigned)(b < 1 ? 1 : b);
}
cudaError_t launch_att_to_il(const SysView& s, int num_sms, const double* x_std, double* il, const int* done,
                             cudaStream_t st, int64_t* launches) {
  k_att_to_il<<<att_grid(s.K, num_sms), 256, 0, st>>>(x_std + s.oA, s.K, il, done);
  ++*launches;
  return cudaGetLastError();
}
cudaError_t launch_att_fold(const SysView& s, int num_sms, double* x_std, double* il, cudaStream_t st, int64_t* launches) {
  k_att_fold<<<att_grid(s.K, num_sms), 256, 0, st>>>(x_std + s.oA, s.K, il);
  ++*launches;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  return cudaMemsetAsync(il, 0, (size_t)(3 * s.K) * sizeof(double), st);
}
cudaError_t launch_att_from_il(const SysView& s, int num_sms, const double* il, double* dst_std_att, cudaStream_t st,
                               int64_t* launches) {
  k_att_from_il<<<att_grid(s.K, num_sms), 256, 0, st>>>(il, s.K, dst_std_att);
  ++*launches;
  return cudaGetLastError();
}

// ---- shared-memory plan of the TMA kernels --------------------------------------------------------
static size_t ring_bytes(int w, int st) { return (size_t)w * st * STAGE_BYTES + (size_t)(w * st + 2) * 8 + 128; }

// Warps per CTA trade latency hiding against room for the instrumental tables.  Measured (B200, fused
// pass / aprod 1 / aprod 2): C3 (I = 6,000) 12 warps without tables 4.89 / 2.39 / 4.25 ms, 8 warps with the
// tables 4.19 / 1.90 / 2.70 ms; C5 (I = 12,000, only one table fits at 8 warps) 14.6 / 8.68 / 12.0 ms with
// 12 warps, 17.6 / 6.82 / 8.48 ms with 8.  So: the most warps (12 down to 8) at which EVERY table the kernel
// wants fits; if there is no such count, 12 warps and whatever still fits.
SmemPlan plan_smem(const SysView& s, const Tuning& t, int what) {
  SmemPlan p;
  p.stages = t.stages > 0 ? t.stages : 2;
  p.gather_smem = p.acc_smem = p.ins_tab = false;
  p.tab_shift = 0;
  p.acc_part = 0;
  const size_t table = ((size_t)s.I * 8 + 15) & ~(size_t)15;
  const bool want_acc = (what & PLAN_APROD2) && t.acc_smem, want_gather = (what & PLAN_APROD1) && t.gather_smem;
  const size_t want = (want_acc ? table : 0) + (want_gather ? table : 0);
  p.warps = t.warps > 0 ? t.warps : 12;
  if (t.warps <= 0 && want > 0)
    for (int w = 12; w >= 8; w--)
      if (ring_bytes(w, p.stages) + want <= SMEM_BUDGET) { p.warps = w; break; }
  size_t ring = ring_bytes(p.warps, p.stages);
  if (ring > SMEM_BUDGET) { p.bytes = ring; return p; }   // caller rejects (cudaErrorInvalidValue)
  size_t left = SMEM_BUDGET - ring;
  // privatised accumulators save 6 L2 reductions per row; the gather copy saves 6 L1/L2 gathers per row
  if (want_acc && table <= left) { p.acc_smem = true; left -= table; }
  if (want_gather && table <= left) { p.gather_smem = true; left -= table; }
  // otherwise the aprod 2 side reduces into die-local chunked copies in L2: room for this CTA's chunk table
  // (32 copies, one per bank, when they fit: 15 KB at C4; else one copy)
  const size_t tab = ((size_t)((s.I + INS_CHUNK - 1) / INS_CHUNK) * sizeof(uint32_t) + 15) & ~(size_t)15;
  if ((what & PLAN_APROD2) && !p.acc_smem) {
    if (t.tab_private && 32 * tab <= left) { p.ins_tab = true; p.tab_shift = 5; left -= 32 * tab; }
    else if (tab <= left) { p.ins_tab = true; left -= tab; }
    const int want_part = what == PLAN_FUSED ? t.acc_part_fused : t.acc_part;
    if (p.ins_tab && want_part) {
      size_t ent = left / 8 & ~(size_t)1;
      if (want_part > 0 && ent > (size_t)want_part) ent = (size_t)want_part & ~(size_t)1;
      if ((int64_t)ent > s.I) ent = (size_t)s.I;
      p.acc_part = (int)ent;
      left -= ((ent + 1) & ~(size_t)1) * 8;
    }
  }
  p.bytes = SMEM_BUDGET - left;
  return p;
}

static cudaError_t launch_tma1(bool gsmem, const SysView& s, const SideData& sd, int grid, const SmemPlan& p,
                               const double* x, const double* att_il, double* y, const double* c0, double* sumsq,
                               int* done, cudaStream_t st) {
  auto k = s.cpr == NSLOT ? (gsmem ? k_aprod1_tma<Rec24, true> : k_aprod1_tma<Rec24, false>)
                          : (gsmem ? k_aprod1_tma<Rec23, true> : k_aprod1_tma<Rec23, false>);
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.bytes);
  if (e != cudaSuccess) return e;
  k<<<grid, p.warps * 32, p.bytes, st>>>(sd.map, s, p.stages, x, att_il, y, c0, sumsq, done);
  return cudaGetLastError();
}

// ---- variant 0: one thread per row, direct global loads (simple device-side cross-check, either record format) ----
__global__ void __launch_bounds__(256) k_aprod1_rowthread(SysView s, const double* __restrict__ x, bool x_il,
                                                          double* __restrict__ y,
                                                          const double* __restrict__ c0p,
                                                          double* sumsq, int* done) {
  if (done) {
    const int d = *done;
    if (d) {
      if (d == 2 && blockIdx.x == 0 && threadIdx.x == 0) *done = 1;
      return;
    }
  }
  const double c0 = c0p ? *c0p : 1.0;
  double sq = 0.0;
  for (int64_t r = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; r < s.M;
       r += (int64_t)gridDim.x * blockDim.x) {
    const int4* ip = reinterpret_cast<const int4*>(s.idx + r * NIDX);
    const int4 i0 = __ldg(ip), i1 = __ldg(ip + 1);
    double a[NSLOT];
    load_record(s, r, a);
    const double* xa = x + 5 * (int64_t)i0.x;
    double acc = 0.0;
#pragma unroll
    for (int k = 0; k < 5; k++) acc = fma(a[k], __ldg(xa + k), acc);
    const int64_t sa = x_il ? 1 : s.K, sj = x_il ? 3 : 1;   // attitude strides: axis, knot
    const double* xt = x + s.oA + i0.y * sj;
#pragma unroll
    for (int ax = 0; ax < 3; ax++)
#pragma unroll
      for (int j = 0; j < 4; j++) acc = fma(a[5 + 4 * ax + j], __ldg(xt + ax * sa + j * sj), acc);
    const double* xi = x + s.oI;
    acc = fma(a[17], __ldg(xi + i0.z), acc);
    acc = fma(a[18], __ldg(xi + i0.w), acc);
    acc = fma(a[19], __ldg(xi + i1.x), acc);
    acc = fma(a[20], __ldg(xi + i1.y), acc);
    acc = fma(a[21], __ldg(xi + i1.z), acc);
    acc = fma(a[22], __ldg(xi + i1.w), acc);
    if (s.G) acc = fma(a[23], __ldg(x + s.oG), acc);
    const double out = fma(c0, y[r], acc);
    y[r] = out;
    sq = fma(out, out, sq);
  }
  if (sumsq) {
    sq = block_sum(sq);
    if (threadIdx.x == 0) atomicAdd(sumsq, sq);
  }
}

// x_il = true: the attitude block of x is already interleaved (LSQR-internal vectors); otherwise x is in
// the API layout and its attitude block is first copied into the side buffer sd.att_il.
cudaError_t launch_aprod1(const SysView& s, const SideData& sd, const Tuning& t, int num_sms, const double* x,
                          bool x_il, double* y, const double* c0, double* sumsq, int* done, cudaStream_t st,
                          int64_t* launches) {
  if (s.M == 0) return cudaSuccess;
  if (t.aprod1_variant == 1) {
    const SmemPlan p = plan_smem(s, t, PLAN_APROD1);
    if (p.bytes > SMEM_BUDGET || p.warps > MAX_TMA_WARPS || p.warps < 1 || p.stages < 1) return cudaErrorInvalidValue;
    const double* att_il = x + s.oA;
    if (!x_il) {
      cudaError_t e = launch_att_to_il(s, num_sms, x, sd.att_il, done, st, launches);
      if (e != cudaSuccess) return e;
      att_il = sd.att_il;
    }
    const int grid = num_sms * (t.ctas_per_sm > 0 ? t.ctas_per_sm : 1);
    ++*launches;
    return launch_tma1(p.gather_smem, s, sd, grid, p, x, att_il, y, c0, sumsq, done, st);
  }
  const int threads = 256;
  int64_t blocks = (s.M + threads - 1) / threads;
  const int64_t cap = (int64_t)num_sms * 8;
  if (blocks > cap) blocks = cap;
  k_aprod1_rowthread<<<(unsigned)blocks, threads, 0, st>>>(s, x, x_il, y, c0, sumsq, done);
  ++*launches;
  return cudaGetLastError();
}

// ---- index-record validation (gsr_create) ------------------------------------------------------
__global__ void k_validate(SysView s, int* flag) {
  for (int64_t r = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; r < s.M;
       r += (int64_t)gridDim.x * blockDim.x) {
    const int32_t* rec = s.idx + r * NIDX;
    int bad = 0;
    const int32_t star = rec[0];
    if (star < 0 || star >= s.S) bad |= 1;
    if (r > 0 && s.idx[(r - 1) * NIDX] > star) bad |= 2;  // rows must be sorted by star
    if (rec[1] < 0 || rec[1] > s.K - 4) bad |= 4;
#pragma unroll
    for (int q = 0; q < 6; q++)
      if (rec[2 + q] < 0 || rec[2 + q] >= s.I) bad |= 8;
    if (bad) atomicOr(flag, bad);
  }
}

cudaError_t launch_validate(const SysView& s, int* flag, cudaStream_t st, int64_t* launches) {
  if (s.M == 0) return cudaSuccess;
  int64_t blocks = (s.M + 255) / 256;
  if (blocks > 148 * 16) blocks = 148 * 16;
  k_validate<<<(unsigned)blocks, 256, 0, st>>>(s, flag);
  ++*launches;
  return cudaGetLastError();
}

}  // namespace gsr
