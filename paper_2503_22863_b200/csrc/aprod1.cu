// aprod1:  y[r] = sum_k a[r][k] * x[col(r,k)] + c0 * y[r]           (Eq. 2)
// with the LSQR u-update and ||u||^2 fused in.
#include "aprod_device.cuh"

namespace gsr {

// ---- variant 1 (default): TMA-staged row tiles, one warp per tile, lane per row -----------------
template <int ATT, bool GSMEM>
__global__ void __launch_bounds__(512, 1)
k_aprod1_tma(const __grid_constant__ CUtensorMap map, SysView s, int nstages, const double* __restrict__ x,
             const double* __restrict__ xw, int64_t xw_axis_stride, double* __restrict__ y,
             const double* __restrict__ c0p, double* sumsq, int* done) {
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

  TileRing ring;
  const int64_t gw = (int64_t)blockIdx.x * nwarps + warp, W = (int64_t)gridDim.x * nwarps;
  ring.init(ring_mem, bars + warp * nstages, &map, s.idx, s.M, gw, W, lane, nstages);
  if (GSMEM) {
    for (int64_t i = threadIdx.x; i < s.I; i += blockDim.x) xi_s[i] = __ldg(x + s.oI + i);
    __syncthreads();
  }
  GatherCtx gc{x, xw, xw_axis_stride, xi_s, x + s.oI, s.G ? __ldg(x + s.oG) : 0.0};
  const double c0 = c0p ? *c0p : 1.0;
  double sq = 0.0;

  for (int64_t t = gw; t < ring.n_tiles; t += W) {
    const int64_t r = t * TILE_ROWS + lane;
    const bool valid = r < s.M;
    const double yin = valid ? y[r] : 0.0;
    const char* tile = ring.acquire();
    RowRegs row;
    load_row(tile, lane, valid, row);
    const double out = fma(c0, yin, row_dot<ATT, GSMEM>(row, gc));
    if (valid) {
      y[r] = out;
      sq = fma(out, out, sq);
    }
    ring.release(lane);   // after the dependent store: every LDS of this tile has completed
  }
  if (sumsq) {
    sq = block_sum(sq);
    if (threadIdx.x == 0) atomicAdd(sumsq, sq);
  }
}

// Expanded attitude windows, rebuilt from x before every gather pass (3K reads, <= 12K writes: << matrix).
//   step 1 (ATT_FULL): xw[(ax*nwin + t)*4 + j] = x[oA + ax*K + t + j],  t = 0 .. K-4
//   step 2 (ATT_HALF): xw[(ax*nwin + w)*4 + j] = x[oA + ax*K + 2w + j], w = 0 .. (K-2)/2
// Elements past the end of x (only pad slots of the very last windows) read as 0.
__global__ void __launch_bounds__(256) k_expand_att(const double* __restrict__ x, int64_t oA, int64_t n, int64_t K,
                                                    int step, int64_t nwin, double* __restrict__ xw, const int* done) {
  if (done && *done) return;
  const int64_t total = 3 * nwin;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t ax = i / nwin, w = i - ax * nwin;
    const int64_t e = oA + ax * K + w * step;
    double v[4];
#pragma unroll
    for (int j = 0; j < 4; j++) v[j] = (e + j < n) ? __ldg(x + e + j) : 0.0;
    double2* o = reinterpret_cast<double2*>(xw + i * 4);
    o[0] = make_double2(v[0], v[1]);
    o[1] = make_double2(v[2], v[3]);
  }
}

cudaError_t launch_expand_att(const SysView& s, const SideData& sd, int num_sms, const double* x, const int* done,
                              cudaStream_t st, int64_t* launches) {
  const int64_t total = 3 * sd.xw_nwin;
  int64_t eb = (total + 255) / 256;
  if (eb > num_sms * 8) eb = num_sms * 8;
  k_expand_att<<<(unsigned)eb, 256, 0, st>>>(x, s.oA, s.n, s.K, sd.att_mode == ATT_FULL ? 1 : 2, sd.xw_nwin, sd.xw, done);
  ++*launches;
  return cudaGetLastError();
}

// ---- shared-memory plan of the TMA kernels --------------------------------------------------------
static size_t ring_bytes(int w, int st) { return (size_t)w * st * STAGE_BYTES + (size_t)(w * st + 2) * 8 + 128; }

SmemPlan plan_smem(const SysView& s, const Tuning& t, int what) {
  SmemPlan p;
  p.warps = t.warps > 0 ? t.warps : 8;
  p.stages = t.stages > 0 ? t.stages : 2;
  p.gather_smem = p.acc_smem = false;
  const size_t table = ((size_t)s.I * 8 + 15) & ~(size_t)15;
  size_t ring = ring_bytes(p.warps, p.stages);
  if (ring > SMEM_BUDGET) { p.bytes = ring; return p; }   // caller rejects (cudaErrorInvalidValue)
  size_t left = SMEM_BUDGET - ring;
  // privatised accumulators save 6 L2 reductions per row; the gather copy saves 6 L1 gathers per row
  if ((what & PLAN_APROD2) && table <= left) { p.acc_smem = true; left -= table; }
  if ((what & PLAN_APROD1) && table <= left) { p.gather_smem = true; left -= table; }
  p.bytes = SMEM_BUDGET - left;
  return p;
}

template <int ATT>
static cudaError_t launch_tma1(bool gsmem, const SysView& s, const SideData& sd, int grid, const SmemPlan& p,
                               const double* x, double* y, const double* c0, double* sumsq, int* done, cudaStream_t st) {
  auto k = gsmem ? k_aprod1_tma<ATT, true> : k_aprod1_tma<ATT, false>;
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.bytes);
  if (e != cudaSuccess) return e;
  k<<<grid, p.warps * 32, p.bytes, st>>>(sd.map, s, p.stages, x, sd.xw, sd.xw_axis_stride, y, c0, sumsq, done);
  return cudaGetLastError();
}

// ---- variant 0: one thread per row, direct global loads (simple device-side cross-check) --------
__global__ void __launch_bounds__(256) k_aprod1_rowthread(SysView s, const double* __restrict__ x,
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
    const double2* ap = reinterpret_cast<const double2*>(s.vals + r * NSLOT);
    const int4* ip = reinterpret_cast<const int4*>(s.idx + r * NIDX);
    const int4 i0 = __ldg(ip), i1 = __ldg(ip + 1);
    double a[NSLOT];
#pragma unroll
    for (int q = 0; q < NSLOT / 2; q++) {
      double2 t = __ldcs(ap + q);
      a[2 * q] = t.x;
      a[2 * q + 1] = t.y;
    }
    const double* xa = x + 5 * (int64_t)i0.x;
    double acc = 0.0;
#pragma unroll
    for (int k = 0; k < 5; k++) acc = fma(a[k], __ldg(xa + k), acc);
    const double* xt = x + s.oA + i0.y;
#pragma unroll
    for (int ax = 0; ax < 3; ax++)
#pragma unroll
      for (int j = 0; j < 4; j++) acc = fma(a[5 + 4 * ax + j], __ldg(xt + ax * s.K + j), acc);
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

cudaError_t launch_aprod1(const SysView& s, const SideData& sd, const Tuning& t, int num_sms, const double* x,
                          double* y, const double* c0, double* sumsq, int* done, cudaStream_t st,
                          int64_t* launches) {
  if (s.M == 0) return cudaSuccess;
  if (t.aprod1_variant == 1) {
    const SmemPlan p = plan_smem(s, t, PLAN_APROD1);
    if (p.bytes > SMEM_BUDGET || p.warps > 16 || p.warps < 1 || p.stages < 1) return cudaErrorInvalidValue;
    cudaError_t e = launch_expand_att(s, sd, num_sms, x, done, st, launches);
    if (e != cudaSuccess) return e;
    const int grid = num_sms * (t.ctas_per_sm > 0 ? t.ctas_per_sm : 1);
    ++*launches;
    return sd.att_mode == ATT_FULL ? launch_tma1<ATT_FULL>(p.gather_smem, s, sd, grid, p, x, y, c0, sumsq, done, st)
                                   : launch_tma1<ATT_HALF>(p.gather_smem, s, sd, grid, p, x, y, c0, sumsq, done, st);
  }
  const int threads = 256;
  int64_t blocks = (s.M + threads - 1) / threads;
  const int64_t cap = (int64_t)num_sms * 8;
  if (blocks > cap) blocks = cap;
  k_aprod1_rowthread<<<(unsigned)blocks, threads, 0, st>>>(s, x, y, c0, sumsq, done);
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
