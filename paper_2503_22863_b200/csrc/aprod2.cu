// aprod2:  x[col(r,k)] += a[r][k] * (yscale * y[r])                  (Eq. 3)
#include "gsr_internal.cuh"
#include "tma.cuh"

namespace gsr {

// ---- variant 1 (default): TMA-staged row tiles, split by parameter block ------------------------
//  astro  (slots 0-4)  : rows are sorted by star, so the lanes of a warp hold runs of equal star;
//                        a segmented warp scan (shuffles) sums each run, the run head issues 5 adds.
//  att    (slots 5-16) : the 12 x 32 products of a tile are walked element-per-lane, so 4 consecutive
//                        lanes cover one 4-knot run: the 4 fp64 reductions of a run travel to L2 as
//                        one request (measured 2.2x the add rate of lane-per-row issue).
//  instr  (slots 17-22): block-privatised accumulators in shared memory (when the slice fits),
//                        flushed to x once per CTA at the end; else reductions at L2.
//  global (slot 23)    : register accumulation, one reduction per CTA.
template <int STAGES, bool INSTR_SMEM>
__global__ void __launch_bounds__(512, 1)
k_aprod2_tma(const __grid_constant__ CUtensorMap map, SysView s, const double* __restrict__ y,
             double* __restrict__ x, const double* __restrict__ yscale, const int* done) {
  if (done && *done) return;
  extern __shared__ char smem_raw[];
  char* smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  char* ring_mem = smem + (size_t)warp * STAGES * STAGE_BYTES;
  double* acc_s = reinterpret_cast<double*>(smem + (size_t)nwarps * STAGES * STAGE_BYTES);
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<char*>(acc_s) + (INSTR_SMEM ? ((s.I * 8 + 15) & ~15ll) : 0));

  TileRing<STAGES> ring;
  const int64_t gw = (int64_t)blockIdx.x * nwarps + warp, W = (int64_t)gridDim.x * nwarps;
  ring.init(ring_mem, bars + warp * STAGES, &map, s.idx, s.M, gw, W, lane);
  if (INSTR_SMEM) {
    for (int64_t i = threadIdx.x; i < s.I; i += blockDim.x) acc_s[i] = 0.0;
    __syncthreads();
  }
  const double ys = yscale ? *yscale : 1.0;
  double* xatt = x + s.oA;
  double* xins = x + s.oI;
  double gacc = 0.0;

  for (int64_t t = gw; t < ring.n_tiles; t += W) {
    const int64_t row0 = t * TILE_ROWS;
    const int64_t r = row0 + lane;
    const bool valid = r < s.M;
    const double yv = valid ? ys * y[r] : 0.0;
    const int nvalid = (s.M - row0) < TILE_ROWS ? (int)(s.M - row0) : TILE_ROWS;
    const char* tile = ring.acquire();
    const double* td = reinterpret_cast<const double*>(tile);
    const int32_t* ti = reinterpret_cast<const int32_t*>(tile + COEF_TILE_BYTES);

    // ---- attitude: element e = 12*row + slot, 4 consecutive lanes = one run of 4 knots
#pragma unroll
    for (int it = 0; it < 12; it++) {
      const int e = it * 32 + lane;
      const int row = e / 12, sl = e - row * 12;
      const double yy = __shfl_sync(0xffffffffu, yv, row);
      if (row < nvalid) {
        const double a = td[row * ROW_STRIDE_D + 5 + sl];
        const int att = ti[row * 8 + 1];
        atomicAdd(xatt + (int64_t)(sl >> 2) * s.K + att + (sl & 3), a * yy);
      }
    }

    // ---- lane-per-row part: astro, instrumental, global
    const double2* ap = reinterpret_cast<const double2*>(tile + lane * (ROW_STRIDE_D * 8));
    const int4* ip = reinterpret_cast<const int4*>(tile + COEF_TILE_BYTES + lane * 32);
    int4 i0 = ip[0], i1 = ip[1];
    const double2 a01 = ap[0], a23 = ap[1], a45 = ap[2];
    const double2 a1617 = ap[8], a1819 = ap[9], a2021 = ap[10], a2223 = ap[11];
    int star = valid ? i0.x : (-1 - lane);
    double p0 = a01.x * yv, p1 = a01.y * yv, p2 = a23.x * yv, p3 = a23.y * yv, p4 = a45.x * yv;
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
      double* xa = x + 5 * (int64_t)star;
      atomicAdd(xa, p0); atomicAdd(xa + 1, p1); atomicAdd(xa + 2, p2); atomicAdd(xa + 3, p3); atomicAdd(xa + 4, p4);
    }
    if (valid) {
      const double v17 = a1617.y * yv, v18 = a1819.x * yv, v19 = a1819.y * yv, v20 = a2021.x * yv,
                   v21 = a2021.y * yv, v22 = a2223.x * yv;
      if (INSTR_SMEM) {
        atomicAdd(acc_s + i0.z, v17); atomicAdd(acc_s + i0.w, v18); atomicAdd(acc_s + i1.x, v19);
        atomicAdd(acc_s + i1.y, v20); atomicAdd(acc_s + i1.z, v21); atomicAdd(acc_s + i1.w, v22);
      } else {
        atomicAdd(xins + i0.z, v17); atomicAdd(xins + i0.w, v18); atomicAdd(xins + i1.x, v19);
        atomicAdd(xins + i1.y, v20); atomicAdd(xins + i1.z, v21); atomicAdd(xins + i1.w, v22);
      }
      gacc = fma(a2223.y, yv, gacc);
    }
    ring.release(lane);
  }
  if (INSTR_SMEM) {
    __syncthreads();
    for (int64_t i = threadIdx.x; i < s.I; i += blockDim.x) {
      const double v = acc_s[i];
      if (v != 0.0) atomicAdd(xins + i, v);
    }
  }
  if (s.G) {
    gacc = block_sum(gacc);
    if (threadIdx.x == 0) atomicAdd(x + s.oG, gacc);
  }
}

// ---- variant 0: one thread per row, fp64 reductions at L2 for every slot (first correct path) --
__global__ void __launch_bounds__(256) k_aprod2_rowthread(SysView s, const double* __restrict__ y,
                                                          double* __restrict__ x,
                                                          const double* __restrict__ yscale,
                                                          const int* done) {
  if (done && *done) return;
  const double ys = yscale ? *yscale : 1.0;
  double gsum = 0.0;
  for (int64_t r0 = blockIdx.x * (int64_t)blockDim.x; r0 < s.M; r0 += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = r0 + threadIdx.x;
    if (r < s.M) {
      const double2* ap = reinterpret_cast<const double2*>(s.vals + r * NSLOT);
      const int4* ip = reinterpret_cast<const int4*>(s.idx + r * NIDX);
      const int4 i0 = __ldg(ip), i1 = __ldg(ip + 1);
      const double yr = ys * y[r];
      double a[NSLOT];
#pragma unroll
      for (int q = 0; q < NSLOT / 2; q++) {
        double2 t = __ldcs(ap + q);
        a[2 * q] = t.x;
        a[2 * q + 1] = t.y;
      }
      double* xa = x + 5 * (int64_t)i0.x;
#pragma unroll
      for (int k = 0; k < 5; k++) atomicAdd(xa + k, a[k] * yr);
      double* xt = x + s.oA + i0.y;
#pragma unroll
      for (int ax = 0; ax < 3; ax++)
#pragma unroll
        for (int j = 0; j < 4; j++) atomicAdd(xt + ax * s.K + j, a[5 + 4 * ax + j] * yr);
      double* xi = x + s.oI;
      atomicAdd(xi + i0.z, a[17] * yr);
      atomicAdd(xi + i0.w, a[18] * yr);
      atomicAdd(xi + i1.x, a[19] * yr);
      atomicAdd(xi + i1.y, a[20] * yr);
      atomicAdd(xi + i1.z, a[21] * yr);
      atomicAdd(xi + i1.w, a[22] * yr);
      gsum = fma(a[23], yr, gsum);
    }
  }
  if (s.G) {
    gsum = block_sum(gsum);
    if (threadIdx.x == 0) atomicAdd(x + s.oG, gsum);
  }
}

template <int STAGES, bool INSTR_SMEM>
static cudaError_t launch_tma2_t(const SysView& s, const SideData& sd, int grid, int warps, size_t smem,
                                 const double* y, double* x, const double* yscale, const int* done, cudaStream_t st) {
  auto k = k_aprod2_tma<STAGES, INSTR_SMEM>;
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k<<<grid, warps * 32, smem, st>>>(sd.map, s, y, x, yscale, done);
  return cudaGetLastError();
}
static cudaError_t launch_tma2(int stages, bool ismem, const SysView& s, const SideData& sd, int grid, int warps,
                               size_t smem, const double* y, double* x, const double* yscale, const int* done,
                               cudaStream_t st) {
#define GSR_A2(ST) (ismem ? launch_tma2_t<ST, true>(s, sd, grid, warps, smem, y, x, yscale, done, st) \
                          : launch_tma2_t<ST, false>(s, sd, grid, warps, smem, y, x, yscale, done, st))
  switch (stages) {
    case 2: return GSR_A2(2);
    case 4: return GSR_A2(4);
    default: return GSR_A2(3);
  }
#undef GSR_A2
}

cudaError_t launch_aprod2(const SysView& s, const SideData& sd, const Tuning& t, int num_sms, const double* y,
                          double* x, const double* yscale, const int* done, cudaStream_t st, int64_t* launches) {
  if (s.M == 0) return cudaSuccess;
  if (t.aprod2_variant == 1) {
    const int warps = t.warps > 0 ? t.warps : 8;
    const int stages = t.stages > 0 ? t.stages : 3;
    const size_t ring = (size_t)warps * stages * STAGE_BYTES + (size_t)warps * stages * 8 + 128 + 16;
    if (ring > SMEM_BUDGET || warps > 16) return cudaErrorInvalidValue;
    const size_t instr = (size_t)((s.I * 8 + 15) & ~15ll);
    const bool ismem = ring + instr <= SMEM_BUDGET;
    const size_t smem = ring + (ismem ? instr : 0);
    const int grid = num_sms * (t.ctas_per_sm > 0 ? t.ctas_per_sm : 1);
    ++*launches;
    return launch_tma2(stages, ismem, s, sd, grid, warps, smem, y, x, yscale, done, st);
  }
  const int threads = 256;
  int64_t blocks = (s.M + threads - 1) / threads;
  const int64_t cap = (int64_t)num_sms * 8;
  if (blocks > cap) blocks = cap;
  k_aprod2_rowthread<<<(unsigned)blocks, threads, 0, st>>>(s, y, x, yscale, done);
  ++*launches;
  return cudaGetLastError();
}

}  // namespace gsr
