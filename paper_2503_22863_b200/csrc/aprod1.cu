// aprod1:  y[r] = c1 * sum_k a[r][k] * x[col(r,k)] + c0 * y[r]      (Eq. 2)
// with the LSQR u-update and ||u||^2 fused in.
#include "gsr_internal.cuh"
#include "tma.cuh"

namespace gsr {

// ---- variant 1 (default): TMA-staged row tiles, one warp per tile, lane per row -----------------
// Data movement per row: 192 B coefficients + 32 B index record arrive by TMA (tma.cuh); the lane
// reads them conflict-free from shared memory.  Gathers from x:
//   astro  : x[5*star .. +4]   (rows are sorted by star: the lanes of a warp share 1-2 stars)
//   att    : ONE 32-byte load per axis from the expanded window table xw[ax][t] = x[t..t+3]
//            (k_expand_att below; 12 scalar gathers per row would saturate the L1 tag pipe)
//   instr  : shared-memory copy of the instrumental slice when it fits, else L2 gathers
//   global : one register.
// y[r] <- (A x)[r] + c0 * y[r], sum of squares accumulated for ||u|| (LSQR fusion).
__device__ __forceinline__ void ld_nc_v4(const double* p, double& a, double& b, double& c, double& d) {
  asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}

template <int STAGES, bool INSTR_SMEM>
__global__ void __launch_bounds__(512, 1)
k_aprod1_tma(const __grid_constant__ CUtensorMap map, SysView s, const double* __restrict__ x,
             const double* __restrict__ xw, double* __restrict__ y, const double* __restrict__ c0p,
             double* sumsq, int* done) {
  if (done) {
    const int d = *done;
    if (d) {  // LSQR already stopped: no-op (and latch "update pending" 2 -> 1, see k_step_scalars)
      if (d == 2 && blockIdx.x == 0 && threadIdx.x == 0) *done = 1;
      return;
    }
  }
  extern __shared__ char smem_raw[];
  char* smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  char* ring_mem = smem + (size_t)warp * STAGES * STAGE_BYTES;
  double* xi_s = reinterpret_cast<double*>(smem + (size_t)nwarps * STAGES * STAGE_BYTES);
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<char*>(xi_s) + (INSTR_SMEM ? ((s.I * 8 + 15) & ~15ll) : 0));

  TileRing<STAGES> ring;
  const int64_t gw = (int64_t)blockIdx.x * nwarps + warp, W = (int64_t)gridDim.x * nwarps;
  ring.init(ring_mem, bars + warp * STAGES, &map, s.idx, s.M, gw, W, lane);
  if (INSTR_SMEM) {
    for (int64_t i = threadIdx.x; i < s.I; i += blockDim.x) xi_s[i] = __ldg(x + s.oI + i);
    __syncthreads();
  }
  const double c0 = c0p ? *c0p : 1.0;
  const double xg = s.G ? __ldg(x + s.oG) : 0.0;
  const int64_t Kw = s.K - 3;           // windows per axis in xw
  const double* xi_g = x + s.oI;
  double sq = 0.0;

  for (int64_t t = gw; t < ring.n_tiles; t += W) {
    const int64_t r = t * TILE_ROWS + lane;
    const bool valid = r < s.M;
    const double yin = valid ? y[r] : 0.0;
    const char* tile = ring.acquire();
    const double2* ap = reinterpret_cast<const double2*>(tile + lane * (ROW_STRIDE_D * 8));
    const int4* ip = reinterpret_cast<const int4*>(tile + COEF_TILE_BYTES + lane * 32);
    int4 i0 = ip[0], i1 = ip[1];
    if (!valid) { i0 = make_int4(0, 0, 0, 0); i1 = i0; }   // tail lanes: coefficients are zero-filled
    double a[NSLOT];
#pragma unroll
    for (int q = 0; q < NSLOT / 2; q++) {
      const double2 v = ap[q];
      a[2 * q] = v.x;
      a[2 * q + 1] = v.y;
    }
    // gathers
    const double* xa = x + 5 * (int64_t)i0.x;
    double g[NSLOT - 1];
#pragma unroll
    for (int k = 0; k < 5; k++) g[k] = __ldg(xa + k);
    const double* w0 = xw + (int64_t)i0.y * 4;
    ld_nc_v4(w0, g[5], g[6], g[7], g[8]);
    ld_nc_v4(w0 + Kw * 4, g[9], g[10], g[11], g[12]);
    ld_nc_v4(w0 + Kw * 8, g[13], g[14], g[15], g[16]);
    if (INSTR_SMEM) {
      g[17] = xi_s[i0.z]; g[18] = xi_s[i0.w]; g[19] = xi_s[i1.x];
      g[20] = xi_s[i1.y]; g[21] = xi_s[i1.z]; g[22] = xi_s[i1.w];
    } else {
      g[17] = __ldg(xi_g + i0.z); g[18] = __ldg(xi_g + i0.w); g[19] = __ldg(xi_g + i1.x);
      g[20] = __ldg(xi_g + i1.y); g[21] = __ldg(xi_g + i1.z); g[22] = __ldg(xi_g + i1.w);
    }
    double acc0 = a[23] * xg, acc1 = 0.0, acc2 = 0.0;
#pragma unroll
    for (int k = 0; k < 21; k += 3) {
      acc0 = fma(a[k], g[k], acc0);
      acc1 = fma(a[k + 1], g[k + 1], acc1);
      acc2 = fma(a[k + 2], g[k + 2], acc2);
    }
    acc0 = fma(a[21], g[21], acc0);
    acc1 = fma(a[22], g[22], acc1);
    const double out = fma(c0, yin, (acc0 + acc1) + acc2);
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

// xw[(ax*(K-3) + t)*4 + j] = x[oA + ax*K + t + j]   (t = 0 .. K-4): every possible 4-knot run as one
// aligned 32-byte record, rebuilt from x at every aprod1 call (3K reads, 12K writes: << the matrix).
__global__ void __launch_bounds__(256) k_expand_att(const double* __restrict__ xatt, int64_t K, double* __restrict__ xw,
                                                    const int* done) {
  if (done && *done) return;
  const int64_t Kw = K - 3, total = 3 * Kw;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
    const int64_t ax = i / Kw, t = i - ax * Kw;
    const double* p = xatt + ax * K + t;
    double2* o = reinterpret_cast<double2*>(xw + i * 4);
    o[0] = make_double2(__ldg(p), __ldg(p + 1));
    o[1] = make_double2(__ldg(p + 2), __ldg(p + 3));
  }
}

// ---- variant 0: one thread per row, direct global loads (first correct path) -----------------
__global__ void __launch_bounds__(256) k_aprod1_rowthread(SysView s, const double* __restrict__ x,
                                                          double* __restrict__ y,
                                                          const double* __restrict__ c0p,
                                                          double* sumsq, int* done) {
  if (done) {
    const int d = *done;
    if (d) {  // LSQR already stopped: no-op (and latch "update pending" 2 -> 1, see k_step_scalars)
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

template <int STAGES, bool INSTR_SMEM>
static cudaError_t launch_tma1(const SysView& s, const SideData& sd, int grid, int warps, size_t smem,
                               const double* x, double* y, const double* c0, double* sumsq, int* done,
                               cudaStream_t st) {
  auto k = k_aprod1_tma<STAGES, INSTR_SMEM>;
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k<<<grid, warps * 32, smem, st>>>(sd.map, s, x, sd.xw, y, c0, sumsq, done);
  return cudaGetLastError();
}

cudaError_t launch_aprod1(const SysView& s, const SideData& sd, const Tuning& t, int num_sms, const double* x,
                          double* y, const double* c0, double* sumsq, int* done, cudaStream_t st,
                          int64_t* launches) {
  if (s.M == 0) return cudaSuccess;
  if (t.aprod1_variant == 1) {
    // expanded attitude windows, then the streaming kernel
    const int64_t total = 3 * (s.K - 3);
    int64_t eb = (total + 255) / 256;
    if (eb > num_sms * 8) eb = num_sms * 8;
    k_expand_att<<<(unsigned)eb, 256, 0, st>>>(x + s.oA, s.K, sd.xw, done);
    ++*launches;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const int warps = t.warps > 0 ? t.warps : 8;
    const int stages = t.stages > 0 ? t.stages : 3;
    const size_t ring = (size_t)warps * stages * STAGE_BYTES + (size_t)warps * stages * 8 + 128 + 16;
    if (ring > SMEM_BUDGET || warps > 16) return cudaErrorInvalidValue;
    const size_t instr = (size_t)((s.I * 8 + 15) & ~15ll);
    const bool ismem = ring + instr <= SMEM_BUDGET;
    const size_t smem = ring + (ismem ? instr : 0);
    const int grid = num_sms * (t.ctas_per_sm > 0 ? t.ctas_per_sm : 1);
    ++*launches;
#define GSR_A1(ST) (ismem ? launch_tma1<ST, true>(s, sd, grid, warps, smem, x, y, c0, sumsq, done, st) \
                          : launch_tma1<ST, false>(s, sd, grid, warps, smem, x, y, c0, sumsq, done, st))
    switch (stages) {
      case 2: return GSR_A1(2);
      case 4: return GSR_A1(4);
      default: return GSR_A1(3);
    }
#undef GSR_A1
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
