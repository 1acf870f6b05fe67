// aprod1:  y[r] = c1 * sum_k a[r][k] * x[col(r,k)] + c0 * y[r]      (Eq. 2)
// with the LSQR u-update and ||u||^2 fused in.
#include "gsr_internal.cuh"

namespace gsr {

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

cudaError_t launch_aprod1(const SysView& s, const Tuning& t, int num_sms, const double* x, double* y,
                          const double* c0, double* sumsq, int* done, cudaStream_t st,
                          int64_t* launches) {
  if (s.M == 0) return cudaSuccess;
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
