// aprod2:  x[col(r,k)] += a[r][k] * (yscale * y[r])                  (Eq. 3)
#include "gsr_internal.cuh"

namespace gsr {

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

cudaError_t launch_aprod2(const SysView& s, const Tuning& t, int num_sms, const double* y, double* x,
                          const double* yscale, const int* done, cudaStream_t st, int64_t* launches) {
  if (s.M == 0) return cudaSuccess;
  const int threads = 256;
  int64_t blocks = (s.M + threads - 1) / threads;
  const int64_t cap = (int64_t)num_sms * 8;
  if (blocks > cap) blocks = cap;
  k_aprod2_rowthread<<<(unsigned)blocks, threads, 0, st>>>(s, y, x, yscale, done);
  ++*launches;
  return cudaGetLastError();
}

}  // namespace gsr
