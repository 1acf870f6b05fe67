// aprod2, deterministic debug variant (gsr_set_option("aprod2_variant", 2); "keep a
// deterministic (sorted-scatter) mode for debugging").  x[col(r,k)] += a[r][k] * (yscale * y[r])   (Eq. 3)
//
// The default kernels reduce with fp64 atomics, so their sums change in the last bits from run to run.  Here every
// sum has ONE fixed order that depends on the sizes only (not on the GPU, the grid or the timing):
//   astro  : rows are sorted by star, so the rows of a star are one contiguous range (found by binary search); one
//            thread owns a star and adds its rows in row order, starting from the value x already holds
//   shared : (attitude, instrumental, global) the rows are cut into C chunks of consecutive rows; chunk c is added up
//            by ONE thread, row by row in slot order, into its private copy of the shared columns; copy 0 starts from
//            the values x holds, the others from zero; then x[j] = copy_0[j] + copy_1[j] + ... in that order.
// No FMA contraction (__dmul_rn / __dadd_rn).  With C = 1 (option det_chunks = 1) the order is that of Eq. (3) written
// out as a loop -- row by row, slot by slot, from x's initial value -- so the result is bit-identical to any plain
// serial implementation of the definition, which is what makes the variant useful: a difference between the fast
// kernels and such an implementation can be split into "order of summation" and "anything else".  Slow by design (C <= 1024 threads do the shared part); not a timed path.
#include "aprod_device.cuh"

namespace gsr {

__device__ __forceinline__ int64_t first_row_of_star(const SysView& s, int64_t star) {
  int64_t lo = 0, hi = s.M;                  // first r with idx[r].star >= star
  while (lo < hi) {
    const int64_t mid = lo + ((hi - lo) >> 1);
    if (__ldg(s.idx + mid * NIDX) < star) lo = mid + 1;
    else hi = mid;
  }
  return lo;
}

__global__ void __launch_bounds__(128) k_aprod2_det_astro(SysView s, const double* __restrict__ y, double* __restrict__ x,
                                                          const double* __restrict__ yscale, const int* done) {
  if (done && *done) return;
  const double ys = yscale ? *yscale : 1.0;
  for (int64_t star = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; star < s.S; star += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r0 = first_row_of_star(s, star);
    if (r0 >= s.M || __ldg(s.idx + r0 * NIDX) != star) continue;     // no row of this section belongs to the star
    double acc[5];
#pragma unroll
    for (int k = 0; k < 5; k++) acc[k] = x[5 * star + k];
    for (int64_t r = r0; r < s.M && __ldg(s.idx + r * NIDX) == star; r++) {
      const double yr = __dmul_rn(ys, y[r]);
      const double* ap = s.vals + r * s.cpr;
#pragma unroll
      for (int k = 0; k < 5; k++) acc[k] = __dadd_rn(acc[k], __dmul_rn(ap[k], yr));
    }
#pragma unroll
    for (int k = 0; k < 5; k++) x[5 * star + k] = acc[k];
  }
}

// position of shared column j (0 <= j < ns, the ABI's order: attitude axis-major, instrumental, global) inside x
__device__ __forceinline__ int64_t shared_pos(const SysView& s, int64_t j, bool x_il) {
  if (x_il && j < 3 * s.K) {
    const int64_t ax = j / s.K, t = j - ax * s.K;
    return s.oA + 3 * t + ax;
  }
  return s.oA + j;
}

// copy 0 <- the shared columns of x ; copies 1 .. C-1 <- 0
__global__ void __launch_bounds__(256) k_aprod2_det_init(SysView s, const double* __restrict__ x, bool x_il,
                                                         double* __restrict__ part, int C, const int* done) {
  if (done && *done) return;
  const int64_t ns = s.n - s.oA, total = ns * C;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x)
    part[i] = i < ns ? x[shared_pos(s, i, x_il)] : 0.0;
}

__global__ void __launch_bounds__(128) k_aprod2_det_shared(SysView s, const double* __restrict__ y, double* __restrict__ part,
                                                           int C, int64_t rows_per_chunk, const double* __restrict__ yscale,
                                                           const int* done) {
  if (done && *done) return;
  const int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (c >= C) return;
  const double ys = yscale ? *yscale : 1.0;
  const int64_t ns = s.n - s.oA;
  double* P = part + c * ns;
  const int64_t r_end = (c + 1) * rows_per_chunk < s.M ? (c + 1) * rows_per_chunk : s.M;
  for (int64_t r = c * rows_per_chunk; r < r_end; r++) {
    const int32_t* rec = s.idx + r * NIDX;
    const double* ap = s.vals + r * s.cpr;
    const double yr = __dmul_rn(ys, y[r]);
    const int64_t t = rec[1];
    for (int ax = 0; ax < 3; ax++)
      for (int j = 0; j < 4; j++) {
        double* p = P + ax * s.K + t + j;
        *p = __dadd_rn(*p, __dmul_rn(ap[5 + 4 * ax + j], yr));
      }
    for (int q = 0; q < 6; q++) {
      double* p = P + 3 * s.K + rec[2 + q];
      *p = __dadd_rn(*p, __dmul_rn(ap[17 + q], yr));
    }
    if (s.G) {
      double* p = P + 3 * s.K + s.I;
      *p = __dadd_rn(*p, __dmul_rn(ap[23], yr));
    }
  }
}

// x[shared column j] = copy_0[j] + copy_1[j] + ... + copy_{C-1}[j], in that order
__global__ void __launch_bounds__(256) k_aprod2_det_fold(SysView s, const double* __restrict__ part, int C,
                                                         double* __restrict__ x, bool x_il, const int* done) {
  if (done && *done) return;
  const int64_t ns = s.n - s.oA;
  for (int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; j < ns; j += (int64_t)gridDim.x * blockDim.x) {
    double sum = part[j];
    for (int c = 1; c < C; c++) sum = __dadd_rn(sum, part[(int64_t)c * ns + j]);
    x[shared_pos(s, j, x_il)] = sum;
  }
}

// det_part: C * (n - 5S) doubles of scratch (gsr_api.cu allocates it on first use)
cudaError_t launch_aprod2_det(const SysView& s, double* det_part, int C, int num_sms, const double* y, double* x, bool x_il,
                              const double* yscale, const int* done, cudaStream_t st, int64_t* launches) {
  if (s.M == 0) return cudaSuccess;
  if (!det_part || C < 1) return cudaErrorInvalidValue;
  const int64_t ns = s.n - s.oA;
  int64_t b = (s.S + 127) / 128;
  if (b > (int64_t)num_sms * 16) b = (int64_t)num_sms * 16;
  k_aprod2_det_astro<<<(unsigned)b, 128, 0, st>>>(s, y, x, yscale, done);
  ++*launches;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  int64_t bi = (ns * C + 255) / 256;
  if (bi > (int64_t)num_sms * 16) bi = (int64_t)num_sms * 16;
  k_aprod2_det_init<<<(unsigned)bi, 256, 0, st>>>(s, x, x_il, det_part, C, done);
  ++*launches;
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  const int64_t rows_per_chunk = (s.M + C - 1) / C;
  k_aprod2_det_shared<<<(unsigned)((C + 127) / 128), 128, 0, st>>>(s, y, det_part, C, rows_per_chunk, yscale, done);
  ++*launches;
  if ((e = cudaGetLastError()) != cudaSuccess) return e;
  int64_t bf = (ns + 255) / 256;
  if (bf > (int64_t)num_sms * 16) bf = (int64_t)num_sms * 16;
  k_aprod2_det_fold<<<(unsigned)bf, 256, 0, st>>>(s, det_part, C, x, x_il, done);
  ++*launches;
  return cudaGetLastError();
}

}  // namespace gsr
