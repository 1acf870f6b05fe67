// aprod2:  x[col(r,k)] += a[r][k] * (yscale * y[r])                  (Eq. 3)
// square = 1:  x[col(r,k)] += a[r][k]^2  (squared column norms: the same pass with the
//              coefficients squared on the fly and y = 1; y may be null)
#include "aprod_device.cuh"

namespace gsr {

// ---- variant 1 (default): TMA-staged row tiles, split by parameter block (aprod_device.cuh) ------
// PART: see lsqr_fused.cu
template <class REC, bool ASMEM, bool PART>
__global__ void __launch_bounds__(MAX_TMA_WARPS * 32, 1)
k_aprod2_tma(const __grid_constant__ CUtensorMap map, SysView s, int nstages, const double* __restrict__ y,
             double* __restrict__ x, double* __restrict__ gatt_il, InstrAcc ia, int use_tab, int tab_shift, int acc_part,
             const double* __restrict__ yscale, const int* done, int square) {
  if (done && *done) return;
  extern __shared__ char smem_raw[];
  char* smem = smem_align128(smem_raw);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  char* ring_mem = smem + (size_t)warp * nstages * STAGE_BYTES;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)nwarps * nstages * STAGE_BYTES);
  double* acc_s = reinterpret_cast<double*>(bars + nwarps * nstages + 2);
  if (!PART) acc_part = 0;
  uint32_t* tab_s = reinterpret_cast<uint32_t*>(acc_s + (ASMEM ? 0 : ((acc_part + 1) & ~1)));

  TileRing<REC> ring;
  const int64_t gw = (int64_t)blockIdx.x * nwarps + warp, W = (int64_t)gridDim.x * nwarps;
  ring.init(ring_mem, bars + warp * nstages, &map, s.vals, s.idx, s.M, gw, W, lane, nstages);
  const int64_t n_acc = ASMEM ? s.I : (PART ? acc_part : 0);   // accumulators privatised in shared memory: all, or the leading columns
  if (ASMEM || PART)
    for (int64_t i = threadIdx.x; i < n_acc; i += blockDim.x) acc_s[i] = 0.0;
  if (!ASMEM && use_tab) load_ins_tab(tab_s, ia, tab_shift);
  if (ASMEM || PART || use_tab) __syncthreads();
  ScatterCtx sc{x, gatt_il, x + s.oI, acc_s, (!ASMEM && use_tab) ? tab_s : nullptr, ia.base, tab_shift, (1 << tab_shift) - 1, acc_part};
  const AttLane al(lane);
  const double ys = yscale ? *yscale : 1.0;
  double gacc = 0.0;

  double ynext = (!square && gw < ring.n_tiles && gw * TILE_ROWS + lane < s.M) ? y[gw * TILE_ROWS + lane] : 1.0;
  for (int64_t t = gw; t < ring.n_tiles; t += W) {
    const int64_t row0 = t * TILE_ROWS;
    const int64_t r = row0 + lane;
    const bool valid = r < s.M;
    const double yv = valid ? ys * ynext : 0.0;
    {  // prefetch the next tile's y
      const int64_t rn = r + W * TILE_ROWS;
      if (!square) ynext = rn < s.M ? y[rn] : 0.0;
    }
    const int nvalid = (s.M - row0) < TILE_ROWS ? (int)(s.M - row0) : TILE_ROWS;
    char* tile = ring.acquire(t, lane);
    RowRegs row;
    load_row<REC>(tile, lane, valid, row);
    if (square) {
      // squared column norms of A as an operator: a column that repeats inside a row (instrumental slots only)
      // contributes (sum of its coefficients)^2 once -- summed in slot order into the first of its slots
      const int col[6] = {row.i0.z, row.i0.w, row.i1.x, row.i1.y, row.i1.z, row.i1.w};
      bool dup[6] = {false, false, false, false, false, false};
#pragma unroll
      for (int q = 0; q < 6; q++) {
        double sum = row.a[17 + q];
#pragma unroll
        for (int p = q + 1; p < 6; p++)
          if (!dup[q] && col[p] == col[q]) { sum += row.a[17 + p]; dup[p] = true; }
        row.a[17 + q] = dup[q] ? 0.0 : sum;
      }
#pragma unroll
      for (int k = 0; k < NSLOT; k++) row.a[k] *= row.a[k];
    }
    int ts[16];
    att_starts(tile, al, ts);
    __syncwarp();   // every lane holds its row: the exchange runs may be written
    att_products<REC>(tile, lane, row, yv);
    __syncwarp();
    att_scatter<REC>(tile, al, ts, gatt_il);
    astro_scatter<REC>(tile, lane, nvalid, valid, row, yv, sc.x, square != 0);
    gacc += scatter_rest<ASMEM, PART>(row, lane, valid, yv, sc);
    ring.release(lane);
  }
  if (ASMEM || PART) {
    __syncthreads();
    double* xins = x + s.oI;
    for (int64_t i = threadIdx.x; i < n_acc; i += blockDim.x) {
      const double v = acc_s[i];
      if (v != 0.0) atomicAdd(xins + i, v);
    }
  }
  if (s.G) {
    gacc = block_sum(gacc);
    if (threadIdx.x == 0) atomicAdd(x + s.oG, gacc);
  }
}

// x_instr[i] += sum over every set (die, copy) of the chunked accumulators; they are cleared for the next call.
// (The instrumental accumulator is replicated when it does not fit shared memory: 60,000 addresses
//  hit by 3e9 reductions are contention-bound at L2 -- 159 vs 193 Gadd/s measured with >= 6e5 addresses.)
__global__ void __launch_bounds__(256) k_fold_instr(double* __restrict__ xins, InstrAcc ia, int64_t I, const int* done) {
  if (done && *done) return;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < I; i += (int64_t)gridDim.x * blockDim.x) {
    double sum = 0.0;
    const int64_t ch = i >> INS_CHUNK_SHIFT, off = i & (INS_CHUNK - 1);
    for (int c = 0; c < ia.n_sets; c++) {
      double* p = ia.chunk_tab[(size_t)c * ia.n_chunks + ch] + off;
      sum += *p;
      *p = 0.0;
    }
    xins[i] += sum;
  }
}

cudaError_t launch_fold_instr(const SysView& s, const SideData& sd, double* x, const int* done, cudaStream_t st,
                              int64_t* launches) {
  int64_t b = (s.I + 255) / 256;
  if (b > 148 * 4) b = 148 * 4;
  k_fold_instr<<<(unsigned)b, 256, 0, st>>>(x + s.oI, sd.ins, s.I, done);
  ++*launches;
  return cudaGetLastError();
}

// ---- variant 0: one thread per row, fp64 reductions at L2 for every slot (simple cross-check, either record format).  square = 1: squared column norms (y = 1, coefficients squared; equal columns of a row
// summed first, reading R22) -----------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_aprod2_rowthread(SysView s, const double* __restrict__ y,
                                                          double* __restrict__ x, bool x_il,
                                                          const double* __restrict__ yscale,
                                                          const int* done, int square) {
  if (done && *done) return;
  const double ys = yscale ? *yscale : 1.0;
  double gsum = 0.0;
  for (int64_t r0 = blockIdx.x * (int64_t)blockDim.x; r0 < s.M; r0 += (int64_t)gridDim.x * blockDim.x) {
    const int64_t r = r0 + threadIdx.x;
    if (r < s.M) {
      const int4* ip = reinterpret_cast<const int4*>(s.idx + r * NIDX);
      const int4 i0 = __ldg(ip), i1 = __ldg(ip + 1);
      const double yr = square ? 1.0 : ys * y[r];
      double a[NSLOT];
      load_record(s, r, a);
      if (square) {
        const int col[6] = {i0.z, i0.w, i1.x, i1.y, i1.z, i1.w};
        bool dup[6] = {false, false, false, false, false, false};
#pragma unroll
        for (int q = 0; q < 6; q++) {
          double sum = a[17 + q];
#pragma unroll
          for (int p = q + 1; p < 6; p++)
            if (!dup[q] && col[p] == col[q]) { sum += a[17 + p]; dup[p] = true; }
          a[17 + q] = dup[q] ? 0.0 : sum;
        }
#pragma unroll
        for (int k = 0; k < NSLOT; k++) a[k] *= a[k];
      }
      double* xa = x + 5 * (int64_t)i0.x;
#pragma unroll
      for (int k = 0; k < 5; k++) atomicAdd(xa + k, a[k] * yr);
      const int64_t sa = x_il ? 1 : s.K, sj = x_il ? 3 : 1;   // attitude strides: axis, knot
      double* xt = x + s.oA + i0.y * sj;
#pragma unroll
      for (int ax = 0; ax < 3; ax++)
#pragma unroll
        for (int j = 0; j < 4; j++) atomicAdd(xt + ax * sa + j * sj, a[5 + 4 * ax + j] * yr);
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

// x_il = true: x is an LSQR-internal vector (attitude block interleaved) and is scattered into directly;
// otherwise the attitude products go to the zeroed side buffer sd.att_acc and are folded into x.
cudaError_t launch_aprod2(const SysView& s, const SideData& sd, const Tuning& t, int num_sms, const double* y,
                          double* x, bool x_il, const double* yscale, const int* done, cudaStream_t st,
                          int64_t* launches, int square) {
  if (s.M == 0) return cudaSuccess;
  if (t.aprod2_variant == 1 || (square && t.aprod2_variant != 0)) {
    const SmemPlan p = plan_smem(s, t, PLAN_APROD2);
    if (p.bytes > SMEM_BUDGET || p.warps > MAX_TMA_WARPS || p.warps < 1 || p.stages < 1) return cudaErrorInvalidValue;
    const int grid = num_sms * (t.ctas_per_sm > 0 ? t.ctas_per_sm : 1);
    const bool use_copies = !p.acc_smem && p.ins_tab && sd.ins.chunk_tab != nullptr && t.instr_copies != 0;
    const bool part = use_copies && p.acc_part > 0;
    auto k = s.cpr == NSLOT
                 ? (p.acc_smem ? k_aprod2_tma<Rec24, true, false> : (part ? k_aprod2_tma<Rec24, false, true> : k_aprod2_tma<Rec24, false, false>))
                 : (p.acc_smem ? k_aprod2_tma<Rec23, true, false> : (part ? k_aprod2_tma<Rec23, false, true> : k_aprod2_tma<Rec23, false, false>));
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.bytes);
    if (e != cudaSuccess) return e;
    InstrAcc ia = sd.ins;
    if (!t.die_local) ia.two_dies = false;
    k<<<grid, p.warps * 32, p.bytes, st>>>(sd.map, s, p.stages, y, x, x_il ? x + s.oA : sd.att_acc, ia,
                                            use_copies ? 1 : 0, p.tab_shift, part ? p.acc_part : 0, yscale, done, square);
    ++*launches;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (!x_il) {   // (never inside LSQR, so no `done` gate is needed)
      e = launch_att_fold(s, num_sms, x, sd.att_acc, st, launches);
      if (e != cudaSuccess) return e;
    }
    if (use_copies) return launch_fold_instr(s, sd, x, done, st, launches);
    return cudaSuccess;
  }
  const int threads = 256;
  int64_t blocks = (s.M + threads - 1) / threads;
  const int64_t cap = (int64_t)num_sms * 8;
  if (blocks > cap) blocks = cap;
  k_aprod2_rowthread<<<(unsigned)blocks, threads, 0, st>>>(s, y, x, x_il, yscale, done, square);
  ++*launches;
  return cudaGetLastError();
}

}  // namespace gsr
