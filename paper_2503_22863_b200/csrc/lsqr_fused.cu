// One LSQR bidiagonalisation step in ONE pass over the matrix.
//
// Paige-Saunders (refs [29,30]):  beta u' = A v - alpha u ;  alpha' v' = A^T u' - beta v.
// Row r's contribution to A^T u' needs only u'[r], which depends only on row r:
//     uh[r] <- a_r . v + c0 * uh[r]          (uh = un-normalised u; c0 = -alpha/beta_prev)   "aprod 1"
//     g     += a_r^T * uh[r]                 (g zeroed before the pass)                       "aprod 2"
//     usq   += uh[r]^2
// and afterwards, with beta = sqrt(usq):  v' (un-normalised) = g / beta - beta v   (n-length kernel).
// Same arithmetic as running aprod1 then aprod2, but the 224 bytes of row r are streamed from HBM
// once per iteration instead of twice, and staged / read from shared memory once.
#include "aprod_device.cuh"

namespace gsr {

// v and g are LSQR-internal n-vectors: their attitude blocks are in the interleaved layout (aprod_device.cuh).
// PART: with the L2 instrumental accumulators, the leading acc_part columns are accumulated in shared memory instead
// (a template parameter: the kernel without them carries none of that code).
template <class REC, bool GSMEM, bool ASMEM, bool PART>
__global__ void __launch_bounds__(MAX_TMA_WARPS * 32, 1)
k_lsqr_fused(const __grid_constant__ CUtensorMap map, SysView s, int nstages, const double* __restrict__ v,
             double* __restrict__ uh, double* __restrict__ g, InstrAcc ia, int use_tab, int tab_shift, int acc_part,
             const double* __restrict__ c0p, double* usq, int* done) {
  {
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
  double* acc_s = reinterpret_cast<double*>(bars + nwarps * nstages + 2);
  if (!PART) acc_part = 0;
  double* xi_s = acc_s + (ASMEM ? ((s.I + 1) & ~1ll) : ((acc_part + 1) & ~1));
  uint32_t* tab_s = reinterpret_cast<uint32_t*>(xi_s + (GSMEM ? ((s.I + 1) & ~1ll) : 0));

  TileRing<REC> ring;
  const int64_t gw = (int64_t)blockIdx.x * nwarps + warp, W = (int64_t)gridDim.x * nwarps;
  ring.init(ring_mem, bars + warp * nstages, &map, s.vals, s.idx, s.M, gw, W, lane, nstages);
  const int64_t n_acc = ASMEM ? s.I : (PART ? acc_part : 0);   // accumulators privatised in shared memory: all, or the leading columns
  if (ASMEM || PART)
    for (int64_t i = threadIdx.x; i < n_acc; i += blockDim.x) acc_s[i] = 0.0;
  if (GSMEM)
    for (int64_t i = threadIdx.x; i < s.I; i += blockDim.x) xi_s[i] = __ldg(v + s.oI + i);
  if (!ASMEM && use_tab) load_ins_tab(tab_s, ia, tab_shift);
  if (ASMEM || PART || GSMEM || use_tab) __syncthreads();
  const double* att_il = v + s.oA;
  GatherCtx gc{v, att_il, xi_s, v + s.oI, s.G ? __ldg(v + s.oG) : 0.0};
  ScatterCtx sc{g, g + s.oA, g + s.oI, acc_s, (!ASMEM && use_tab) ? tab_s : nullptr, ia.base, tab_shift, (1 << tab_shift) - 1, acc_part};
  const AttLane al(lane);
  const double c0 = *c0p;
  double sq = 0.0, gacc = 0.0;

  double unext = (gw < ring.n_tiles && gw * TILE_ROWS + lane < s.M) ? uh[gw * TILE_ROWS + lane] : 0.0;
  for (int64_t t = gw; t < ring.n_tiles; t += W) {
    const int64_t row0 = t * TILE_ROWS;
    const int64_t r = row0 + lane;
    const bool valid = r < s.M;
    const double uin = unext;
    {  // prefetch the next tile's u: a DRAM round trip that would otherwise sit on every tile's critical path
      const int64_t rn = r + W * TILE_ROWS;
      unext = rn < s.M ? uh[rn] : 0.0;
    }
    const int nvalid = (s.M - row0) < TILE_ROWS ? (int)(s.M - row0) : TILE_ROWS;
    char* tile = ring.acquire(t, lane);
    RowRegs row;
    load_row<REC>(tile, lane, valid, row);
    int ts[16];
    att_starts(tile, al, ts);
    __syncwarp();   // every lane holds its row: the exchange runs may be written
    att_gather<REC>(tile, al, ts, att_il);
    const double rest = row_dot_rest<GSMEM>(row, gc);
    __syncwarp();
    double out = fma(c0, uin, att_dot_row<REC>(tile, lane, row) + rest);
    if (valid) {
      uh[r] = out;
      sq = fma(out, out, sq);
    } else {
      out = 0.0;
    }
    att_products<REC>(tile, lane, row, out);
    __syncwarp();
    att_scatter<REC>(tile, al, ts, sc.gatt_il);
    astro_scatter<REC>(tile, lane, nvalid, valid, row, out, sc.x);
    gacc += scatter_rest<ASMEM, PART>(row, lane, valid, out, sc);
    ring.release(lane);
  }
  if (ASMEM || PART) {
    __syncthreads();
    double* gins = g + s.oI;
    for (int64_t i = threadIdx.x; i < n_acc; i += blockDim.x) {
      const double a = acc_s[i];
      if (a != 0.0) atomicAdd(gins + i, a);
    }
  }
  sq = block_sum(sq);
  if (threadIdx.x == 0) atomicAdd(usq, sq);
  if (s.G) {
    __syncthreads();
    gacc = block_sum(gacc);
    if (threadIdx.x == 0) atomicAdd(g + s.oG, gacc);
  }
}

// fused pass ; [fold instrumental copies into g]
cudaError_t launch_lsqr_fused(const SysView& s, const SideData& sd, const Tuning& t, int num_sms, const double* v,
                              double* uh, double* g, const double* c0, double* usq, int* done, cudaStream_t st,
                              int64_t* launches) {
  if (s.M == 0) return cudaSuccess;
  const SmemPlan p = plan_smem(s, t, PLAN_FUSED);
  if (p.bytes > SMEM_BUDGET || p.warps > MAX_TMA_WARPS || p.warps < 1 || p.stages < 1) return cudaErrorInvalidValue;
  const int grid = num_sms * (t.ctas_per_sm > 0 ? t.ctas_per_sm : 1);
  const bool use_copies = !p.acc_smem && p.ins_tab && sd.ins.chunk_tab != nullptr && t.instr_copies != 0;
  void (*k)(const CUtensorMap, SysView, int, const double*, double*, double*, InstrAcc, int, int, int, const double*, double*, int*);
  const bool part = use_copies && p.acc_part > 0;
  if (s.cpr == NSLOT) {
    if (p.gather_smem) k = p.acc_smem ? k_lsqr_fused<Rec24, true, true, false> : (part ? k_lsqr_fused<Rec24, true, false, true> : k_lsqr_fused<Rec24, true, false, false>);
    else k = p.acc_smem ? k_lsqr_fused<Rec24, false, true, false> : (part ? k_lsqr_fused<Rec24, false, false, true> : k_lsqr_fused<Rec24, false, false, false>);
  } else {
    if (p.gather_smem) k = p.acc_smem ? k_lsqr_fused<Rec23, true, true, false> : (part ? k_lsqr_fused<Rec23, true, false, true> : k_lsqr_fused<Rec23, true, false, false>);
    else k = p.acc_smem ? k_lsqr_fused<Rec23, false, true, false> : (part ? k_lsqr_fused<Rec23, false, false, true> : k_lsqr_fused<Rec23, false, false, false>);
  }
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.bytes);
  if (e != cudaSuccess) return e;
  ++*launches;
  InstrAcc ia = sd.ins;
  if (!t.die_local) ia.two_dies = false;
  k<<<grid, p.warps * 32, p.bytes, st>>>(sd.map, s, p.stages, v, uh, g, ia, use_copies ? 1 : 0, p.tab_shift, part ? p.acc_part : 0, c0, usq, done);
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (use_copies) return launch_fold_instr(s, sd, g, done, st, launches);
  return cudaSuccess;
}

}  // namespace gsr
