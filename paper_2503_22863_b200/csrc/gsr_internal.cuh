// Internal declarations of libgsr (not part of the ABI; the ABI is include/gsr.h).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "gsr.h"

namespace gsr {

constexpr int NSLOT = 24;  // PAPER.md:39 : 5 astro + 12 attitude + 6 instrumental + 1 global
constexpr int NIDX = 8;    // {star, att_start, instr[6]}

// Read-only view of a system, passed by value to kernels.
struct SysView {
  const double* vals;   // M x 24
  const int32_t* idx;   // M x 8
  int64_t M, S, K, I;
  int32_t G;
  int64_t oA, oI, oG, n;  // block offsets in x: attitude, instrumental, global; n unknowns
  int32_t cpr;            // coefficients stored per row = record stride in doubles: 24, or 23 (GSR_LAYOUT_COEFF23, G = 0)
};

// Device-resident LSQR scalars.  One instance per system.
struct DevScalars {
  double alpha, beta, rhobar, phibar, bnorm, rnorm, arnorm, anorm, acond, ddnorm, xnorm, xxnorm,
      z, cs2, sn2;
  double usq, vsq, wsq;          // sum-of-squares accumulators (atomically added by kernels)
  double c0_u;                   // aprod1 fused update: u_hat <- A v + c0_u * u_hat  (= -alpha/beta)
  double s_y;                    // aprod2 input scale (1/beta: u = u_hat / beta is never stored)
  double t1, t2, inv_alpha;      // x/w/v update coefficients of the current iteration
  double inv_rho;                // 1 / rho of the current plane rotation (variance update)
  long long itn;
  int istop;
  int done;                      // 1 once a stopping rule fired: later kernels are no-ops
};

struct Tuning {
  int aprod1_variant = 1;  // 1 = TMA-staged tiles (default), 0 = one thread per row (simple)
  int aprod2_variant = 1;  // 1 = TMA-staged tiles, split by parameter block (default), 0 = one thread per row,
                           // 2 = deterministic debug variant (aprod2_det.cu): fixed summation order, bit-reproducible
  int det_chunks = 0;      // variant 2: row chunks with a private copy of the shared columns each (0 = as many as fit 256 MB,
                           // at most 1024; 1 = Eq. (3) as a plain loop: row by row, slot by slot)
  int ctas_per_sm = 0;     // 0 = default of the variant
  int warps = 0;           // warps per CTA of the TMA kernels (0 = the planner's choice: 12, down to 8 if that lets the tables fit)
  int stages = 0;          // ring depth per warp (0 = default 2)
  int check_every = 16;    // LSQR iterations between host polls of the stop flag
  int instr_copies = 1;    // replicate the instrumental accumulator in global memory when it cannot be privatised
  int fused = 1;           // LSQR: one fused pass over the matrix per iteration (lsqr_fused.cu)
  int graph = 1;           // LSQR: replay batches of iterations of small (launch-bound) systems as a CUDA graph
  int acc_smem = 1;        // instrumental accumulators: 1 = privatised in shared memory when they fit, 0 = always L2 copies
  int die_local = 1;       // L2 instrumental accumulators: 1 = each CTA reduces into a copy homed on its own die, 0 = die-0 copies for all (control)
  int gather_smem = 1;     // instrumental slice of x: 1 = staged in shared memory when it fits, 0 = L1/L2 gathers
  // L2 instrumental accumulators: leading columns privatised in whatever shared memory is left (-1 = all that fit,
  // 0 = none, n = at most n); kernels instantiated with PART = true.  Measured at the C4 shape in a first form with a
  // branch per slot (profiles/r02_summary.md): standalone aprod 2 at 2e7 rows 1.363 -> 1.222 ms with 6,000 of the
  // 60,000 columns in shared memory, at 5e8 rows 36.8 -> 36.4 ms with 4,000; the fused pass lost 15-40 %.  The
  // committed form (predicated reductions) has not run on hardware (the GPU pool closed first), so both are OFF by
  // default: the default kernels are the PART = false instances, instruction for instruction those measured in round 1.
  int acc_part = 0;        // standalone aprod 2
  int acc_part_fused = 0;  // fused LSQR pass
  int tab_private = 0;     // die-local chunk table: 1 = one copy per shared-memory bank (no LDS bank conflicts; measured -0.4 %:
                           // shared-memory wavefronts are not what bounds the pass), 0 = one copy (leaves 15 KB to acc_part)
};

// Replicated instrumental accumulators for systems whose slice does not fit shared memory.
// B200 is two dies; an fp64 reduction executes in the L2 slice that is the HOME of its address, and the
// home die of an address is a hash of its physical 4 KB granule.  Measured on this part (gsr_api.cu,
// probe_homes): an atomic to a near-die granule returns in ~330 cycles, to a far-die granule in ~720, and a
// far reduction costs a second L2 tag lookup on the way (`lts__t_requests_srcunit_ltcfabric`).  So the
// accumulators are built from 4 KB chunks (512 doubles) whose home die was probed at gsr_create, one set of
// copies per die, and every CTA reduces into a copy homed on the die its SM sits on.
constexpr int INS_CHUNK = 512;        // doubles per chunk (4 KB granule)
constexpr int INS_CHUNK_SHIFT = 9;
constexpr int SMID_SLOTS = 1024;      // entries of the SM-id -> die table
struct InstrAcc {
  double** chunk_tab = nullptr;  // device: [n_sets][n_chunks] chunk pointers; set = die * copies_per_die + copy
  int* sm_die = nullptr;         // device: [SMID_SLOTS] die (0 / 1) of an SM id
  void* pool = nullptr;          // device: the chunk pool (zero between calls)
  double* base = nullptr;        // first 4 KB-aligned chunk of the pool (chunk pointers are base + 512 * index)
  int copies_per_die = 0, n_chunks = 0, n_sets = 0;   // n_sets = 2 * copies_per_die (copies_per_die if one die was seen)
  bool two_dies = false;
};

// Side structures owned by the library (built in gsr_create).
struct SideData {
  CUtensorMap map;         // 48 x floor(M/2) fp64 tensor (row pairs), box 50 x 16 (tma.cuh)
  double* att_il = nullptr;   // 3K: interleaved copy of x's attitude block (standalone aprod 1)
  double* att_acc = nullptr;  // 3K: interleaved attitude accumulator, zero between calls (standalone aprod 2)
  InstrAcc ins;               // die-local replicated instrumental accumulators (global memory, L2-resident)
  double* det_part = nullptr; // aprod2 variant 2: det_cap private copies of the shared columns (allocated on first use)
  int det_cap = 0;
};

#ifndef GSR_MAX_TMA_WARPS
#define GSR_MAX_TMA_WARPS 12
#endif
constexpr int MAX_TMA_WARPS = GSR_MAX_TMA_WARPS;   // warps per CTA of the TMA kernels (register budget 65536 / 384 = 170)
constexpr size_t SMEM_BUDGET = 227 * 1024 - 512;   // dynamic shared memory we allow one CTA (static: block_sum)

// Launchers (each returns cudaGetLastError()).  Null coefficient pointers mean 1.0 / "no".
// *_il = the n-vector is LSQR-internal: its attitude block is interleaved, il[3*t + ax] (aprod_device.cuh).
//   aprod1: y[r] = c1 * (A x)[r] + c0 * y[r]      (c0 = c1 = 1 -> Eq. 2);  *sumsq += sum y[r]^2
cudaError_t launch_aprod1(const SysView& s, const SideData& sd, const Tuning& t, int num_sms, const double* x,
                          bool x_il, double* y, const double* c0, double* sumsq, int* done, cudaStream_t st,
                          int64_t* launches);
//   aprod2: x += A^T (yscale * y)
cudaError_t launch_aprod2(const SysView& s, const SideData& sd, const Tuning& t, int num_sms, const double* y,
                          double* x, bool x_il, const double* yscale, const int* done, cudaStream_t st,
                          int64_t* launches, int square = 0);
//   aprod2, deterministic debug variant (aprod2_det.cu): C chunks of rows, det_part = C * (n - 5S) doubles of scratch
cudaError_t launch_aprod2_det(const SysView& s, double* det_part, int C, int num_sms, const double* y, double* x, bool x_il,
                              const double* yscale, const int* done, cudaStream_t st, int64_t* launches);
cudaError_t launch_validate(const SysView& s, int* flag, cudaStream_t st, int64_t* launches);
//   fused LSQR step: uh <- A v + c0 uh ; g += A^T uh ; usq += ||uh||^2   (lsqr_fused.cu; v, g internal layout)
cudaError_t launch_lsqr_fused(const SysView& s, const SideData& sd, const Tuning& t, int num_sms, const double* v,
                              double* uh, double* g, const double* c0, double* usq, int* done, cudaStream_t st,
                              int64_t* launches);
cudaError_t launch_att_to_il(const SysView& s, int num_sms, const double* x_std, double* il, const int* done,
                             cudaStream_t st, int64_t* launches);
cudaError_t launch_att_fold(const SysView& s, int num_sms, double* x_std, double* il, cudaStream_t st, int64_t* launches);
cudaError_t launch_att_from_il(const SysView& s, int num_sms, const double* il, double* dst_std_att, cudaStream_t st,
                               int64_t* launches);
cudaError_t launch_fold_instr(const SysView& s, const SideData& sd, double* x, const int* done, cudaStream_t st,
                              int64_t* launches);
// (n_sq: how many leading elements enter the kernel's sum of squares; -1 = all n.  Only a row-sharded solve passes less.)
cudaError_t lsqr_launch_vcombine(double* v, const double* g, int64_t n, DevScalars* sc, const double* dinv,
                                 cudaStream_t st, int64_t* launches, int64_t n_sq = -1);

// LSQR vector / scalar kernels (lsqr_kernels.cu)
cudaError_t lsqr_launch_init_u(const double* b, double* u, int64_t M, DevScalars* sc, cudaStream_t st, int64_t* launches);
cudaError_t lsqr_launch_init_s1(DevScalars* sc, cudaStream_t st, int64_t* launches);
cudaError_t lsqr_launch_sumsq_v(double* v, int64_t n, DevScalars* sc, const double* dinv, cudaStream_t st,
                                int64_t* launches, int64_t n_sq = -1);
cudaError_t lsqr_launch_init_s2(DevScalars* sc, cudaStream_t st, int64_t* launches);
cudaError_t lsqr_launch_init_vw(double* v, double* w, double* x, int64_t n, DevScalars* sc, double* vs,
                                const double* dinv, double* var, cudaStream_t st, int64_t* launches, int64_t n_sq = -1);
cudaError_t lsqr_launch_vscale(double* v, int64_t n, DevScalars* sc, cudaStream_t st, int64_t* launches);
cudaError_t lsqr_launch_step_scalars(DevScalars* sc, int64_t itnlim, double atol, double btol, double conlim,
                                     cudaStream_t st, int64_t* launches);
cudaError_t lsqr_launch_update(double* v, double* w, double* x, int64_t n, DevScalars* sc, double* vs,
                               const double* dinv, double* var, cudaStream_t st, int64_t* launches, int64_t n_sq = -1);
cudaError_t lsqr_launch_cov_update(const SysView& s, const double* w, const DevScalars* sc, const int64_t* j1,
                                   const int64_t* j2, int64_t n_pairs, double* cov, cudaStream_t st, int64_t* launches);
cudaError_t lsqr_launch_cov_unscale(const SysView& s, const double* dinv, const int64_t* j1, const int64_t* j2,
                                    int64_t n_pairs, double* cov, cudaStream_t st, int64_t* launches);
cudaError_t lsqr_launch_check_pairs(const int64_t* j1, const int64_t* j2, int64_t n_pairs, int64_t n, int* bad,
                                    cudaStream_t st, int64_t* launches);
cudaError_t lsqr_launch_colnorm_finish(double* d, int64_t n, int mode, cudaStream_t st, int64_t* launches);
cudaError_t lsqr_launch_scale_by(double* dst, const double* src, const double* s, int64_t n, int power, cudaStream_t st,
                                 int64_t* launches);
cudaError_t lsqr_launch_export_u(const double* uhat, double* u, int64_t M, const DevScalars* sc, cudaStream_t st, int64_t* launches);
// row-sharded solve: which partial sums travel with the exchange buffer (lsqr_kernels.cu, k_shard_xfer)
enum { SHARD_X_NONE = 0, SHARD_X_USQ = 1, SHARD_X_VSQ = 2, SHARD_X_USQ_WSQ = 3 };
cudaError_t lsqr_launch_shard_xfer(double* vec, int64_t ns, DevScalars* sc, double* xbuf, int what, int unpack,
                                   cudaStream_t st, int64_t* launches);

// ---- device helpers -----------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Block-wide sum (blockDim.x multiple of 32, <= 1024); result valid in thread 0.
__device__ __forceinline__ double block_sum(double v) {
  __shared__ double part[32];
  v = warp_sum(v);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) part[w] = v;
  __syncthreads();
  const int nw = (blockDim.x + 31) >> 5;
  v = (threadIdx.x < nw) ? part[threadIdx.x] : 0.0;
  if (w == 0) v = warp_sum(v);
  return v;
}

}  // namespace gsr
