/*
 * gsr.h -- C ABI of the B200-native AVU-GSR hot path (aprod1, aprod2, LSQR).
 *
 * The operations are the ones the paper states (arxiv 2503.22863, /root/reference/PAPER.md):
 *   the system  A x = b                     PAPER.md:37   Sec. 2, Eq. (1)
 *   the storage: <= 24 non-zeros per row,   PAPER.md:39   Sec. 2 (N_Astro=5, N_Att=12,
 *                fp64                                      N_Instr=6, N_Glob=1)
 *   aprod 1:  b^itn += A   x^(itn-1)        PAPER.md:45   Sec. 2, Eq. (2)
 *   aprod 2:  x^itn += A^T b^itn            PAPER.md:49   Sec. 2, Eq. (3)
 *   the LSQR loop around them               PAPER.md:53-64 Sec. 2 (steps 3-4), Sec. 2.1,
 *                                           refs [29,30] (Paige & Saunders) PAPER.md:234-235
 * The call list (gsr_create / gsr_aprod1 / gsr_aprod2 / gsr_lsqr) is the one named by
 * BASELINE.json:north_star; the paper itself defines no API.
 *
 * DATA LAYOUT.  S stars, M rows, K attitude knots per axis, I instrumental
 * parameters, G in {0,1} global parameters.
 *   unknowns  x[n], n = 5S + 3K + I + G, blocks in the paper's order
 *             [ astrometric 5S | attitude 3K (axis-major, axis offset K) | instrumental I | global G ]
 *   values    M x 24 fp64, row-major: slots 0-4 astrometric, 5-16 attitude (axis a, knot j at
 *             slot 5+4a+j), 17-22 instrumental, 23 global (ignored when G = 0)
 *   indices   M x 8 int32, row-major: {star, att_start, instr_col[0..5]}
 *   column of slot k of row r:
 *             k < 5        : 5*star + k
 *             5 <= k < 17  : 5S + a*K + att_start + j          (a = (k-5)/4, j = (k-5)%4)
 *             17 <= k < 23 : 5S + 3K + instr_col[k-17]
 *             k == 23      : 5S + 3K + I
 *   Rows must be sorted by star (non-decreasing star id); this is validated.
 *
 * POINTERS.  Unless a parameter says "host", every array argument is a DEVICE pointer owned by
 * the caller.  `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 * All calls are for one GPU (the current device); there is no CPU fallback: without a CUDA
 * device every call that would compute returns GSR_ECUDA.
 *
 * ERRORS.  Every int-returning call returns GSR_OK (0) or a negative code; nothing is printed,
 * nothing throws, nothing exits.  gsr_strerror() names a code.
 *
 * THREADS AND STREAMS.  A gsr_system is NOT re-entrant: every call on one system shares its scratch
 * (interleaved attitude buffers, the replicated instrumental accumulators, which are assumed zero
 * between calls, the LSQR work vectors and the single set of device-resident scalars).  All calls on
 * one system must therefore be issued on ONE stream, or be ordered externally (events) so that no two
 * of them overlap; two gsr_aprod2 calls, or gsr_aprod2 / gsr_colnorms next to gsr_lsqr_iterate, running
 * concurrently on one system corrupt each other's results silently.  Different systems may run
 * concurrently on different streams from ONE host thread; the library is not thread-safe across
 * systems either (kernel attributes such as the dynamic shared-memory limit are process-global and are
 * set at launch time), so calls from several host threads must be serialised by the caller.
 *
 * DETERMINISM.  aprod2 uses fp64 reductions at L2 (red.global.add.f64) for the attitude block;
 * the order of those additions varies run to run, so results are reproducible to rounding
 * (normwise ~1e-15), not bit for bit.  aprod1 is bit-reproducible.  For debugging, option
 * aprod2_variant = 2 selects a slow aprod2 whose summation order is fixed (gsr_set_option below).
 */
#ifndef GSR_H
#define GSR_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GSR_OK 0
#define GSR_EINVAL (-1)  /* null pointer, bad size, n_glob not 0/1, misaligned pointer          */
#define GSR_ELAYOUT (-2) /* index records violate the layout (star order/range, att_start, col) */
#define GSR_ENOMEM (-3)  /* device or host allocation failed                                    */
#define GSR_ECUDA (-4)   /* a CUDA call failed (sticky; see gsr_last_cuda_error)                */
#define GSR_ESTATE (-5)  /* call out of order (e.g. iterate before init)                        */

typedef struct gsr_system gsr_system; /* opaque */

typedef struct {
  int64_t n_rows;  /* M : observation rows + constraint rows            */
  int64_t n_stars; /* S : astrometric block = 5*S columns                             */
  int64_t n_knots; /* K : attitude block = 3*K columns, axis offset K; K >= 4         */
  int64_t n_instr; /* I : instrumental block; I >= 1                                  */
  int32_t n_glob;  /* G : 0 or 1 (the paper's tests use 0)              */
  int32_t flags;   /* 0, or GSR_LAYOUT_TRUSTED: the caller guarantees that every index record
                      is in range and that rows are sorted by star; gsr_create then skips its
                      device-side validation pass (4 ms at 5e8 rows).  Other bits: GSR_EINVAL */
} gsr_layout;
#define GSR_LAYOUT_TRUSTED 1
#define GSR_LAYOUT_COEFF23 2 /* values records hold 23 doubles (184 B): the production record without the global
                                slot (N_Glob = 0; requires n_glob = 0).  Slots keep their numbers.
                                Served by the same tile kernels through a tensor view of 4-row groups (4 x 184 B = 736 B
                                is a whole number of 16-byte units); every call of this header
                                works for it, the fused LSQR pass and column-norm preconditioning included.             */

typedef struct {
  int32_t istop; /* Paige-Saunders stop code 0..7 (not an error)                      */
  int64_t itn;   /* iterations performed                                              */
  double r1norm, r2norm; /* ||b - A x|| estimate (equal: damp = 0)                    */
  double anorm, acond, arnorm, xnorm, bnorm;
} gsr_lsqr_result;

/* Scalars of the LSQR recurrences, as exported by gsr_lsqr_get_state (host struct). */
typedef struct {
  int64_t itn;
  int32_t istop;
  double alpha, beta, rhobar, phibar, bnorm, rnorm, arnorm, anorm, acond, ddnorm, xnorm, xxnorm,
      z, cs2, sn2;
} gsr_lsqr_scalars;

/* ---- system -------------------------------------------------------------------------------
 * gsr_create: bind a system to its device-resident matrix (PAPER.md:39 storage).
 *   layout  : host pointer, copied.
 *   values  : device, M*24 fp64, 32-byte aligned.  BORROWED, not copied (at 5e8 rows the matrix
 *   indices : device, M*8 int32, 32-byte aligned.   is 112 GB): the caller keeps both alive and
 *             unmodified until gsr_destroy.
 *   Validates every index record on the device (GSR_ELAYOUT on violation), builds the side
 *   structures (a few MB) and synchronises `stream` once.  M = 0 is allowed.
 * gsr_destroy: frees everything the library allocated (never values/indices). NULL is a no-op. */
int gsr_create(gsr_system **out, const gsr_layout *layout, const double *values,
               const int32_t *indices, void *stream);
void gsr_destroy(gsr_system *sys);
int gsr_dims(const gsr_system *sys, int64_t *n_rows, int64_t *n_unknowns); /* host out-pointers */
/* gsr_attach_constraints: the constraint equations as a section of their own ("a set of constraints
 *   equations", "~1 % of the entire system, is replicated among the MPI processes").
 *   n_rows records in the system's own format (values: n_rows x 24, or x 23 with GSR_LAYOUT_COEFF23; indices:
 *   n_rows x 8; device, 32-byte aligned, BORROWED until gsr_destroy or the next call), sorted by star among
 *   themselves, validated like gsr_create's.  The system then has n_rows(create) + n_rows(constraints) rows, the
 *   constraint rows LAST: every M-vector (y of the products, b of LSQR) carries them after the observation rows.
 *   Every product and every LSQR pass runs over both sections.  Voids a solve in progress (GSR_ESTATE until the next
 *   gsr_lsqr_init); n_rows = 0 detaches.  Synchronises `stream` once. */
int gsr_attach_constraints(gsr_system *sys, int64_t n_rows, const double *values, const int32_t *indices, void *stream);

/* ---- the two products (asynchronous on `stream`) --------------------------------------------
 * gsr_aprod1:  y[r] += sum_k a[r][k] * x[col(r,k)]      Eq. (2).  x: n, y: M.
 * gsr_aprod2:  x[col(r,k)] += a[r][k] * y[r]            Eq. (3).  y: M, x: n.
 * Both ACCUMULATE into their output (the paper's "+="); the input vector is not modified;
 * input and output must not overlap.  Repeated instrumental columns inside a row accumulate. */
int gsr_aprod1(gsr_system *sys, const double *x, double *y, void *stream);
int gsr_aprod2(gsr_system *sys, const double *y, double *x, void *stream);

/* ---- LSQR (Paige-Saunders, damp = 0) ---------------------------------
 * gsr_lsqr: solve min ||A x - b||_2 from x = 0.
 *   b (device, M) is not modified; x (device, n) is overwritten with the solution.
 *   itnlim >= 0; atol, btol >= 0; conlim >= 0 (0 = no condition-number test).
 *   res (HOST pointer) receives istop, itn and the norm estimates.
 *   Returns after the result is on the host (synchronises `stream`).
 *   istop: 0 x=0 is exact; 1 Ax=b to atol/btol; 2 least-squares solution to atol; 3 acond >=
 *   conlim; 4,5,6 the same three at machine precision; 7 itnlim reached.
 * Work vectors (u: M; v, w, x: n) are allocated on the first call and reused.
 *
 * The same solve, in steps (used by the benchmark to time exactly K iterations and by the
 * parity tests to compare one iteration at a time):
 *   gsr_lsqr_init    : x = 0; beta u = b; alpha v = A^T u; w = v     ("initial
 *                      conditions are set with aprod 2").  Asynchronous.
 *   gsr_lsqr_iterate : up to n_iters further iterations (each: aprod 1, aprod 2, the vector
 *                      updates, norms and stopping tests, all on the device); iterations after
 *                      a stop (istop != 0) are no-ops.  Asynchronous; the stopping rule is
 *                      evaluated on the device with the given tolerances.
 *   gsr_lsqr_result_get : copy the solution into x_out (device, n; may be NULL) and fill *res
 *                      (host).  Synchronises `stream`.
 *   gsr_lsqr_get_state : export the normalised Golub-Kahan vectors u (M), v, w, x (n) (device
 *                      pointers, any may be NULL) and the scalars (host).  Synchronises.      */
int gsr_lsqr(gsr_system *sys, const double *b, double *x, int64_t itnlim, double atol,
             double btol, double conlim, gsr_lsqr_result *res, void *stream);
int gsr_lsqr_init(gsr_system *sys, const double *b, void *stream);
int gsr_lsqr_iterate(gsr_system *sys, int64_t n_iters, int64_t itnlim, double atol, double btol,
                     double conlim, void *stream);
int gsr_lsqr_result_get(gsr_system *sys, double *x_out, gsr_lsqr_result *res, void *stream);
int gsr_lsqr_get_state(gsr_system *sys, double *u, double *v, double *w, double *x,
                       gsr_lsqr_scalars *scalars, void *stream);

/* ---- whole solve from HOST buffers (end-to-end path) ----------------------------------------
 * Allocates device memory, copies values / indices / b host->device, runs gsr_create + gsr_lsqr,
 * copies x device->host, frees everything.  All four arrays are HOST pointers (pinned or
 * pageable; values_host holds 24, or with GSR_LAYOUT_COEFF23 23, doubles per row); x_host (n) is overwritten.
 * Blocking. */
int gsr_lsqr_host(const gsr_layout *layout, const double *values_host, const int32_t *indices_host,
                  const double *b_host, double *x_host, int64_t itnlim, double atol, double btol,
                  double conlim, gsr_lsqr_result *res);

/* ---- the steps either side of the LSQR loop in the paper's solver -------------
 * PAPER.md:56 "the system is preconditioned", "the variances of the solution are computed /
 * the solution and its errors are de-preconditioned".  The paper gives no formulas; the reading taken
 * (R7) is diagonal column scaling: D = diag(||A e_j||_2), 1 for a column no row touches; LSQR runs
 * on (A D^-1) z = b and returns x = D^-1 z.  The variances are Paige-Saunders' estimate of diag((A^T A)^-1),
 * var += (w / rho)^2 at every iteration, returned in the units of x (var_x = D^-2 var_z).
 *
 * gsr_colnorms : out[j] = ||A e_j||_2 for every unknown (device, n, the ABI's column order), one pass over A.
 * gsr_lsqr_ex  : gsr_lsqr with `var` (device, n, overwritten; NULL = not wanted) and `flags`
 *                (GSR_PRECOND_COLNORM or 0).  The norms in `res` are those of the system LSQR iterated on
 *                (the scaled one when preconditioned), as in the paper's loop.  Errors as gsr_lsqr;
 *                GSR_ESTATE if the two-pass schedule (option fused=0) is combined with preconditioning. */
/* gsr_set_cov_pairs : covariances of chosen pairs of unknowns, Eq. (4): Cov[p] += factor^itn *
 *                x^itn[j1[p]] * x^itn[j2[p]] at every iteration.  Reading (R21): the off-diagonal companion
 *                of var, x^itn = the direction w of the iteration, factor = 1/rho^2, so a pair (j, j) gives var[j].
 *                j1, j2 (device, n_pairs x int64, columns in the ABI's order) and cov (device, n_pairs doubles) are
 *                BORROWED until the next gsr_set_cov_pairs or gsr_destroy; every later gsr_lsqr_ex zeroes cov,
 *                accumulates into it on the device (the paper's file pipeline between two programs is not needed when
 *                x lives in one GPU) and returns it in the units of x.  n_pairs = 0 unregisters.
 *                GSR_EINVAL if an index is outside [0, n). */
#define GSR_PRECOND_COLNORM 1
int gsr_set_cov_pairs(gsr_system *sys, const int64_t *j1, const int64_t *j2, int64_t n_pairs, double *cov, void *stream);
int gsr_colnorms(gsr_system *sys, double *out, void *stream);
int gsr_lsqr_ex(gsr_system *sys, const double *b, double *x, double *var, int32_t flags, int64_t itnlim,
                double atol, double btol, double conlim, gsr_lsqr_result *res, void *stream);

/* ---- row-sharded LSQR over several GPUs, in phases --------------------------------
 * PAPER.md:72 "the computation related to a subset of the total number of observations (rows in matrix A) is
 * assigned to a different MPI process ... the astrometric part ... is distributed over the MPI processes, whereas the
 * attitude, instrumental, and global parts are replicated"; "two reduce operations per LSQR iteration,
 * performed at the end of each aprod 1 and aprod 2 call".
 *
 * One process per GPU.  Every rank creates its own gsr_system over a contiguous range of rows cut at a star boundary,
 * with the GLOBAL n_stars / n_knots / n_instr / n_glob (star ids stay global, so the borrowed index records need no
 * rewriting; a rank's n-vectors have full length and their astrometric entries outside its own stars stay exactly 0).
 * The constraint section, if any, is attached on ONE rank.  The library does all the arithmetic of a phase on the
 * rank's rows; what the ranks must add up between two phases is the first *xcount doubles of the exchange buffer
 * `xbuf` (device, gsr_shard_exchange_len() doubles = 3K + I + G + 2, caller-owned, borrowed until the solve ends):
 * the caller sums them over the ranks IN PLACE (one NCCL allreduce(sum) on `stream`) before the next phase call.
 * Because aprod 1 and aprod 2 of an iteration share one pass over A here, an iteration needs ONE vector reduce (the
 * replicated tail of A^T u, 24.5 MB at C4, with sum u^2 and sum w^2 riding along) and one scalar reduce (sum v^2)
 * instead of the paper's two vector reduces.  Every rank then evaluates the same scalars and the same stopping rule.
 *
 *   gsr_shard_begin : start a solve of min ||A x - b|| with b = this rank's rows of the right-hand side.
 *                     counts_shared = 1 on exactly ONE rank (the replicated tail of v and w enters the norms once),
 *                     0 on the others.  Runs phase 0 (u = b, partial sum b^2); *xcount = 1.
 *   gsr_shard_phase : run the next phase; *xcount = doubles of xbuf to sum over the ranks before the next call
 *                     (0 = nothing to exchange); *status = GSR_SHARD_MORE, GSR_SHARD_INIT_DONE (x = 0, v, w set up) or
 *                     GSR_SHARD_ITER_DONE (one more LSQR iteration complete).  Phases: init b, c, d, then a, b, c of
 *                     every iteration.  Asynchronous; iterations after a stop are no-ops, as in gsr_lsqr_iterate.
 *   gsr_shard_poll  : *stopped = 1 once a stopping rule has fired (same value on every rank); *res (host, may be
 *                     NULL) as gsr_lsqr.  Synchronises `stream`.  The solution is read with gsr_lsqr_result_get: the
 *                     astrometric block holds this rank's stars (0 elsewhere: the sum over ranks is the whole block),
 *                     the other blocks are identical on every rank.
 * Plain LSQR on the one-pass schedule only (GSR_ESTATE with option fused=0); gsr_lsqr_iterate
 * returns GSR_ESTATE while a sharded solve is in progress; gsr_lsqr_init / gsr_lsqr end it.                          */
#define GSR_SHARD_MORE 0
#define GSR_SHARD_INIT_DONE 1
#define GSR_SHARD_ITER_DONE 2
int gsr_shard_exchange_len(const gsr_system *sys, int64_t *n_doubles);
int gsr_shard_begin(gsr_system *sys, const double *b, double *xbuf, int32_t counts_shared, int64_t itnlim, double atol,
                    double btol, double conlim, int64_t *xcount, void *stream);
int gsr_shard_phase(gsr_system *sys, int64_t *xcount, int32_t *status, void *stream);
int gsr_shard_poll(gsr_system *sys, int32_t *stopped, gsr_lsqr_result *res, void *stream);

/* ---- diagnostics ----------------------------------------------------------------------------
 * gsr_launch_count : kernels launched by this system object so far (host out-pointer).
 * gsr_profile      : enable (1) / disable (0) CUDA-event timing of the matrix-pass kernels issued by
 *                    gsr_lsqr_iterate and gsr_aprod1/2, on their own stream.
 * gsr_profile_get  : after a synchronise, mean duration in ms and launch count since the last
 *                    call, per kernel class: which = 1 aprod1, 2 aprod2, 3 the fused LSQR pass
 *                    (aprod 1 + aprod 2 of one iteration in one sweep over A) (host out-pointers).
 * gsr_set_option   : tuning knobs (measured in profiles/r01_summary.md section 3);
 *                    unknown names -> GSR_EINVAL.  Names (value 0 = default of the planner unless stated):
 *                      warps, stages     warps per CTA (<= 12; planner default 12, down to 8 when that lets the instrumental
 *                                        tables fit shared memory) and TMA ring depth per warp (default 2) of the tile kernels
 *                      ctas_per_sm       CTAs per SM (default 1)
 *                      acc_smem          1 (default) privatise the instrumental accumulators in shared memory
 *                                        when they fit, 0 always reduce into the L2-resident copies
 *                      die_local         1 (default) L2-resident instrumental accumulators: every CTA reduces into a copy whose
 *                                        4 KB chunks are homed on the L2 of its own die (probed at gsr_create), 0 control
 *                      acc_part, acc_part_fused   when the accumulators live in L2: how many leading instrumental columns are
 *                                        accumulated in left-over shared memory instead (-1 all that fit, 0 none = default of both:
 *                                        the committed form has not been timed on hardware)
 *                      tab_private       1: the table of die-local chunks is replicated once per shared-memory bank, 0 (default) one copy
 *                      gather_smem       1 (default) stage the instrumental slice of x in shared memory when it fits
 *                      instr_copies      1 (default) use the replicated accumulators, 0 reduce straight into x
 *                      fused             1 (default) one pass over A per LSQR iteration, 0 aprod 1 then aprod 2
 *                      aprod1_variant, aprod2_variant   1 (default) TMA tiles, 0 one thread per row (cross-check);
 *                                        aprod2_variant = 2: DETERMINISTIC debug variant -- every sum of gsr_aprod2 (and of the
 *                                        aprod 2 inside gsr_lsqr_init and the two-pass schedule) has one fixed order that
 *                                        depends on the sizes only, so results are bit-reproducible run to run and GPU to GPU;
 *                                        slow by design (at most 1024 threads add up the shared columns), either record format
 *                      det_chunks        variant 2: row chunks, each with a private copy of the shared columns (0 = default: as
 *                                        many as fit 256 MB, at most 1024); 1 = row by row, slot by slot from x's initial value,
 *                                        i.e. Eq. (3) written out as a plain loop: bit-identical to such a serial implementation
 *                      graph             1 (default) small, launch-bound systems (matrix <= 256 MB): the launches of a batch
 *                                        of LSQR iterations are captured once into a CUDA graph and replayed, 0 never
 *                      check_every       LSQR iterations between host polls of the stop flag (default 16)      */
int gsr_launch_count(const gsr_system *sys, int64_t *n_launches);
int gsr_profile(gsr_system *sys, int enable);
int gsr_profile_get(gsr_system *sys, int which, double *mean_ms, int64_t *count);
int gsr_set_option(gsr_system *sys, const char *name, int64_t value);
/* gsr_instr_acc_info : what gsr_create found when it probed the L2 home die of the instrumental accumulator
 *                      chunks.  info (host, 5 x int32) = {two dies seen (0/1), copies per
 *                      die, 4 KB chunks per copy, SMs found on die 0, SMs found on die 1}.                        */
int gsr_instr_acc_info(const gsr_system *sys, int32_t *info);
const char *gsr_strerror(int code);
const char *gsr_last_cuda_error(void); /* text of the last CUDA failure in this thread, or "" */
const char *gsr_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GSR_H */
