/*
 * CPU ORACLE for the AVU-GSR hot path -- TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, link or call this.  It shares no code with the CUDA library
 * (paper_2503_22863_b200/csrc, include/gsr.h) and never reads its outputs.
 *
 * What it computes, and where the paper defines it:
 *   orc_aprod1 : y += A x            PAPER.md:45  (Sec. 2, Eq. 2, "aprod 1")
 *   orc_aprod2 : x += A^T y          PAPER.md:49  (Sec. 2, Eq. 3, "aprod 2")
 *   orc_lsqr   : Paige-Saunders LSQR PAPER.md:35, 41, 53-64 (Sec. 2 solver outline),
 *                refs [29,30] at PAPER.md:234-235; damp = 0, no preconditioning
 *                (reading R7).
 *   orc_colnorm2, orc_scale_columns, and in oracle/__init__.py lsqr_var / lsqr_precond / lsqr_cov (written over
 *                orc_lsqr_init / orc_lsqr_step): the steps either side of the loop
 *                (preconditioning, variances) and PAPER.md:86-92 Eq. 4 (covariances).  The paper gives no
 *                formulas for these: the readings R7 / R21 of DESIGN.md are what is implemented -- PARITY UNPINNED
 *                BY THE PAPER for the choice of reading; the functions themselves are pinned (dense matrix,
 *                scipy's var, (A^T A)^-1, dense least squares).
 * The matrix is the paper's compressed storage: 24 fp64 coefficients per
 * row = 5 astrometric + 12 attitude + 6 instrumental + 1 global; the column of every
 * slot is derived from the 8-int32 index record {star, att_start, instr[6]} as fixed
 * by BASELINE.json (readings R1, R2).
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): dense brute force, adjoint
 * identity, += semantics, numpy.linalg.lstsq, scipy.sparse.linalg.lsqr, residual
 * identities, closed forms.  The paper prints no worked numerical example for this
 * path, so there is no paper-value pin.
 *
 * Plain fp64, IEEE round-to-nearest, slot order, no FMA contraction (-ffp-contract=off).
 */
#ifndef GSR_ORACLE_H
#define GSR_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int64_t n_stars;  /* S : astrometric block = 5*S columns            */
  int64_t n_knots;  /* K : attitude block = 3*K columns, axis offset K */
  int64_t n_instr;  /* I                                               */
  int32_t n_glob;   /* 0 or 1 (PAPER.md:141 uses 0, BASELINE configs 1) */
  int32_t coeffs_per_row; /* record stride in doubles: 0 or 24 = the 24-slot record; 23 = the production record without
                             the global slot (requires n_glob = 0)                      */
} orc_layout;

typedef struct {
  int32_t istop;
  int64_t itn;
  double r1norm, r2norm, anorm, acond, arnorm, xnorm, bnorm;
} orc_lsqr_result;

int64_t orc_n_unknowns(const orc_layout *L);
/* column of slot k (0..23) of a row with index record rec[8]; -1 if the slot is unused */
int64_t orc_col(const orc_layout *L, const int32_t *rec, int k);

/* a: nrows*24 (or nrows*23, see coeffs_per_row) row-major, idx: nrows*8, chunk-local (row 0 of the chunk first). */
void orc_aprod1(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
                const double *x, double *y);
void orc_aprod2(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
                const double *y, double *x);
/* Neumaier-compensated aprod2: x holds the running sums, comp (same length, zeroed by
 * the caller before the first chunk) the compensation; final value = x[j] + comp[j]. */
void orc_aprod2_comp(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
                     const double *y, double *x, double *comp);
/* s[r] = |y_in[r]| + sum_k |a[r][k] * x[col(r,k)]| : denominator of the aprod1 forward bound */
void orc_aprod1_abs(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
                    const double *x, const double *y_in, double *s);

/* Column scaling (R7): squared column 2-norms (accumulated into nrm2sq, n),
 * and a_out = A diag(s) with the same index records. */
void orc_colnorm2(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx, double *nrm2sq);
void orc_scale_columns(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx, const double *s,
                       double *a_out);

/* OpenMP variants (timed CPU baseline; deterministic for a fixed thread count). */
void orc_aprod1_omp(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
                    const double *x, double *y, int threads);
void orc_aprod2_omp(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
                    const double *y, double *x, int threads);

/* Explicit LSQR state, so that one iteration can be replayed from any state (used by the
 * GPU parity tests: two correct LSQR runs drift apart chaotically once Lanczos
 * orthogonality is lost, reading R16, so each iteration is also checked on its
 * own from a shared state).  u (m), v, w, x (n) are caller-owned. */
typedef struct {
  int64_t itn;
  int32_t istop;
  double alpha, beta, rhobar, phibar, bnorm, rnorm, arnorm, anorm, acond, ddnorm, xnorm,
      xxnorm, z, cs2, sn2;
  double *u, *v, *w, *x;
} orc_lsqr_state;

void orc_lsqr_init(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
                   const double *b, int threads, orc_lsqr_state *s);
void orc_lsqr_step(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
                   int64_t itnlim, double atol, double btol, double conlim, int threads,
                   orc_lsqr_state *s);

/* LSQR, damp = 0 (= orc_lsqr_init + orc_lsqr_step until istop != 0).  b is not modified; x (n) is overwritten.  threads <= 1 -> serial
 * routines above (the parity reference); > 1 -> the OpenMP ones.
 * rnorm_hist / arnorm_hist: optional (may be NULL) arrays of length itnlim+1 receiving the
 * estimates after each iteration (entry 0 = initial). Returns 0, or -1 on allocation failure. */
int orc_lsqr(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
             const double *b, double *x, int64_t itnlim, double atol, double btol,
             double conlim, int threads, orc_lsqr_result *res, double *rnorm_hist,
             double *arnorm_hist);

int orc_max_threads(void);

#ifdef __cplusplus
}
#endif
#endif
