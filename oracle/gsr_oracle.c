/* CPU oracle -- see gsr_oracle.h for scope, citations and the "test infrastructure only" rule.
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC gsr_oracle.c -o libgsr_oracle.so -lm
 */
#include "gsr_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NSLOT 24  /* N_Astro 5 + N_Att 12 + N_Instr 6 + N_Glob 1 */
/* Coefficients stored per row = record stride in doubles: 24, or 23 for the production record without the
 * global slot (N_Glob = 0).  Slots keep their numbers either way. */
static int nslot_of(const orc_layout *L) { return L->coeffs_per_row == 23 ? 23 : NSLOT; }
#define NIDX 8    /* {star, att_start, instr[6]}                              */

int orc_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

int64_t orc_n_unknowns(const orc_layout *L) {
  return 5 * L->n_stars + 3 * L->n_knots + L->n_instr + L->n_glob;
}

/* Slot -> column map.  x = [astro 5S | attitude 3K | instrumental I | global G]
 * (order of PAPER.md:39; reading R1). */
int64_t orc_col(const orc_layout *L, const int32_t *rec, int k) {
  const int64_t oA = 5 * L->n_stars;
  const int64_t oI = oA + 3 * L->n_knots;
  const int64_t oG = oI + L->n_instr;
  if (k < 5) return 5 * (int64_t)rec[0] + k;                 /* astrometric            */
  if (k < 17) {                                              /* attitude, axis-major    */
    int ax = (k - 5) / 4, j = (k - 5) % 4;
    return oA + ax * L->n_knots + (int64_t)rec[1] + j;
  }
  if (k < 23) return oI + (int64_t)rec[2 + (k - 17)];        /* instrumental            */
  return L->n_glob ? oG : -1;                                /* global (absent if G=0)  */
}

/* Eq. 2: y[r] += sum_k a[r][k] * x[col(r,k)], rows in order, slots in order. */
void orc_aprod1(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
                const double *x, double *y) {
  const int ns = nslot_of(L);
  for (int64_t r = 0; r < nrows; r++) {
    const double *ar = a + r * ns;
    const int32_t *rec = idx + r * NIDX;
    double s = 0.0;
    for (int k = 0; k < ns; k++) {
      int64_t c = orc_col(L, rec, k);
      if (c >= 0) s += ar[k] * x[c];
    }
    y[r] += s;
  }
}

/* Eq. 3: x[col(r,k)] += a[r][k] * y[r], rows in order, slots in order.
 * Repeated columns inside one row simply accumulate. */
void orc_aprod2(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
                const double *y, double *x) {
  const int ns = nslot_of(L);
  for (int64_t r = 0; r < nrows; r++) {
    const double *ar = a + r * ns;
    const int32_t *rec = idx + r * NIDX;
    const double yr = y[r];
    for (int k = 0; k < ns; k++) {
      int64_t c = orc_col(L, rec, k);
      if (c >= 0) x[c] += ar[k] * yr;
    }
  }
}

/* Same sum as orc_aprod2 with Neumaier's compensated accumulation per x entry. */
void orc_aprod2_comp(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
                     const double *y, double *x, double *comp) {
  const int ns = nslot_of(L);
  for (int64_t r = 0; r < nrows; r++) {
    const double *ar = a + r * ns;
    const int32_t *rec = idx + r * NIDX;
    const double yr = y[r];
    for (int k = 0; k < ns; k++) {
      int64_t c = orc_col(L, rec, k);
      if (c < 0) continue;
      double t = ar[k] * yr;
      double s = x[c] + t;
      if (fabs(x[c]) >= fabs(t)) comp[c] += (x[c] - s) + t;
      else                       comp[c] += (t - s) + x[c];
      x[c] = s;
    }
  }
}

void orc_aprod1_abs(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
                    const double *x, const double *y_in, double *s_out) {
  const int ns = nslot_of(L);
  for (int64_t r = 0; r < nrows; r++) {
    const double *ar = a + r * ns;
    const int32_t *rec = idx + r * NIDX;
    double s = y_in ? fabs(y_in[r]) : 0.0;
    for (int k = 0; k < ns; k++) {
      int64_t c = orc_col(L, rec, k);
      if (c >= 0) s += fabs(ar[k] * x[c]);
    }
    s_out[r] = s;
  }
}

/* ------------------------------------------------------------------ OpenMP variants */
/* the steps either side of the LSQR loop in the paper's solver (PAPER.md:56,
 * 61, 63: "preconditioned" system, variances of the solution).  The paper gives no formulas; the
 * reading taken (R7) is diagonal column scaling by the column 2-norms.
 * nrm2sq[j] += sum_r (A[r][j])^2, where A[r][j] = sum of the a[r][k] with col(r,k) = j : the squared 2-norm of
 * column j of A as an operator.  A column can repeat inside a row (instrumental slots): the
 * coefficients of equal columns are summed first, in slot order, and the sum is squared once. */
void orc_colnorm2(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx, double *nrm2sq) {
  const int ns = nslot_of(L);
  for (int64_t r = 0; r < nrows; r++)
    for (int k = 0; k < ns; k++) {
      int64_t c = orc_col(L, idx + r * NIDX, k);
      if (c < 0) continue;
      int seen = 0;                         /* an earlier slot of this row already carried column c */
      for (int k0 = 0; k0 < k; k0++)
        if (orc_col(L, idx + r * NIDX, k0) == c) seen = 1;
      if (seen) continue;
      double arj = a[r * ns + k];        /* A[r][c]: this slot and every later slot on the same column */
      for (int k1 = k + 1; k1 < ns; k1++)
        if (orc_col(L, idx + r * NIDX, k1) == c) arj += a[r * ns + k1];
      nrm2sq[c] += arj * arj;
    }
}
/* a_out[r][k] = a[r][k] * s[col(r,k)] : the matrix A diag(s), same index records. */
void orc_scale_columns(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx, const double *s,
                       double *a_out) {
  const int ns = nslot_of(L);
  for (int64_t r = 0; r < nrows; r++)
    for (int k = 0; k < ns; k++) {
      int64_t c = orc_col(L, idx + r * NIDX, k);
      a_out[r * ns + k] = c >= 0 ? a[r * ns + k] * s[c] : a[r * ns + k];
    }
}

static int clamp_threads(int threads) {
  int mx = orc_max_threads();
  if (threads < 1) threads = 1;
  return threads > mx ? mx : threads;
}

void orc_aprod1_omp(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
                    const double *x, double *y, int threads) {
  threads = clamp_threads(threads);
#pragma omp parallel num_threads(threads)
  {
#ifdef _OPENMP
    int t = omp_get_thread_num(), T = omp_get_num_threads();
#else
    int t = 0, T = 1;
#endif
    int64_t r0 = nrows * t / T, r1 = nrows * (t + 1) / T;
    orc_aprod1(L, r1 - r0, a + r0 * nslot_of(L), idx + r0 * NIDX, x, y + r0);
  }
}

/* first row >= r whose star differs from row r-1 (so a star is never split) */
static int64_t star_aligned(const int32_t *idx, int64_t nrows, int64_t r) {
  if (r <= 0) return 0;
  while (r < nrows && idx[r * NIDX] == idx[(r - 1) * NIDX]) r++;
  return r;
}

/* Row partition aligned to star boundaries: the astrometric columns of different threads
 * are disjoint and are written in place; attitude / instrumental / global go to per-thread
 * private accumulators that are added to x in thread order (deterministic for fixed T). */
void orc_aprod2_omp(const orc_layout *L, int64_t nrows, const double *a, const int32_t *idx,
                    const double *y, double *x, int threads) {
  const int ns = nslot_of(L);
  threads = clamp_threads(threads);
  const int64_t oA = 5 * L->n_stars;
  const int64_t nshared = 3 * L->n_knots + L->n_instr + L->n_glob;
  double *priv = (double *)calloc((size_t)threads * (size_t)(nshared > 0 ? nshared : 1), sizeof(double));
  if (!priv) { orc_aprod2(L, nrows, a, idx, y, x); return; }
#pragma omp parallel num_threads(threads)
  {
#ifdef _OPENMP
    int t = omp_get_thread_num(), T = omp_get_num_threads();
#else
    int t = 0, T = 1;
#endif
    int64_t r0 = star_aligned(idx, nrows, nrows * t / T);
    int64_t r1 = (t == T - 1) ? nrows : star_aligned(idx, nrows, nrows * (t + 1) / T);
    double *p = priv + (size_t)t * nshared;
    for (int64_t r = r0; r < r1; r++) {
      const double *ar = a + r * ns;
      const int32_t *rec = idx + r * NIDX;
      const double yr = y[r];
      for (int k = 0; k < ns; k++) {
        int64_t c = orc_col(L, rec, k);
        if (c < 0) continue;
        if (c < oA) x[c] += ar[k] * yr;
        else        p[c - oA] += ar[k] * yr;
      }
    }
#pragma omp barrier
    /* each thread reduces a slice of the shared columns over threads, in thread order */
    int64_t c0 = nshared * t / T, c1 = nshared * (t + 1) / T;
    for (int tt = 0; tt < T; tt++) {
      const double *q = priv + (size_t)tt * nshared;
      for (int64_t c = c0; c < c1; c++) x[oA + c] += q[c];
    }
  }
  free(priv);
}

/* ------------------------------------------------------------------ LSQR helpers */
static double nrm2(const double *v, int64_t n, int threads) {
  if (threads <= 1) {
    double s = 0.0;
    for (int64_t i = 0; i < n; i++) s += v[i] * v[i];
    return sqrt(s);
  }
  double part[256];
  int T = threads > 256 ? 256 : threads;
  for (int t = 0; t < T; t++) part[t] = 0.0;
#pragma omp parallel num_threads(T)
  {
#ifdef _OPENMP
    int t = omp_get_thread_num(), TT = omp_get_num_threads();
#else
    int t = 0, TT = 1;
#endif
    double s = 0.0;
    for (int64_t i = n * t / TT; i < n * (t + 1) / TT; i++) s += v[i] * v[i];
    part[t] = s;
  }
  double s = 0.0;
  for (int t = 0; t < T; t++) s += part[t];
  return sqrt(s);
}

static void scal(double *v, int64_t n, double c, int threads) {
#pragma omp parallel for num_threads(threads) schedule(static) if (threads > 1)
  for (int64_t i = 0; i < n; i++) v[i] *= c;
}

static void do_aprod1(const orc_layout *L, int64_t m, const double *a, const int32_t *idx,
                      const double *x, double *y, int threads) {
  if (threads <= 1) orc_aprod1(L, m, a, idx, x, y);
  else orc_aprod1_omp(L, m, a, idx, x, y, threads);
}
static void do_aprod2(const orc_layout *L, int64_t m, const double *a, const int32_t *idx,
                      const double *y, double *x, int threads) {
  if (threads <= 1) orc_aprod2(L, m, a, idx, y, x);
  else orc_aprod2_omp(L, m, a, idx, y, x, threads);
}

/* Paige & Saunders, "LSQR: an algorithm for sparse linear equations and sparse least
 * squares" (paper refs [29,30]), Algorithm LSQR with damp = 0, in the
 * order and notation of SURVEY.md section 8(c.3) / DESIGN.md section 4.  The solver outline is
 * "initial conditions are set with aprod 2" (step 3), then per iteration
 * aprod 1 (4a) and aprod 2 (4b).
 *
 * init:  x = 0; beta u = b; alpha v = A^T u; w = v  */
void orc_lsqr_init(const orc_layout *L, int64_t m, const double *a, const int32_t *idx,
                   const double *b, int threads, orc_lsqr_state *s) {
  threads = clamp_threads(threads);
  const int64_t n = orc_n_unknowns(L);
  s->itn = 0; s->istop = 0;
  s->anorm = s->acond = s->ddnorm = s->xnorm = s->xxnorm = s->z = 0.0;
  s->cs2 = -1.0; s->sn2 = 0.0;
  s->alpha = 0.0;
  for (int64_t i = 0; i < n; i++) { s->x[i] = 0.0; s->v[i] = 0.0; }
  memcpy(s->u, b, sizeof(double) * (size_t)m);
  s->beta = nrm2(s->u, m, threads);
  if (s->beta > 0.0) {
    scal(s->u, m, 1.0 / s->beta, threads);
    do_aprod2(L, m, a, idx, s->u, s->v, threads);
    s->alpha = nrm2(s->v, n, threads);
  }
  if (s->alpha > 0.0) scal(s->v, n, 1.0 / s->alpha, threads);
  memcpy(s->w, s->v, sizeof(double) * (size_t)n);
  s->arnorm = s->alpha * s->beta;
  s->rhobar = s->alpha; s->phibar = s->beta; s->bnorm = s->beta; s->rnorm = s->beta;
}

/* One LSQR iteration from the state in *s (steps 1-8 of DESIGN.md section 4); sets s->istop. */
void orc_lsqr_step(const orc_layout *L, int64_t m, const double *a, const int32_t *idx,
                   int64_t itnlim, double atol, double btol, double conlim, int threads,
                   orc_lsqr_state *s) {
  threads = clamp_threads(threads);
  const int64_t n = orc_n_unknowns(L);
  const double ctol = conlim > 0.0 ? 1.0 / conlim : 0.0;
  double *u = s->u, *v = s->v, *w = s->w, *x = s->x;
  double alpha = s->alpha, beta;
  s->itn++;
  /* 1: beta u = A v - alpha u */
  scal(u, m, -alpha, threads);
  do_aprod1(L, m, a, idx, v, u, threads);
  beta = nrm2(u, m, threads);
  /* 2: alpha v = A^T u - beta v */
  if (beta > 0.0) {
    scal(u, m, 1.0 / beta, threads);
    s->anorm = sqrt(s->anorm * s->anorm + alpha * alpha + beta * beta);
    scal(v, n, -beta, threads);
    do_aprod2(L, m, a, idx, u, v, threads);
    alpha = nrm2(v, n, threads);
    if (alpha > 0.0) scal(v, n, 1.0 / alpha, threads);
  }
  /* 3: plane rotation eliminating beta */
  double rho = sqrt(s->rhobar * s->rhobar + beta * beta);
  double cs = s->rhobar / rho, sn = beta / rho;
  double theta = sn * alpha;
  s->rhobar = -cs * alpha;
  double phi = cs * s->phibar;
  s->phibar = sn * s->phibar;
  double tau = sn * phi;
  /* 4: x, w update (x uses the old w) and ||w/rho||^2 */
  double t1 = phi / rho, t2 = -theta / rho, rinv = 1.0 / rho, dsum = 0.0;
  for (int64_t i = 0; i < n; i++) {
    double wi = w[i];
    double dk = rinv * wi;
    dsum += dk * dk;
    x[i] = x[i] + t1 * wi;
    w[i] = v[i] + t2 * wi;
  }
  s->ddnorm += dsum;
  /* 5: estimate of ||x|| */
  double delta = s->sn2 * rho, gambar = -s->cs2 * rho, rhs = phi - delta * s->z;
  double zbar = rhs / gambar;
  s->xnorm = sqrt(s->xxnorm + zbar * zbar);
  double gamma = sqrt(gambar * gambar + theta * theta);
  s->cs2 = gambar / gamma; s->sn2 = theta / gamma;
  s->z = rhs / gamma;
  s->xxnorm += s->z * s->z;
  /* 6: norm estimates */
  s->acond = s->anorm * sqrt(s->ddnorm);
  s->rnorm = fabs(s->phibar);
  s->arnorm = alpha * fabs(tau);
  s->alpha = alpha; s->beta = beta;
  /* 7: stopping quantities */
  double test1 = s->rnorm / s->bnorm;
  double den2 = s->anorm * s->rnorm;
  double test2 = den2 > 0.0 ? s->arnorm / den2 : 0.0;
  double test3 = 1.0 / s->acond;
  double t1p = test1 / (1.0 + s->anorm * s->xnorm / s->bnorm);
  double rtol = btol + atol * s->anorm * s->xnorm / s->bnorm;
  /* 8: later tests override earlier ones */
  int istop = 0;
  if (s->itn >= itnlim) istop = 7;
  if (1.0 + test3 <= 1.0) istop = 6;
  if (1.0 + test2 <= 1.0) istop = 5;
  if (1.0 + t1p <= 1.0) istop = 4;
  if (test3 <= ctol) istop = 3;
  if (test2 <= atol) istop = 2;
  if (test1 <= rtol) istop = 1;
  s->istop = istop;
}

int orc_lsqr(const orc_layout *L, int64_t m, const double *a, const int32_t *idx,
             const double *b, double *x, int64_t itnlim, double atol, double btol,
             double conlim, int threads, orc_lsqr_result *res, double *rnorm_hist,
             double *arnorm_hist) {
  const int64_t n = orc_n_unknowns(L);
  orc_lsqr_state s;
  s.u = (double *)malloc(sizeof(double) * (size_t)(m > 0 ? m : 1));
  s.v = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
  s.w = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
  s.x = x;
  if (!s.u || !s.v || !s.w) { free(s.u); free(s.v); free(s.w); return -1; }
  orc_lsqr_init(L, m, a, idx, b, threads, &s);
  if (rnorm_hist) rnorm_hist[0] = s.rnorm;
  if (arnorm_hist) arnorm_hist[0] = s.arnorm;
  if (s.arnorm == 0.0) {
    s.istop = 0;                                   /* x = 0 is the exact solution */
  } else if (itnlim <= 0) {
    s.istop = 7;
  } else {
    while (s.istop == 0) {
      orc_lsqr_step(L, m, a, idx, itnlim, atol, btol, conlim, threads, &s);
      if (rnorm_hist) rnorm_hist[s.itn] = s.rnorm;
      if (arnorm_hist) arnorm_hist[s.itn] = s.arnorm;
    }
  }
  res->istop = s.istop; res->itn = s.itn;
  res->r1norm = s.rnorm; res->r2norm = s.rnorm;    /* damp = 0 */
  res->anorm = s.anorm; res->acond = s.acond; res->arnorm = s.arnorm;
  res->xnorm = s.xnorm; res->bnorm = s.bnorm;
  free(s.u); free(s.v); free(s.w);
  return 0;
}
