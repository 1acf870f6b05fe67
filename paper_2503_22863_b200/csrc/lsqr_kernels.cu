// LSQR vector updates, norms, scalar recurrences and stopping tests, all on the device
// (Paige-Saunders LSQR, paper refs [29,30]; solver outline PAPER.md:53-64;
// SURVEY.md section 8a rows a6-a10).
//
// u is kept UN-normalised (u_hat = beta * u): the scale 1/beta is applied by the consumer
// (aprod2 reads yscale = 1/beta), so no M-length scale pass exists.  v, w, x are n-length
// (n << M) and are kept in the textbook (normalised) form.
#include "gsr_internal.cuh"

namespace gsr {

static inline unsigned grid_for(int64_t n, int threads, int per_thread) {
  int64_t b = (n + (int64_t)threads * per_thread - 1) / ((int64_t)threads * per_thread);
  if (b < 1) b = 1;
  if (b > 148 * 8) b = 148 * 8;
  return (unsigned)b;
}

// u_hat = b ; usq = sum b^2                                                       (init)
__global__ void __launch_bounds__(256) k_init_u(const double* __restrict__ b, double* __restrict__ u,
                                                int64_t M, DevScalars* sc) {
  double sq = 0.0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < M;
       i += (int64_t)gridDim.x * blockDim.x) {
    const double t = b[i];
    u[i] = t;
    sq = fma(t, t, sq);
  }
  sq = block_sum(sq);
  if (threadIdx.x == 0) atomicAdd(&sc->usq, sq);
}

// beta = ||b||                                                                      (init)
__global__ void k_init_s1(DevScalars* sc) {
  const double beta = sqrt(sc->usq);
  sc->beta = beta;
  sc->bnorm = beta;
  sc->s_y = beta > 0.0 ? 1.0 / beta : 0.0;
  sc->usq = 0.0;
  sc->vsq = 0.0;
  sc->wsq = 0.0;
  sc->done = 0;
  sc->istop = 0;
  sc->itn = 0;
}

// vsq = ||v||^2; with a preconditioner, v <- D^-1 v first (v = A^T u becomes (A D^-1)^T u)
// n_sq (here and in the three n-length kernels below): only elements i < n_sq enter the sum of squares.  n_sq = n
// except in a row-sharded solve (gsr_shard_*), where the replicated tail of the vector is counted by one rank only.
__global__ void __launch_bounds__(256) k_sumsq_v(double* __restrict__ v, int64_t n, DevScalars* sc,
                                                 const double* __restrict__ dinv, int64_t n_sq) {
  if (sc->done) return;
  double sq = 0.0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x) {
    double t = v[i];
    if (dinv) { t *= dinv[i]; v[i] = t; }
    if (i < n_sq) sq = fma(t, t, sq);
  }
  sq = block_sum(sq);
  if (threadIdx.x == 0) atomicAdd(&sc->vsq, sq);
}

// alpha = ||A^T u||; the remaining initial scalars                                   (init)
__global__ void k_init_s2(DevScalars* sc) {
  const double beta = sc->beta;
  const double alpha = beta > 0.0 ? sqrt(sc->vsq) : 0.0;
  sc->alpha = alpha;
  sc->inv_alpha = alpha > 0.0 ? 1.0 / alpha : 0.0;
  sc->arnorm = alpha * beta;
  sc->rhobar = alpha;
  sc->phibar = beta;
  sc->rnorm = beta;
  sc->anorm = 0.0; sc->acond = 0.0; sc->ddnorm = 0.0; sc->xnorm = 0.0; sc->xxnorm = 0.0;
  sc->z = 0.0; sc->cs2 = -1.0; sc->sn2 = 0.0;
  sc->c0_u = beta > 0.0 ? -alpha / beta : 0.0;
  sc->vsq = 0.0;
  if (alpha * beta == 0.0) { sc->istop = 0; sc->done = 1; }   // x = 0 is the exact solution
}

// v /= alpha ; w = v ; x = 0 ; wsq = ||w||^2                                         (init)
// (vs = D^-1 v is what the matrix pass gathers when a preconditioner is on; var starts at 0)
__global__ void __launch_bounds__(256) k_init_vw(double* __restrict__ v, double* __restrict__ w,
                                                 double* __restrict__ x, int64_t n, DevScalars* sc,
                                                 double* __restrict__ vs, const double* __restrict__ dinv,
                                                 double* __restrict__ var, int64_t n_sq) {
  const double ia = sc->inv_alpha;
  double sq = 0.0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x) {
    const double t = v[i] * ia;
    v[i] = t;
    w[i] = t;
    x[i] = 0.0;
    if (vs) vs[i] = t * dinv[i];
    if (var) var[i] = 0.0;
    if (i < n_sq) sq = fma(t, t, sq);
  }
  sq = block_sum(sq);
  if (threadIdx.x == 0) atomicAdd(&sc->wsq, sq);
}

// step 2a: beta = ||u_hat||; v <- -beta v (then aprod2 adds A^T u).  Thread 0 publishes beta,
// 1/beta and anorm; usq is left intact for the other blocks and cleared by k_step_scalars.
__global__ void __launch_bounds__(256) k_vscale(double* __restrict__ v, int64_t n, DevScalars* sc) {
  if (sc->done) return;
  const double beta = sqrt(sc->usq);
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    sc->beta = beta;
    sc->s_y = beta > 0.0 ? 1.0 / beta : 0.0;
    if (beta > 0.0) sc->anorm = sqrt(sc->anorm * sc->anorm + sc->alpha * sc->alpha + beta * beta);
  }
  if (!(beta > 0.0)) return;                         // P-S: v, alpha unchanged when beta = 0
  const double nb = -beta;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x)
    v[i] *= nb;
}

// fused path, step 2: beta = ||u_hat||; v <- g / beta - beta v (un-normalised v'), vsq = ||v'||^2.
// g = A^T u_hat was accumulated by the fused pass.  Thread 0 publishes beta, 1/beta and anorm.
// With a preconditioner g holds A^T u_hat and the operator's transpose is D^-1 A^T: g is scaled on the fly.
__global__ void __launch_bounds__(256) k_vcombine(double* __restrict__ v, const double* __restrict__ g, int64_t n,
                                                  DevScalars* sc, const double* __restrict__ dinv, int64_t n_sq) {
  if (sc->done) return;
  const double beta = sqrt(sc->usq);
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    sc->beta = beta;
    sc->s_y = beta > 0.0 ? 1.0 / beta : 0.0;
    if (beta > 0.0) sc->anorm = sqrt(sc->anorm * sc->anorm + sc->alpha * sc->alpha + beta * beta);
  }
  if (!(beta > 0.0)) return;                         // P-S: v, alpha unchanged when beta = 0
  const double ib = 1.0 / beta, nb = -beta;
  double sq = 0.0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x) {
    const double gi = dinv ? g[i] * dinv[i] : g[i];
    const double t = fma(nb, v[i], gi * ib);
    v[i] = t;
    if (i < n_sq) sq = fma(t, t, sq);
  }
  sq = block_sum(sq);
  if (threadIdx.x == 0) atomicAdd(&sc->vsq, sq);
}

// steps 2b-8 of DESIGN.md section 4 (scalars only): alpha, plane rotation, norm estimates, stopping rule
__global__ void k_step_scalars(DevScalars* sc, int64_t itnlim, double atol, double btol, double conlim) {
  if (sc->done) return;
  const double beta = sc->beta;
  double alpha = sc->alpha;
  if (beta > 0.0) alpha = sqrt(sc->vsq);
  sc->inv_alpha = (beta > 0.0 && alpha > 0.0) ? 1.0 / alpha : 1.0;
  // 3: plane rotation
  const double rho = sqrt(sc->rhobar * sc->rhobar + beta * beta);
  const double cs = sc->rhobar / rho, sn = beta / rho;
  const double theta = sn * alpha;
  sc->rhobar = -cs * alpha;
  const double phi = cs * sc->phibar;
  sc->phibar = sn * sc->phibar;
  const double tau = sn * phi;
  // 4: coefficients of the x / w update; ||w/rho||^2 = wsq / rho^2
  sc->t1 = phi / rho;
  sc->t2 = -theta / rho;
  sc->inv_rho = 1.0 / rho;
  sc->ddnorm += sc->wsq / (rho * rho);
  // 5: ||x|| estimate
  const double delta = sc->sn2 * rho, gambar = -sc->cs2 * rho, rhs = phi - delta * sc->z;
  const double zbar = rhs / gambar;
  sc->xnorm = sqrt(sc->xxnorm + zbar * zbar);
  const double gamma = sqrt(gambar * gambar + theta * theta);
  sc->cs2 = gambar / gamma;
  sc->sn2 = theta / gamma;
  sc->z = rhs / gamma;
  sc->xxnorm += sc->z * sc->z;
  // 6: norm estimates
  sc->acond = sc->anorm * sqrt(sc->ddnorm);
  sc->rnorm = fabs(sc->phibar);
  sc->arnorm = alpha * fabs(tau);
  sc->alpha = alpha;
  sc->c0_u = beta > 0.0 ? -alpha / beta : 0.0;      // next aprod1: u_hat <- A v - (alpha/beta) u_hat
  const long long itn = ++sc->itn;
  // 7-8: stopping rule (later tests override earlier ones)
  const double ctol = conlim > 0.0 ? 1.0 / conlim : 0.0;
  const double test1 = sc->rnorm / sc->bnorm;
  const double den2 = sc->anorm * sc->rnorm;
  const double test2 = den2 > 0.0 ? sc->arnorm / den2 : 0.0;
  const double test3 = 1.0 / sc->acond;
  const double t1p = test1 / (1.0 + sc->anorm * sc->xnorm / sc->bnorm);
  const double rtol = btol + atol * sc->anorm * sc->xnorm / sc->bnorm;
  int istop = 0;
  if (itn >= itnlim) istop = 7;
  if (1.0 + test3 <= 1.0) istop = 6;
  if (1.0 + test2 <= 1.0) istop = 5;
  if (1.0 + t1p <= 1.0) istop = 4;
  if (test3 <= ctol) istop = 3;
  if (test2 <= atol) istop = 2;
  if (test1 <= rtol) istop = 1;
  sc->istop = istop;
  sc->usq = 0.0;
  sc->vsq = 0.0;
  sc->wsq = 0.0;
  if (istop) sc->done = 2;  // 2 = stopped, but this iteration's k_update must still run (P-S updates x
                            // before testing); the next aprod1 launch latches 2 -> 1
}

// step 4 (vectors): v /= alpha ; x += t1 w ; w = v + t2 w ; wsq = ||w_new||^2
// optional: var += (w_old / rho)^2 (Paige-Saunders' variance estimate); vs = D^-1 v (preconditioned gather vector)
__global__ void __launch_bounds__(256) k_update(double* __restrict__ v, double* __restrict__ w,
                                                double* __restrict__ x, int64_t n, DevScalars* sc,
                                                double* __restrict__ vs, const double* __restrict__ dinv,
                                                double* __restrict__ var, int64_t n_sq) {
  if (sc->done == 1) return;
  const double ia = sc->inv_alpha, t1 = sc->t1, t2 = sc->t2, ir = sc->inv_rho;
  double sq = 0.0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n;
       i += (int64_t)gridDim.x * blockDim.x) {
    const double vi = v[i] * ia, wi = w[i];
    v[i] = vi;
    if (vs) vs[i] = vi * dinv[i];
    if (var) { const double dk = ir * wi; var[i] = fma(dk, dk, var[i]); }
    x[i] = fma(t1, wi, x[i]);
    const double wn = fma(t2, wi, vi);
    w[i] = wn;
    if (i < n_sq) sq = fma(wn, wn, sq);
  }
  sq = block_sum(sq);
  if (threadIdx.x == 0) atomicAdd(&sc->wsq, sq);
}

// u = u_hat / beta (export only)
__global__ void __launch_bounds__(256) k_export_u(const double* __restrict__ uhat, double* __restrict__ u,
                                                  int64_t M, const DevScalars* sc) {
  const double s = sc->s_y;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < M;
       i += (int64_t)gridDim.x * blockDim.x)
    u[i] = uhat[i] * s;
}

#define LAUNCHED() (++*launches, cudaGetLastError())

cudaError_t lsqr_launch_init_u(const double* b, double* u, int64_t M, DevScalars* sc, cudaStream_t st, int64_t* launches) {
  k_init_u<<<grid_for(M, 256, 4), 256, 0, st>>>(b, u, M, sc);
  return LAUNCHED();
}
cudaError_t lsqr_launch_init_s1(DevScalars* sc, cudaStream_t st, int64_t* launches) {
  k_init_s1<<<1, 1, 0, st>>>(sc);
  return LAUNCHED();
}
cudaError_t lsqr_launch_sumsq_v(double* v, int64_t n, DevScalars* sc, const double* dinv, cudaStream_t st,
                                int64_t* launches, int64_t n_sq) {
  k_sumsq_v<<<grid_for(n, 256, 4), 256, 0, st>>>(v, n, sc, dinv, n_sq < 0 ? n : n_sq);
  return LAUNCHED();
}
cudaError_t lsqr_launch_init_s2(DevScalars* sc, cudaStream_t st, int64_t* launches) {
  k_init_s2<<<1, 1, 0, st>>>(sc);
  return LAUNCHED();
}
cudaError_t lsqr_launch_init_vw(double* v, double* w, double* x, int64_t n, DevScalars* sc, double* vs,
                                const double* dinv, double* var, cudaStream_t st, int64_t* launches, int64_t n_sq) {
  k_init_vw<<<grid_for(n, 256, 4), 256, 0, st>>>(v, w, x, n, sc, vs, dinv, var, n_sq < 0 ? n : n_sq);
  return LAUNCHED();
}
cudaError_t lsqr_launch_vscale(double* v, int64_t n, DevScalars* sc, cudaStream_t st, int64_t* launches) {
  k_vscale<<<grid_for(n, 256, 4), 256, 0, st>>>(v, n, sc);
  return LAUNCHED();
}
cudaError_t lsqr_launch_vcombine(double* v, const double* g, int64_t n, DevScalars* sc, const double* dinv,
                                 cudaStream_t st, int64_t* launches, int64_t n_sq) {
  k_vcombine<<<grid_for(n, 256, 4), 256, 0, st>>>(v, g, n, sc, dinv, n_sq < 0 ? n : n_sq);
  return LAUNCHED();
}
cudaError_t lsqr_launch_step_scalars(DevScalars* sc, int64_t itnlim, double atol, double btol, double conlim,
                                     cudaStream_t st, int64_t* launches) {
  k_step_scalars<<<1, 1, 0, st>>>(sc, itnlim, atol, btol, conlim);
  return LAUNCHED();
}
cudaError_t lsqr_launch_update(double* v, double* w, double* x, int64_t n, DevScalars* sc, double* vs,
                               const double* dinv, double* var, cudaStream_t st, int64_t* launches, int64_t n_sq) {
  k_update<<<grid_for(n, 256, 4), 256, 0, st>>>(v, w, x, n, sc, vs, dinv, var, n_sq < 0 ? n : n_sq);
  return LAUNCHED();
}

// ---- column norms and the diagonal preconditioner (reading R7) ----------
// The squared column norms are accumulated by the aprod 2 tile kernel with its coefficients squared on the
// fly (aprod2.cu, square = 1), into an LSQR-internal n-vector (attitude block interleaved).
// mode 0: d <- sqrt(d2) (column norms); mode 1: d <- 1 / sqrt(d2), 1 for a column no row touches (D^-1)
__global__ void __launch_bounds__(256) k_colnorm_finish(double* __restrict__ d, int64_t n, int mode) {
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const double q = sqrt(d[i]);
    d[i] = mode == 0 ? q : (q > 0.0 ? 1.0 / q : 1.0);
  }
}
// dst = src * s (power 1) or src * s^2 (power 2): x = D^-1 z, var_x = D^-2 var_z
__global__ void __launch_bounds__(256) k_scale_by(double* __restrict__ dst, const double* __restrict__ src,
                                                  const double* __restrict__ s, int64_t n, int power) {
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const double f = s[i];
    dst[i] = src[i] * (power == 2 ? f * f : f);
  }
}
// ---- covariances of chosen pairs (Eq. 4; R21) ---------
// position of API column j inside an LSQR-internal n-vector (attitude block interleaved: il[3*t + ax])
__device__ __forceinline__ int64_t internal_index(const SysView& s, int64_t j) {
  if (j < s.oA || j >= s.oI) return j;
  const int64_t e = j - s.oA, ax = e / s.K, t = e - ax * s.K;
  return s.oA + 3 * t + ax;
}
// cov[p] += (1/rho^2) * w[j1[p]] * w[j2[p]] with the w BEFORE this iteration's update (run before k_update);
// a gather-multiply-accumulate over the pair list, 24 bytes of list + accumulator traffic per pair.
__global__ void __launch_bounds__(256) k_cov_update(SysView s, const double* __restrict__ w, const DevScalars* sc,
                                                    const int64_t* __restrict__ j1, const int64_t* __restrict__ j2,
                                                    int64_t n_pairs, double* __restrict__ cov) {
  if (sc->done == 1) return;
  const double f = sc->inv_rho * sc->inv_rho;
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < n_pairs; p += (int64_t)gridDim.x * blockDim.x)
    cov[p] = fma(f * __ldg(w + internal_index(s, j1[p])), __ldg(w + internal_index(s, j2[p])), cov[p]);
}
// preconditioned run: cov_x = dinv[j1] * dinv[j2] * cov_z
__global__ void __launch_bounds__(256) k_cov_unscale(SysView s, const double* __restrict__ dinv,
                                                     const int64_t* __restrict__ j1, const int64_t* __restrict__ j2,
                                                     int64_t n_pairs, double* __restrict__ cov) {
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < n_pairs; p += (int64_t)gridDim.x * blockDim.x)
    cov[p] *= __ldg(dinv + internal_index(s, j1[p])) * __ldg(dinv + internal_index(s, j2[p]));
}
__global__ void __launch_bounds__(256) k_check_pairs(const int64_t* __restrict__ j1, const int64_t* __restrict__ j2,
                                                     int64_t n_pairs, int64_t n, int* bad) {
  for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < n_pairs; p += (int64_t)gridDim.x * blockDim.x)
    if (j1[p] < 0 || j1[p] >= n || j2[p] < 0 || j2[p] >= n) *bad = 1;
}
cudaError_t lsqr_launch_cov_update(const SysView& s, const double* w, const DevScalars* sc, const int64_t* j1,
                                   const int64_t* j2, int64_t n_pairs, double* cov, cudaStream_t st, int64_t* launches) {
  if (n_pairs == 0) return cudaSuccess;
  k_cov_update<<<grid_for(n_pairs, 256, 4), 256, 0, st>>>(s, w, sc, j1, j2, n_pairs, cov);
  return LAUNCHED();
}
cudaError_t lsqr_launch_cov_unscale(const SysView& s, const double* dinv, const int64_t* j1, const int64_t* j2,
                                    int64_t n_pairs, double* cov, cudaStream_t st, int64_t* launches) {
  if (n_pairs == 0) return cudaSuccess;
  k_cov_unscale<<<grid_for(n_pairs, 256, 4), 256, 0, st>>>(s, dinv, j1, j2, n_pairs, cov);
  return LAUNCHED();
}
cudaError_t lsqr_launch_check_pairs(const int64_t* j1, const int64_t* j2, int64_t n_pairs, int64_t n, int* bad,
                                    cudaStream_t st, int64_t* launches) {
  if (n_pairs == 0) return cudaSuccess;
  k_check_pairs<<<grid_for(n_pairs, 256, 4), 256, 0, st>>>(j1, j2, n_pairs, n, bad);
  return LAUNCHED();
}
cudaError_t lsqr_launch_colnorm_finish(double* d, int64_t n, int mode, cudaStream_t st, int64_t* launches) {
  k_colnorm_finish<<<grid_for(n, 256, 4), 256, 0, st>>>(d, n, mode);
  return LAUNCHED();
}
cudaError_t lsqr_launch_scale_by(double* dst, const double* src, const double* s, int64_t n, int power, cudaStream_t st,
                                 int64_t* launches) {
  k_scale_by<<<grid_for(n, 256, 4), 256, 0, st>>>(dst, src, s, n, power);
  return LAUNCHED();
}
cudaError_t lsqr_launch_export_u(const double* uhat, double* u, int64_t M, const DevScalars* sc, cudaStream_t st, int64_t* launches) {
  k_export_u<<<grid_for(M, 256, 4), 256, 0, st>>>(uhat, u, M, sc);
  return LAUNCHED();
}

// ---- row-sharded solve (gsr.h gsr_shard_*) --------------------------
// Between two phases of a sharded solve the caller sums the exchange buffer over the ranks.  This kernel moves the
// replicated tail of an n-vector (attitude, instrumental, global: ns doubles from `vec`) and the partial sums of
// squares between the library's own state and that buffer.  No-op once the solve has stopped.
//   pack   : xbuf[0..ns) = vec (when ns > 0) ; then the scalars named by `what`, appended after the vector part
//   unpack : the reverse
__global__ void __launch_bounds__(256) k_shard_xfer(double* __restrict__ vec, int64_t ns, DevScalars* sc,
                                                    double* __restrict__ xbuf, int what, int unpack) {
  if (sc->done) return;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < ns; i += (int64_t)gridDim.x * blockDim.x) {
    if (unpack) vec[i] = xbuf[i];
    else xbuf[i] = vec[i];
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    double* q = xbuf + ns;
    if (what == SHARD_X_USQ) { if (unpack) sc->usq = q[0]; else q[0] = sc->usq; }
    else if (what == SHARD_X_VSQ) { if (unpack) sc->vsq = q[0]; else q[0] = sc->vsq; }
    else if (what == SHARD_X_USQ_WSQ) {
      if (unpack) { sc->usq = q[0]; sc->wsq = q[1]; }
      else { q[0] = sc->usq; q[1] = sc->wsq; }
    }
  }
}
cudaError_t lsqr_launch_shard_xfer(double* vec, int64_t ns, DevScalars* sc, double* xbuf, int what, int unpack,
                                   cudaStream_t st, int64_t* launches) {
  k_shard_xfer<<<grid_for(ns, 256, 4), 256, 0, st>>>(vec, ns, sc, xbuf, what, unpack);
  return LAUNCHED();
}

}  // namespace gsr
