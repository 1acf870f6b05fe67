// C ABI of libgsr (include/gsr.h): argument checking, ownership, the LSQR driver.
// Every step of the path runs in the kernels of aprod1.cu / aprod2.cu / lsqr_kernels.cu.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "gsr_internal.cuh"
#include "tma.cuh"

using namespace gsr;

static thread_local char g_cuda_err[256] = "";

static int cuda_fail(cudaError_t e, const char* where) {
  snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", where, cudaGetErrorString(e));
  return GSR_ECUDA;
}
#define CU(call)                                           \
  do {                                                     \
    cudaError_t e_ = (call);                               \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call);    \
  } while (0)

// cudaMalloc with the ABI's error mapping: an allocation failure is GSR_ENOMEM (and is not left pending).
static int dev_alloc(void** p, size_t bytes, const char* what) {
  cudaError_t e = cudaMalloc(p, bytes);
  if (e == cudaSuccess) return GSR_OK;
  *p = nullptr;
  cudaGetLastError();
  return e == cudaErrorMemoryAllocation ? GSR_ENOMEM : cuda_fail(e, what);
}
#define ALLOC(ptr, bytes)                                                        \
  do {                                                                           \
    int rc_ = dev_alloc(reinterpret_cast<void**>(&(ptr)), (bytes), #ptr);        \
    if (rc_) return rc_;                                                         \
  } while (0)

struct EventPair {
  cudaEvent_t a, b;
  int which;
};

struct IterGraph;
struct gsr_system {
  SysView v;
  SideData side;
  // the constraint equations as a section of their own, rows M .. M + con.M - 1
  SysView con;
  SideData con_side;          // its tensor map; every other member aliases `side`
  bool has_con = false;
  Tuning tune;
  int device = 0;
  int num_sms = 148;
  int64_t launches = 0;
  // LSQR workspace (allocated on first use)
  double *u = nullptr, *vv = nullptr, *w = nullptr, *x = nullptr, *g = nullptr;
  DevScalars* sc = nullptr;
  bool lsqr_ready = false;   // gsr_lsqr_init has run
  IterGraph* iter_graph = nullptr;   // cached CUDA graph of a batch of iterations (small systems)
  cudaStream_t cap_stream = nullptr; // the stream those batches are captured on
  // column-norm preconditioning and variances (gsr_lsqr_ex); buffers allocated on first use
  double *dinv = nullptr, *vs = nullptr, *var = nullptr;   // D^-1, D^-1 v (the vector the matrix pass gathers), var
  bool opt_precond = false, opt_var = false;               // options of the run set up by the last lsqr init
  // covariances of chosen pairs (gsr_set_cov_pairs); the three arrays are borrowed
  const int64_t *cov_j1 = nullptr, *cov_j2 = nullptr;
  double* cov = nullptr;
  int64_t n_cov = 0;
  bool opt_cov = false, opt_cov_next = false;              // (opt_cov_next: set by gsr_lsqr_ex for its own init)
  // row-sharded solve in phases (gsr_shard_*); -1 = none in progress
  int shard_next = -1;                                     // the phase the next gsr_shard_phase call runs
  bool shard_counts_shared = false;                        // this rank counts the replicated tail in the sums of squares
  double* shard_xbuf = nullptr;                            // borrowed exchange buffer (n - 5S + 2 doubles)
  int64_t shard_itnlim = 0;
  double shard_atol = 0, shard_btol = 0, shard_conlim = 0;
  // profiling
  bool profile = false;
  std::vector<EventPair> pending;
  std::vector<EventPair> pool;
  double prof_ms[4] = {0, 0, 0, 0};
  int64_t prof_n[4] = {0, 0, 0, 0};
};

static inline cudaStream_t S(void* s) { return reinterpret_cast<cudaStream_t>(s); }
static inline int64_t m_total(const gsr_system* s) { return s->v.M + s->con.M; }      // observation + constraint rows
// one pass over A per LSQR iteration (the TMA tile kernels, either record format)
static inline bool fused_path(const gsr_system* s) { return s->tune.fused != 0; }

extern "C" const char* gsr_strerror(int code) {
  switch (code) {
    case GSR_OK: return "ok";
    case GSR_EINVAL: return "invalid argument";
    case GSR_ELAYOUT: return "index records violate the layout";
    case GSR_ENOMEM: return "out of memory";
    case GSR_ECUDA: return "CUDA error";
    case GSR_ESTATE: return "call out of order";
    default: return "unknown error";
  }
}
extern "C" const char* gsr_last_cuda_error(void) { return g_cuda_err; }
extern "C" const char* gsr_version(void) { return "gsr-b200 0.1 (sm_100a)"; }

static bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda).
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static int make_row_tensor_map(CUtensorMap* map, const double* values, int64_t M, int cpr) {
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
  if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn)
    return cuda_fail(e != cudaSuccess ? e : cudaErrorUnknown, "cudaGetDriverEntryPoint(cuTensorMapEncodeTiled)");
  // group view (tma.cuh): one tensor row = a GROUP of matrix rows (two 192-byte or four 184-byte records: a whole number
  // of 16-byte units, which the pitch needs); the last M mod GROUP rows are not covered (TileRing::acquire copies them)
  const int group = cpr == NSLOT ? Rec24::GROUP : Rec23::GROUP;
  const cuuint64_t dims[2] = {(cuuint64_t)(group * cpr), (cuuint64_t)(M >= group ? M / group : 1)};
  const cuuint64_t strides[1] = {(cuuint64_t)(group * cpr) * sizeof(double)};
  const cuuint32_t box[2] = {(cuuint32_t)(cpr == NSLOT ? Rec24::BOX_COLS : Rec23::BOX_COLS),      // the group + zero-filled pad columns
                             (cuuint32_t)(TILE_ROWS / group)};
  const cuuint32_t estr[2] = {1u, 1u};
  CUresult r = reinterpret_cast<EncodeTiledFn>(fn)(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(values),
                                                   dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                                   CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
    return GSR_ECUDA;
  }
  return GSR_OK;
}

// Side buffers for the standalone products: the attitude block in the interleaved layout (aprod 1 input
// copy, aprod 2 accumulator).  LSQR-internal vectors are interleaved already and do not use them.
static int build_att_buffers(gsr_system* s) {
  const size_t bytes = (size_t)(3 * s->v.K) * sizeof(double);
  cudaError_t e = cudaMalloc(&s->side.att_il, bytes);
  if (e == cudaSuccess) e = cudaMalloc(&s->side.att_acc, bytes);
  if (e != cudaSuccess) { cudaGetLastError(); return e == cudaErrorMemoryAllocation ? GSR_ENOMEM : cuda_fail(e, "cudaMalloc att"); }
  e = cudaMemset(s->side.att_acc, 0, bytes);
  if (e != cudaSuccess) return cuda_fail(e, "cudaMemset att_acc");
  return GSR_OK;
}

// ---- die-local replicated instrumental accumulators (InstrAcc, gsr_internal.cuh) ------------------
// probe_homes: which die is the L2 home of each 4 KB chunk of the pool, and on which die does each SM sit?
// Thread 0 of every block times a short chain of dependent fp64 atomics (add 0.0) to each of N_REF
// reference chunks: the latencies fall into two groups, ~330 and ~720 cycles on B200 (near / far die).
// Die 0 is DEFINED as the home of reference chunk 0; an SM that sees that chunk near sits on die 0.  The
// block then classifies its share of the pool the same way.  A wrong call only costs speed, never
// correctness: every chunk is a valid accumulator whoever reduces into it.
constexpr int N_REF = 16;
#ifdef GSR_HOST_EMULATION
// (tests/emu: no dies on the host; every chunk answers alike, so the probe reports one die)
__device__ __forceinline__ float atom_latency(double* p, int reps) { atomicAdd(p, 0.0); return 100.0f + 0.0f * (float)reps; }
#else
__device__ __forceinline__ float atom_latency(double* p, int reps) {
  double v;
  asm volatile("atom.global.add.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "d"(0.0) : "memory");   // warm
  const long long t0 = clock64();
  for (int r = 0; r < reps; r++) {
    double* q = p + (long long)(v * 0.0);   // address depends on the previous result: a serial chain
    asm volatile("atom.global.add.f64 %0, [%1], %2;" : "=d"(v) : "l"(q), "d"(0.0) : "memory");
  }
  const long long t1 = clock64();
  return (float)(t1 - t0) / (float)reps + (float)(v * 0.0);
}
#endif
__global__ void k_probe_homes(double* pool, int n_pool, int* sm_die, signed char* home, int* bimodal) {
  if (threadIdx.x != 0) return;
  unsigned smid;
#ifdef GSR_HOST_EMULATION
  smid = emu::smid();
#else
  asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
#endif
  float ref[N_REF], srt[N_REF];
  const int off = (int)((blockIdx.x * 4u) % INS_CHUNK);   // own sector of every reference chunk: no same-address contention
  for (int c = 0; c < N_REF; c++) atom_latency(pool + (size_t)c * INS_CHUNK + off, 2);   // untimed pass: TLB, first touch
  for (int c = 0; c < N_REF; c++) srt[c] = ref[c] = atom_latency(pool + (size_t)c * INS_CHUNK + off, 8);
  for (int i = 1; i < N_REF; i++)   // insertion sort; the threshold is the middle of the widest gap
    for (int j = i; j > 0 && srt[j] < srt[j - 1]; j--) { const float t = srt[j]; srt[j] = srt[j - 1]; srt[j - 1] = t; }
  int g = 1;
  for (int i = 2; i < N_REF; i++)
    if (srt[i] - srt[i - 1] > srt[g] - srt[g - 1]) g = i;
  if (srt[g] < 1.4f * srt[g - 1]) { atomicAnd(bimodal, 0); return; }   // no two groups seen from this SM: one die (or an unknown part)
  const float thr = 0.5f * (srt[g] + srt[g - 1]);
  const int my_die = ref[0] < thr ? 0 : 1;
  if (smid < (unsigned)SMID_SLOTS) sm_die[smid] = my_die;
  for (int c = blockIdx.x; c < n_pool; c += gridDim.x) {
    const bool near_ = atom_latency(pool + (size_t)c * INS_CHUNK, 8) < thr;
    home[c] = (signed char)(near_ ? my_die : 1 - my_die);
  }
}

// Copies per die: enough that a copy is shared by few CTAs (60,000 addresses hit by 3e9 reductions are
// contention-bound otherwise), within ~4 MB in total, at least 4 per die.
static int build_instr_copies(gsr_system* s) {
  const SysView& v = s->v;
  InstrAcc& ia = s->side.ins;
  int64_t cpd = (int64_t)(2u << 20) / (v.I * 8);   // (1 to 16 MB per die measured the same at C4)
  if (cpd > s->num_sms / 2) cpd = s->num_sms / 2;
  if (cpd < 4) cpd = 4;
  const int64_t n_chunks = (v.I + INS_CHUNK - 1) / INS_CHUNK;
  const int64_t need = 2 * cpd * n_chunks;
  const int64_t n_pool = need + need / 4 + 64 + N_REF;
  const size_t chunk_bytes = INS_CHUNK * sizeof(double);
  int* bimodal = nullptr;
  signed char* home = nullptr;
  cudaError_t e = cudaMalloc(&ia.pool, (size_t)(n_pool + 1) * chunk_bytes);
  if (e == cudaSuccess) e = cudaMalloc(&ia.sm_die, SMID_SLOTS * sizeof(int));
  if (e == cudaSuccess) e = cudaMalloc(&ia.chunk_tab, (size_t)need * sizeof(double*));
  if (e == cudaSuccess) e = cudaMalloc(&home, (size_t)n_pool);
  if (e == cudaSuccess) e = cudaMalloc(&bimodal, sizeof(int));
  if (e != cudaSuccess) { cudaGetLastError(); cudaFree(home); cudaFree(bimodal); return e == cudaErrorMemoryAllocation ? GSR_ENOMEM : cuda_fail(e, "cudaMalloc instr accumulators"); }
  double* base = reinterpret_cast<double*>((reinterpret_cast<uintptr_t>(ia.pool) + chunk_bytes - 1) / chunk_bytes * chunk_bytes);
  const int one = 1;
  e = cudaMemset(ia.pool, 0, (size_t)(n_pool + 1) * chunk_bytes);
  if (e == cudaSuccess) e = cudaMemset(ia.sm_die, 0xff, SMID_SLOTS * sizeof(int));
  if (e == cudaSuccess) e = cudaMemset(home, 0, (size_t)n_pool);
  if (e == cudaSuccess) e = cudaMemcpy(bimodal, &one, sizeof(int), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    k_probe_homes<<<2 * s->num_sms, 32>>>(base, (int)n_pool, ia.sm_die, home, bimodal);
    ++s->launches;
    e = cudaGetLastError();
  }
  std::vector<signed char> h((size_t)n_pool);
  int two = 0;
  if (e == cudaSuccess) e = cudaMemcpy(h.data(), home, (size_t)n_pool, cudaMemcpyDeviceToHost);
  if (e == cudaSuccess) e = cudaMemcpy(&two, bimodal, sizeof(int), cudaMemcpyDeviceToHost);
  cudaFree(home);
  cudaFree(bimodal);
  if (e != cudaSuccess) return cuda_fail(e, "probe_homes");
  // sets 0 .. cpd-1: chunks homed on die 0; sets cpd .. 2 cpd-1: die 1 (a die that runs short borrows from the other)
  std::vector<int64_t> by_die[2];
  for (int64_t c = N_REF; c < n_pool; c++) by_die[two ? (h[(size_t)c] != 0) : (c & 1)].push_back(c);
  std::vector<double*> tab((size_t)need);
  size_t take[2] = {0, 0};
  for (int d = 0; d < 2; d++)
    for (int64_t k = 0; k < cpd * n_chunks; k++) {
      int src = take[d] < by_die[d].size() ? d : 1 - d;
      tab[(size_t)(d * cpd * n_chunks + k)] = base + (size_t)by_die[src][take[src]++] * INS_CHUNK;
    }
  e = cudaMemcpy(ia.chunk_tab, tab.data(), (size_t)need * sizeof(double*), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) return cuda_fail(e, "cudaMemcpy chunk table");
  ia.base = base;
  ia.copies_per_die = (int)cpd;
  ia.n_chunks = (int)n_chunks;
  ia.two_dies = two != 0;
  ia.n_sets = (int)(2 * cpd);   // with one die, load_ins_tab uses sets 0 .. cpd-1 only; the others stay zero
  return GSR_OK;
}

static int check_layout(const gsr_layout* L) {
  if (!L) return GSR_EINVAL;
  if (L->n_rows < 0 || L->n_stars < 1 || L->n_knots < 4 || L->n_instr < 1) return GSR_EINVAL;
  if (L->n_glob != 0 && L->n_glob != 1) return GSR_EINVAL;
  if (L->flags & ~(GSR_LAYOUT_TRUSTED | GSR_LAYOUT_COEFF23)) return GSR_EINVAL;
  if ((L->flags & GSR_LAYOUT_COEFF23) && L->n_glob != 0) return GSR_EINVAL;   // the 23-slot record has no global slot
  if (L->n_stars > INT32_MAX || L->n_knots > INT32_MAX || L->n_instr > INT32_MAX) return GSR_EINVAL;
  return GSR_OK;
}

extern "C" int gsr_create(gsr_system** out, const gsr_layout* L, const double* values,
                          const int32_t* indices, void* stream) {
  if (!out) return GSR_EINVAL;
  *out = nullptr;
  if (check_layout(L)) return GSR_EINVAL;
  if (L->n_rows > 0 && (!values || !indices)) return GSR_EINVAL;
  if (!aligned(values, 32) || !aligned(indices, 32)) return GSR_EINVAL;
  int dev = 0;
  CU(cudaGetDevice(&dev));
  gsr_system* s = new (std::nothrow) gsr_system();
  if (!s) return GSR_ENOMEM;
  s->device = dev;
  cudaError_t e = cudaDeviceGetAttribute(&s->num_sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) { delete s; return cuda_fail(e, "cudaDeviceGetAttribute"); }
  SysView& v = s->v;
  v.vals = values; v.idx = indices;
  v.M = L->n_rows; v.S = L->n_stars; v.K = L->n_knots; v.I = L->n_instr; v.G = L->n_glob;
  v.oA = 5 * v.S; v.oI = v.oA + 3 * v.K; v.oG = v.oI + v.I; v.n = v.oG + v.G;
  v.cpr = (L->flags & GSR_LAYOUT_COEFF23) ? NSLOT - 1 : NSLOT;
  s->con = v;
  s->con.vals = nullptr; s->con.idx = nullptr; s->con.M = 0;
  // device-side validation of every index record (skipped when the caller vouches for them)
  if (!(L->flags & GSR_LAYOUT_TRUSTED)) {
    int* flag = nullptr;
    int rc = dev_alloc(reinterpret_cast<void**>(&flag), sizeof(int), "cudaMalloc flag");
    if (rc) { delete s; return rc; }
    int h = 0;
    cudaStream_t st = S(stream);
    e = cudaMemsetAsync(flag, 0, sizeof(int), st);
    if (e == cudaSuccess) e = launch_validate(v, flag, st, &s->launches);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(flag);
    if (e != cudaSuccess) { delete s; return cuda_fail(e, "gsr_create validation"); }
    if (h != 0) { delete s; return GSR_ELAYOUT; }
  }
  // side structures: the row-tile tensor map, the interleaved attitude buffers, instrumental replicas
  if (v.M > 0) {
    int rc = make_row_tensor_map(&s->side.map, values, v.M, v.cpr);
    if (rc) { delete s; return rc; }
  }
  int rc2 = build_att_buffers(s);
  if (rc2 == GSR_OK) rc2 = build_instr_copies(s);
  if (rc2) { gsr_destroy(s); return rc2; }
  *out = s;
  return GSR_OK;
}

static void free_events(gsr_system* s) {
  for (auto& p : s->pending) { cudaEventDestroy(p.a); cudaEventDestroy(p.b); }
  for (auto& p : s->pool) { cudaEventDestroy(p.a); cudaEventDestroy(p.b); }
  s->pending.clear();
  s->pool.clear();
}

static void free_iter_graph(gsr_system* s);

extern "C" void gsr_destroy(gsr_system* s) {
  if (!s) return;
  free_iter_graph(s);
  cudaFree(s->u); cudaFree(s->vv); cudaFree(s->w); cudaFree(s->x); cudaFree(s->sc);
  cudaFree(s->side.att_il); cudaFree(s->side.att_acc); cudaFree(s->side.ins.pool); cudaFree(s->side.ins.sm_die); cudaFree(s->side.ins.chunk_tab); cudaFree(s->g); cudaFree(s->side.det_part);
  cudaFree(s->dinv); cudaFree(s->vs); cudaFree(s->var);
  free_events(s);
  delete s;
}

extern "C" int gsr_attach_constraints(gsr_system* s, int64_t n_rows, const double* values, const int32_t* indices,
                                      void* stream) {
  if (!s || n_rows < 0) return GSR_EINVAL;
  if (n_rows > 0 && (!values || !indices)) return GSR_EINVAL;
  if (!aligned(values, 32) || !aligned(indices, 32)) return GSR_EINVAL;
  s->lsqr_ready = false;                 // the row count changes: work vectors are re-made, a running solve is void
  s->shard_next = -1;
  free_iter_graph(s);
  cudaFree(s->u); s->u = nullptr;
  cudaFree(s->vv); cudaFree(s->w); cudaFree(s->x); cudaFree(s->g); cudaFree(s->sc);
  s->vv = s->w = s->x = s->g = nullptr; s->sc = nullptr;
  s->has_con = false;
  s->con.vals = nullptr; s->con.idx = nullptr; s->con.M = 0;
  if (n_rows == 0) return GSR_OK;
  SysView c = s->v;
  c.vals = values; c.idx = indices; c.M = n_rows;
  int* flag = nullptr;
  int rc = dev_alloc(reinterpret_cast<void**>(&flag), sizeof(int), "cudaMalloc flag");
  if (rc) return rc;
  int h = 0;
  cudaStream_t st = S(stream);
  cudaError_t e = cudaMemsetAsync(flag, 0, sizeof(int), st);
  if (e == cudaSuccess) e = launch_validate(c, flag, st, &s->launches);
  if (e == cudaSuccess) e = cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(flag);
  if (e != cudaSuccess) return cuda_fail(e, "gsr_attach_constraints validation");
  if (h != 0) return GSR_ELAYOUT;
  s->con_side = s->side;                 // shares the attitude buffers and the instrumental replicas (never freed twice:
                                         // gsr_destroy frees `side` only)
  if ((rc = make_row_tensor_map(&s->con_side.map, values, n_rows, c.cpr))) return rc;
  s->con = c;
  s->has_con = true;
  return GSR_OK;
}

extern "C" int gsr_dims(const gsr_system* s, int64_t* m, int64_t* n) {
  if (!s) return GSR_EINVAL;
  if (m) *m = s->v.M + s->con.M;
  if (n) *n = s->v.n;
  return GSR_OK;
}

// ---- profiling helpers ---------------------------------------------------------------------
static bool prof_begin(gsr_system* s, int which, cudaStream_t st, EventPair* ep) {
  if (!s->profile) return false;
  if (!s->pool.empty()) { *ep = s->pool.back(); s->pool.pop_back(); }
  else {
    if (cudaEventCreate(&ep->a) != cudaSuccess) return false;
    if (cudaEventCreate(&ep->b) != cudaSuccess) { cudaEventDestroy(ep->a); return false; }
  }
  ep->which = which;
  cudaEventRecord(ep->a, st);
  return true;
}
static void prof_end(gsr_system* s, cudaStream_t st, EventPair* ep) {
  cudaEventRecord(ep->b, st);
  s->pending.push_back(*ep);
}

static int do_aprod1(gsr_system* s, const double* x, bool x_il, double* y, const double* c0, double* sumsq,
                     int* done, cudaStream_t st) {
  EventPair ep;
  const bool p = prof_begin(s, 1, st, &ep);
  cudaError_t e = launch_aprod1(s->v, s->side, s->tune, s->num_sms, x, x_il, y, c0, sumsq, done, st, &s->launches);
  if (e == cudaSuccess && s->has_con)   // (a stopped LSQR: the first launch latches done 2 -> 1, this one sees 1)
    e = launch_aprod1(s->con, s->con_side, s->tune, s->num_sms, x, x_il, y + s->v.M, c0, sumsq, done, st, &s->launches);
  if (p) prof_end(s, st, &ep);
  if (e != cudaSuccess) return cuda_fail(e, "aprod1 launch");
  return GSR_OK;
}
// deterministic debug variant: how many row chunks (each with a private copy of the shared columns), from the sizes alone
static int det_chunk_count(const gsr_system* s) {
  if (s->tune.det_chunks > 0) return s->tune.det_chunks;
  const int64_t ns = s->v.n - s->v.oA;
  int64_t c = (int64_t)(256u << 20) / (ns * 8);
  return (int)(c < 1 ? 1 : (c > 1024 ? 1024 : c));
}
static int ensure_det_pool(gsr_system* s, int C) {
  if (s->side.det_part && s->side.det_cap >= C) return GSR_OK;
  cudaFree(s->side.det_part);
  s->side.det_part = nullptr; s->side.det_cap = 0;
  ALLOC(s->side.det_part, (size_t)C * (size_t)(s->v.n - s->v.oA) * sizeof(double));
  s->side.det_cap = C;
  return GSR_OK;
}

static int do_aprod2(gsr_system* s, const double* y, double* x, bool x_il, const double* yscale, const int* done,
                     cudaStream_t st) {
  EventPair ep;
  cudaError_t e;
  if (s->tune.aprod2_variant == 2) {      // deterministic debug variant, both record formats, both sections in row order
    const int C = det_chunk_count(s);
    int rc = ensure_det_pool(s, C);
    if (rc) return rc;
    const bool p = prof_begin(s, 2, st, &ep);
    e = launch_aprod2_det(s->v, s->side.det_part, C, s->num_sms, y, x, x_il, yscale, done, st, &s->launches);
    if (e == cudaSuccess && s->has_con)
      e = launch_aprod2_det(s->con, s->side.det_part, C, s->num_sms, y + s->v.M, x, x_il, yscale, done, st, &s->launches);
    if (p) prof_end(s, st, &ep);
    if (e != cudaSuccess) return cuda_fail(e, "aprod2 (deterministic) launch");
    return GSR_OK;
  }
  const bool p = prof_begin(s, 2, st, &ep);
  e = launch_aprod2(s->v, s->side, s->tune, s->num_sms, y, x, x_il, yscale, done, st, &s->launches);
  if (e == cudaSuccess && s->has_con)
    e = launch_aprod2(s->con, s->con_side, s->tune, s->num_sms, y + s->v.M, x, x_il, yscale, done, st, &s->launches);
  if (p) prof_end(s, st, &ep);
  if (e != cudaSuccess) return cuda_fail(e, "aprod2 launch");
  return GSR_OK;
}

extern "C" int gsr_aprod1(gsr_system* s, const double* x, double* y, void* stream) {
  if (!s || !x || (!y && m_total(s) > 0)) return GSR_EINVAL;
  return do_aprod1(s, x, false, y, nullptr, nullptr, nullptr, S(stream));
}
extern "C" int gsr_aprod2(gsr_system* s, const double* y, double* x, void* stream) {
  if (!s || !x || (!y && m_total(s) > 0)) return GSR_EINVAL;
  return do_aprod2(s, y, x, false, nullptr, nullptr, S(stream));
}

// ---- LSQR ------------------------------------------------------------------------------------
static int ensure_workspace(gsr_system* s) {
  if (s->sc) return GSR_OK;
  const size_t m = (size_t)(m_total(s) > 0 ? m_total(s) : 1), n = (size_t)s->v.n;
  cudaError_t e;
  if ((e = cudaMalloc(&s->u, m * sizeof(double))) != cudaSuccess ||
      (e = cudaMalloc(&s->vv, n * sizeof(double))) != cudaSuccess ||
      (e = cudaMalloc(&s->w, n * sizeof(double))) != cudaSuccess ||
      (e = cudaMalloc(&s->x, n * sizeof(double))) != cudaSuccess ||
      (e = cudaMalloc(&s->g, n * sizeof(double))) != cudaSuccess ||
      (e = cudaMalloc(&s->sc, sizeof(DevScalars))) != cudaSuccess) {
    cudaFree(s->u); cudaFree(s->vv); cudaFree(s->w); cudaFree(s->x); cudaFree(s->g); cudaFree(s->sc);
    s->u = s->vv = s->w = s->x = s->g = nullptr; s->sc = nullptr;
    cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? GSR_ENOMEM : cuda_fail(e, "cudaMalloc workspace");
  }
  return GSR_OK;
}

// D^-1 (internal layout): one pass over A for the squared column norms, then 1/sqrt with the empty-column guard.
static int build_dinv(gsr_system* s, cudaStream_t st) {
  const size_t n = (size_t)s->v.n;
  if (!s->dinv) ALLOC(s->dinv, n * sizeof(double));
  if (!s->vs) ALLOC(s->vs, n * sizeof(double));
  CU(cudaMemsetAsync(s->dinv, 0, n * sizeof(double), st));
  CU(launch_aprod2(s->v, s->side, s->tune, s->num_sms, nullptr, s->dinv, true, nullptr, nullptr, st, &s->launches, 1));
  if (s->has_con)
    CU(launch_aprod2(s->con, s->con_side, s->tune, s->num_sms, nullptr, s->dinv, true, nullptr, nullptr, st, &s->launches, 1));
  CU(lsqr_launch_colnorm_finish(s->dinv, s->v.n, 1, st, &s->launches));
  return GSR_OK;
}

static int lsqr_init_with(gsr_system* s, const double* b, bool precond, bool want_var, void* stream);
static int lsqr_run(gsr_system* s, const double* b, double* x, double* var, int32_t flags, int64_t itnlim, double atol,
                    double btol, double conlim, gsr_lsqr_result* res, void* stream, bool with_cov);

extern "C" int gsr_lsqr_init(gsr_system* s, const double* b, void* stream) {
  return lsqr_init_with(s, b, false, false, stream);
}

static int lsqr_init_with(gsr_system* s, const double* b, bool precond, bool want_var, void* stream) {
  if (!s || (!b && m_total(s) > 0)) return GSR_EINVAL;
  if (precond && !fused_path(s)) return GSR_ESTATE;
  int rc = ensure_workspace(s);
  if (rc) return rc;
  s->shard_next = -1;                      // (a sharded solve in progress is void)
  s->opt_precond = precond;
  s->opt_var = want_var;
  if (precond && (rc = build_dinv(s, S(stream)))) return rc;
  if (want_var && !s->var) ALLOC(s->var, (size_t)s->v.n * sizeof(double));
  s->opt_cov = s->opt_cov_next && s->n_cov > 0;
  if (s->opt_cov) CU(cudaMemsetAsync(s->cov, 0, (size_t)s->n_cov * sizeof(double), S(stream)));
  cudaStream_t st = S(stream);
  const int64_t M = m_total(s), n = s->v.n;
  CU(cudaMemsetAsync(s->sc, 0, sizeof(DevScalars), st));
  CU(cudaMemsetAsync(s->vv, 0, (size_t)n * sizeof(double), st));
  CU(lsqr_launch_init_u(b, s->u, M, s->sc, st, &s->launches));           // u_hat = b, usq
  CU(lsqr_launch_init_s1(s->sc, st, &s->launches));                      // beta
  rc = do_aprod2(s, s->u, s->vv, true, &s->sc->s_y, nullptr, st);        // v = A^T u
  if (rc) return rc;
  const double* dinv = s->opt_precond ? s->dinv : nullptr;               // v = (A D^-1)^T u = D^-1 (A^T u)
  CU(lsqr_launch_sumsq_v(s->vv, n, s->sc, dinv, st, &s->launches));
  CU(lsqr_launch_init_s2(s->sc, st, &s->launches));                      // alpha and the rest
  CU(lsqr_launch_init_vw(s->vv, s->w, s->x, n, s->sc, s->opt_precond ? s->vs : nullptr, dinv,
                         s->opt_var ? s->var : nullptr, st, &s->launches));
  s->lsqr_ready = true;
  return GSR_OK;
}

// Issue the launches of n_iters LSQR iterations on st (eagerly, or into a stream capture).
static int issue_iterations(gsr_system* s, int64_t n_iters, int64_t itnlim, double atol, double btol, double conlim,
                            cudaStream_t st) {
  const int64_t n = s->v.n;
  DevScalars* sc = s->sc;
  const double* dinv = s->opt_precond ? s->dinv : nullptr;
  double* vs = s->opt_precond ? s->vs : nullptr;          // the matrix pass gathers D^-1 v
  double* var = s->opt_var ? s->var : nullptr;
  const bool fused = fused_path(s);
  for (int64_t it = 0; it < n_iters && fused; ++it) {
    // 1+2 in one pass over A: u_hat <- A v - (alpha/beta) u_hat ; usq = ||u_hat||^2 ; g = A^T u_hat
    CU(cudaMemsetAsync(s->g, 0, (size_t)n * sizeof(double), st));
    EventPair ep;
    const bool p = prof_begin(s, 3, st, &ep);
    cudaError_t e = launch_lsqr_fused(s->v, s->side, s->tune, s->num_sms, vs ? vs : s->vv, s->u, s->g, &sc->c0_u,
                                      &sc->usq, &sc->done, st, &s->launches);
    if (e == cudaSuccess && s->has_con)   // the constraint section: same pass, rows M .. (done: 2 -> 1 latched by the first)
      e = launch_lsqr_fused(s->con, s->con_side, s->tune, s->num_sms, vs ? vs : s->vv, s->u + s->v.M, s->g, &sc->c0_u,
                            &sc->usq, &sc->done, st, &s->launches);
    if (p) prof_end(s, st, &ep);
    if (e != cudaSuccess) return cuda_fail(e, "fused LSQR pass launch");
    // beta ; v <- g / beta - beta v ; vsq = ||v||^2
    CU(lsqr_launch_vcombine(s->vv, s->g, n, sc, dinv, st, &s->launches));
    // 3-8: scalars, stopping rule ; then the x / w / v update
    CU(lsqr_launch_step_scalars(sc, itnlim, atol, btol, conlim, st, &s->launches));
    if (s->opt_cov) CU(lsqr_launch_cov_update(s->v, s->w, sc, s->cov_j1, s->cov_j2, s->n_cov, s->cov, st, &s->launches));
    CU(lsqr_launch_update(s->vv, s->w, s->x, n, sc, vs, dinv, var, st, &s->launches));
  }
  for (int64_t it = 0; it < n_iters && !fused; ++it) {
    // 1: u_hat <- A v - (alpha/beta) u_hat ; usq = ||u_hat||^2              (aprod 1)
    int rc = do_aprod1(s, s->vv, true, s->u, &sc->c0_u, &sc->usq, &sc->done, st);
    if (rc) return rc;
    // 2: beta ; v <- -beta v ; v += A^T (u_hat / beta) ; vsq = ||v||^2      (aprod 2)
    CU(lsqr_launch_vscale(s->vv, n, sc, st, &s->launches));
    rc = do_aprod2(s, s->u, s->vv, true, &sc->s_y, &sc->done, st);
    if (rc) return rc;
    CU(lsqr_launch_sumsq_v(s->vv, n, sc, nullptr, st, &s->launches));
    // 3-8: scalars, stopping rule ; then the x / w / v update
    CU(lsqr_launch_step_scalars(sc, itnlim, atol, btol, conlim, st, &s->launches));
    if (s->opt_cov) CU(lsqr_launch_cov_update(s->v, s->w, sc, s->cov_j1, s->cov_j2, s->n_cov, s->cov, st, &s->launches));
    CU(lsqr_launch_update(s->vv, s->w, s->x, n, sc, nullptr, nullptr, var, st, &s->launches));
  }
  return GSR_OK;
}

// Small systems are launch-bound: one iteration is a memset and 4-5 kernels, ~39 us at C1 of which the matrix
// pass is 15 us.  There the launches of a batch of iterations are captured once into a CUDA graph and replayed
// (the kernels read every iteration-dependent scalar from device memory, so the graph never changes).  The
// key holds everything that is baked into the captured launches.
struct IterGraph {
  cudaGraphExec_t exec = nullptr;
  int64_t n_iters = 0, itnlim = 0, launches = 0, n_cov = 0;
  double atol = 0, btol = 0, conlim = 0;
  int fused = 0, warps = 0, stages = 0, acc_smem = 0, gather_smem = 0, die_local = 0, instr_copies = 0, ctas = 0;
  int a1v = 0, a2v = 0, tabp = 0, accp = 0, accpf = 0, detc = 0;
  bool precond = false, var = false, cov = false;
  const void *j1 = nullptr, *j2 = nullptr, *covp = nullptr;
};
static bool same_key(const IterGraph& a, const IterGraph& b) {
  return a.n_iters == b.n_iters && a.itnlim == b.itnlim && a.atol == b.atol && a.btol == b.btol && a.conlim == b.conlim &&
         a.fused == b.fused && a.warps == b.warps && a.stages == b.stages && a.acc_smem == b.acc_smem &&
         a.gather_smem == b.gather_smem && a.die_local == b.die_local && a.instr_copies == b.instr_copies &&
         a.ctas == b.ctas && a.a1v == b.a1v && a.a2v == b.a2v && a.tabp == b.tabp && a.accp == b.accp && a.accpf == b.accpf && a.detc == b.detc && a.precond == b.precond && a.var == b.var &&
         a.cov == b.cov && a.n_cov == b.n_cov && a.j1 == b.j1 && a.j2 == b.j2 && a.covp == b.covp;
}

static void free_iter_graph(gsr_system* s) {
  if (s->iter_graph) {
    if (s->iter_graph->exec) cudaGraphExecDestroy(s->iter_graph->exec);
    delete s->iter_graph;
    s->iter_graph = nullptr;
  }
  if (s->cap_stream) { cudaStreamDestroy(s->cap_stream); s->cap_stream = nullptr; }
}

// a batch of n_iters iterations is replayed as a CUDA graph (small, launch-bound systems only)
static bool graph_path(const gsr_system* s, int64_t n_iters) {
  const bool small = (double)m_total(s) * 224.0 <= 256.0 * 1024 * 1024;
  return s->tune.graph && !s->profile && n_iters >= 2 && small;
}

extern "C" int gsr_lsqr_iterate(gsr_system* s, int64_t n_iters, int64_t itnlim, double atol, double btol,
                                double conlim, void* stream) {
  if (!s || n_iters < 0 || itnlim < 0 || !(atol >= 0) || !(btol >= 0) || !(conlim >= 0)) return GSR_EINVAL;
  if (!s->lsqr_ready) return GSR_ESTATE;
  if (s->shard_next >= 0) return GSR_ESTATE;                 // a sharded solve advances through gsr_shard_phase only
  if (s->opt_precond && !fused_path(s)) return GSR_ESTATE;   // the preconditioned operator exists on the fused path only
  cudaStream_t st = S(stream);
  if (!graph_path(s, n_iters)) return issue_iterations(s, n_iters, itnlim, atol, btol, conlim, st);
  IterGraph key;
  key.n_iters = n_iters; key.itnlim = itnlim; key.atol = atol; key.btol = btol; key.conlim = conlim;
  key.fused = s->tune.fused; key.warps = s->tune.warps; key.stages = s->tune.stages; key.acc_smem = s->tune.acc_smem;
  key.gather_smem = s->tune.gather_smem; key.die_local = s->tune.die_local; key.instr_copies = s->tune.instr_copies;
  key.ctas = s->tune.ctas_per_sm; key.a1v = s->tune.aprod1_variant; key.a2v = s->tune.aprod2_variant; key.tabp = s->tune.tab_private; key.accp = s->tune.acc_part; key.accpf = s->tune.acc_part_fused; key.detc = s->tune.det_chunks;
  key.precond = s->opt_precond; key.var = s->opt_var; key.cov = s->opt_cov; key.n_cov = s->n_cov;
  key.j1 = s->cov_j1; key.j2 = s->cov_j2; key.covp = s->cov;
  IterGraph* g = s->iter_graph;
  if (g && g->exec && same_key(*g, key)) {
    CU(cudaGraphLaunch(g->exec, st));
    s->launches += g->launches;
    return GSR_OK;
  }
  if (!g) g = s->iter_graph = new (std::nothrow) IterGraph();
  if (!g) return GSR_ENOMEM;
  if (g->exec) { cudaGraphExecDestroy(g->exec); g->exec = nullptr; }
  const int64_t before = s->launches;
  // captured on a stream of our own (the caller's may be the legacy default stream, which cannot capture;
  // nothing executes during a capture, so no ordering with st is needed); the graph is launched into st
  if (!s->cap_stream) CU(cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking));
  CU(cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal));
  const int rc = issue_iterations(s, n_iters, itnlim, atol, btol, conlim, s->cap_stream);
  cudaGraph_t graph = nullptr;
  cudaError_t e = cudaStreamEndCapture(s->cap_stream, &graph);
  if (rc != GSR_OK || e != cudaSuccess || !graph) {
    if (graph) cudaGraphDestroy(graph);
    cudaGetLastError();
    s->launches = before;
    if (rc != GSR_OK) return rc;
    return issue_iterations(s, n_iters, itnlim, atol, btol, conlim, st);   // capture refused: run eagerly
  }
  cudaGraphExec_t exec = nullptr;
  e = cudaGraphInstantiate(&exec, graph, 0);
  cudaGraphDestroy(graph);
  if (e != cudaSuccess) {
    cudaGetLastError();
    s->launches = before;
    return issue_iterations(s, n_iters, itnlim, atol, btol, conlim, st);
  }
  *g = key;
  g->exec = exec;
  g->launches = s->launches - before;      // what one replay launches (counted once by the capture itself)
  CU(cudaGraphLaunch(exec, st));
  return GSR_OK;
}

// Copy an LSQR-internal n-vector (attitude block interleaved) to a caller's vector in the API layout.
static int export_nvec(gsr_system* s, const double* src, double* dst, cudaStream_t st) {
  const SysView& v = s->v;
  CU(cudaMemcpyAsync(dst, src, (size_t)v.oA * sizeof(double), cudaMemcpyDeviceToDevice, st));
  CU(launch_att_from_il(v, s->num_sms, src + v.oA, dst + v.oA, st, &s->launches));
  CU(cudaMemcpyAsync(dst + v.oI, src + v.oI, (size_t)(v.n - v.oI) * sizeof(double), cudaMemcpyDeviceToDevice, st));
  return GSR_OK;
}

static int fetch_scalars(gsr_system* s, DevScalars* h, cudaStream_t st) {
  CU(cudaMemcpyAsync(h, s->sc, sizeof(DevScalars), cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  return GSR_OK;
}

static void fill_result(const DevScalars& h, gsr_lsqr_result* res) {
  res->istop = h.istop; res->itn = h.itn;
  res->r1norm = h.rnorm; res->r2norm = h.rnorm;
  res->anorm = h.anorm; res->acond = h.acond; res->arnorm = h.arnorm;
  res->xnorm = h.xnorm; res->bnorm = h.bnorm;
}

extern "C" int gsr_lsqr_result_get(gsr_system* s, double* x_out, gsr_lsqr_result* res, void* stream) {
  if (!s || !res) return GSR_EINVAL;
  if (!s->lsqr_ready) return GSR_ESTATE;
  cudaStream_t st = S(stream);
  int rc;
  if (x_out) {
    const double* src = s->x;
    if (s->opt_precond) {   // x = D^-1 z (g is free between iterations)
      CU(lsqr_launch_scale_by(s->g, s->x, s->dinv, s->v.n, 1, st, &s->launches));
      src = s->g;
    }
    if ((rc = export_nvec(s, src, x_out, st))) return rc;
  }
  DevScalars h;
  rc = fetch_scalars(s, &h, st);
  if (rc) return rc;
  fill_result(h, res);
  return GSR_OK;
}

extern "C" int gsr_lsqr_get_state(gsr_system* s, double* u, double* v, double* w, double* x,
                                  gsr_lsqr_scalars* out, void* stream) {
  if (!s) return GSR_EINVAL;
  if (!s->lsqr_ready) return GSR_ESTATE;
  cudaStream_t st = S(stream);
  int rc;
  if (u && m_total(s) > 0) CU(lsqr_launch_export_u(s->u, u, m_total(s), s->sc, st, &s->launches));
  if (v && (rc = export_nvec(s, s->vv, v, st))) return rc;
  if (w && (rc = export_nvec(s, s->w, w, st))) return rc;
  if (x && (rc = export_nvec(s, s->x, x, st))) return rc;
  DevScalars h;
  rc = fetch_scalars(s, &h, st);
  if (rc) return rc;
  if (out) {
    out->itn = h.itn; out->istop = h.istop;
    out->alpha = h.alpha; out->beta = h.beta; out->rhobar = h.rhobar; out->phibar = h.phibar;
    out->bnorm = h.bnorm; out->rnorm = h.rnorm; out->arnorm = h.arnorm; out->anorm = h.anorm;
    out->acond = h.acond; out->ddnorm = h.ddnorm; out->xnorm = h.xnorm; out->xxnorm = h.xxnorm;
    out->z = h.z; out->cs2 = h.cs2; out->sn2 = h.sn2;
  }
  return GSR_OK;
}

extern "C" int gsr_lsqr(gsr_system* s, const double* b, double* x, int64_t itnlim, double atol,
                        double btol, double conlim, gsr_lsqr_result* res, void* stream) {
  return lsqr_run(s, b, x, nullptr, 0, itnlim, atol, btol, conlim, res, stream, false);
}

extern "C" int gsr_set_cov_pairs(gsr_system* s, const int64_t* j1, const int64_t* j2, int64_t n_pairs, double* cov,
                                 void* stream) {
  if (!s || n_pairs < 0) return GSR_EINVAL;
  if (n_pairs > 0 && (!j1 || !j2 || !cov)) return GSR_EINVAL;
  s->cov_j1 = s->cov_j2 = nullptr; s->cov = nullptr; s->n_cov = 0;
  if (n_pairs == 0) return GSR_OK;
  cudaStream_t st = S(stream);
  int* bad = nullptr;
  int h = 0;
  ALLOC(bad, sizeof(int));
  cudaError_t e = cudaMemsetAsync(bad, 0, sizeof(int), st);
  if (e == cudaSuccess) e = lsqr_launch_check_pairs(j1, j2, n_pairs, s->v.n, bad, st, &s->launches);
  if (e == cudaSuccess) e = cudaMemcpyAsync(&h, bad, sizeof(int), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(bad);
  if (e != cudaSuccess) return cuda_fail(e, "gsr_set_cov_pairs");
  if (h) return GSR_EINVAL;
  s->cov_j1 = j1; s->cov_j2 = j2; s->cov = cov; s->n_cov = n_pairs;
  return GSR_OK;
}

extern "C" int gsr_colnorms(gsr_system* s, double* out, void* stream) {
  if (!s || !out) return GSR_EINVAL;
  int rc = ensure_workspace(s);
  if (rc) return rc;
  cudaStream_t st = S(stream);
  CU(cudaMemsetAsync(s->g, 0, (size_t)s->v.n * sizeof(double), st));
  CU(launch_aprod2(s->v, s->side, s->tune, s->num_sms, nullptr, s->g, true, nullptr, nullptr, st, &s->launches, 1));
  if (s->has_con)
    CU(launch_aprod2(s->con, s->con_side, s->tune, s->num_sms, nullptr, s->g, true, nullptr, nullptr, st, &s->launches, 1));
  CU(lsqr_launch_colnorm_finish(s->g, s->v.n, 0, st, &s->launches));
  return export_nvec(s, s->g, out, st);
}

extern "C" int gsr_lsqr_ex(gsr_system* s, const double* b, double* x, double* var, int32_t flags, int64_t itnlim,
                           double atol, double btol, double conlim, gsr_lsqr_result* res, void* stream) {
  return lsqr_run(s, b, x, var, flags, itnlim, atol, btol, conlim, res, stream, true);
}

static int lsqr_run(gsr_system* s, const double* b, double* x, double* var, int32_t flags, int64_t itnlim, double atol,
                    double btol, double conlim, gsr_lsqr_result* res, void* stream, bool with_cov) {
  if (!s || !x || !res || itnlim < 0 || (flags & ~GSR_PRECOND_COLNORM)) return GSR_EINVAL;
  if ((flags & GSR_PRECOND_COLNORM) && !fused_path(s)) return GSR_ESTATE;
  s->opt_cov_next = with_cov;   // gsr_lsqr_ex accumulates the registered covariance pairs; gsr_lsqr / gsr_lsqr_init do not
  int rc = lsqr_init_with(s, b, (flags & GSR_PRECOND_COLNORM) != 0, var != nullptr, stream);
  s->opt_cov_next = false;
  if (rc) return rc;
  cudaStream_t st = S(stream);
  DevScalars h;
  if ((rc = fetch_scalars(s, &h, st))) return rc;
  if (!h.done && itnlim == 0) {
    h.istop = 7;
    CU(cudaMemcpyAsync(&s->sc->istop, &h.istop, sizeof(int), cudaMemcpyHostToDevice, st));
  }
  int64_t issued = 0;
  while (!h.done && issued < itnlim) {
    int64_t batch = s->tune.check_every > 0 ? s->tune.check_every : 16;
    // On the graph path the batch size is baked into the cached graph, so the last batch stays whole: iterations past
    // itnlim are no-ops on the device (k_step_scalars sets istop = 7 and the stop flag).  Eagerly, issue what is left.
    if (batch > itnlim - issued && !graph_path(s, batch)) batch = itnlim - issued;
    if ((rc = gsr_lsqr_iterate(s, batch, itnlim, atol, btol, conlim, stream))) return rc;
    issued += batch;
    if ((rc = fetch_scalars(s, &h, st))) return rc;   // poll the device-side stop flag
  }
  if (s->opt_cov && s->opt_precond)
    CU(lsqr_launch_cov_unscale(s->v, s->dinv, s->cov_j1, s->cov_j2, s->n_cov, s->cov, st, &s->launches));
  if (var) {   // var_x = D^-2 var_z (g is free between iterations)
    const double* src = s->var;
    if (s->opt_precond) {
      CU(lsqr_launch_scale_by(s->g, s->var, s->dinv, s->v.n, 2, st, &s->launches));
      src = s->g;
    }
    if ((rc = export_nvec(s, src, var, st))) return rc;
  }
  return gsr_lsqr_result_get(s, x, res, stream);
}

// ---- row-sharded LSQR in phases -----------------------------------
// The same kernels as gsr_lsqr_init / gsr_lsqr_iterate, cut where a sum over the ranks is needed.  What travels is
// the replicated tail of g (or v) and the partial sums of squares, through the caller's exchange buffer; the
// astrometric part of every n-vector is non-zero on its owner only and never travels.
enum { SH_INIT_B = 1, SH_INIT_C = 2, SH_INIT_D = 3, SH_ITER_A = 4, SH_ITER_B = 5, SH_ITER_C = 6 };

extern "C" int gsr_shard_exchange_len(const gsr_system* s, int64_t* n_doubles) {
  if (!s || !n_doubles) return GSR_EINVAL;
  *n_doubles = (s->v.n - s->v.oA) + 2;
  return GSR_OK;
}

extern "C" int gsr_shard_begin(gsr_system* s, const double* b, double* xbuf, int32_t counts_shared, int64_t itnlim,
                               double atol, double btol, double conlim, int64_t* xcount, void* stream) {
  if (!s || !xbuf || !xcount || (!b && m_total(s) > 0)) return GSR_EINVAL;
  if (itnlim < 0 || !(atol >= 0) || !(btol >= 0) || !(conlim >= 0)) return GSR_EINVAL;
  if (!fused_path(s)) return GSR_ESTATE;              // the phases are those of the one-pass schedule
  int rc = ensure_workspace(s);
  if (rc) return rc;
  s->lsqr_ready = false;
  s->opt_precond = s->opt_var = s->opt_cov = false;
  s->shard_xbuf = xbuf;
  s->shard_counts_shared = counts_shared != 0;
  s->shard_itnlim = itnlim; s->shard_atol = atol; s->shard_btol = btol; s->shard_conlim = conlim;
  cudaStream_t st = S(stream);
  const int64_t M = m_total(s), n = s->v.n;
  CU(cudaMemsetAsync(s->sc, 0, sizeof(DevScalars), st));
  CU(cudaMemsetAsync(s->vv, 0, (size_t)n * sizeof(double), st));
  CU(lsqr_launch_init_u(b, s->u, M, s->sc, st, &s->launches));                               // u_hat = b ; partial sum b^2
  CU(lsqr_launch_shard_xfer(nullptr, 0, s->sc, xbuf, SHARD_X_USQ, 0, st, &s->launches));     // -> xbuf[0]
  *xcount = 1;
  s->shard_next = SH_INIT_B;
  return GSR_OK;
}

extern "C" int gsr_shard_phase(gsr_system* s, int64_t* xcount, int32_t* status, void* stream) {
  if (!s || !xcount || !status) return GSR_EINVAL;
  if (s->shard_next < 0) return GSR_ESTATE;
  cudaStream_t st = S(stream);
  DevScalars* sc = s->sc;
  double* xb = s->shard_xbuf;
  const int64_t n = s->v.n, oA = s->v.oA, ns = n - oA;
  const int64_t n_sq = s->shard_counts_shared ? n : oA;     // the replicated tail is counted by one rank only
  int rc;
  *xcount = 0;
  *status = GSR_SHARD_MORE;
  switch (s->shard_next) {
    case SH_INIT_B:   // beta = ||b|| ; v = A^T u (this rank's rows)                        exchange: the tail of v
      CU(lsqr_launch_shard_xfer(nullptr, 0, sc, xb, SHARD_X_USQ, 1, st, &s->launches));
      CU(lsqr_launch_init_s1(sc, st, &s->launches));
      if ((rc = do_aprod2(s, s->u, s->vv, true, &sc->s_y, nullptr, st))) return rc;
      CU(lsqr_launch_shard_xfer(s->vv + oA, ns, sc, xb, SHARD_X_NONE, 0, st, &s->launches));
      *xcount = ns;
      s->shard_next = SH_INIT_C;
      break;
    case SH_INIT_C:   // partial ||v||^2                                                    exchange: one scalar
      CU(lsqr_launch_shard_xfer(s->vv + oA, ns, sc, xb, SHARD_X_NONE, 1, st, &s->launches));
      CU(lsqr_launch_sumsq_v(s->vv, n, sc, nullptr, st, &s->launches, n_sq));
      CU(lsqr_launch_shard_xfer(nullptr, 0, sc, xb, SHARD_X_VSQ, 0, st, &s->launches));
      *xcount = 1;
      s->shard_next = SH_INIT_D;
      break;
    case SH_INIT_D:   // alpha ; v /= alpha ; w = v ; x = 0 ; partial ||w||^2 (travels with the first iteration)
      CU(lsqr_launch_shard_xfer(nullptr, 0, sc, xb, SHARD_X_VSQ, 1, st, &s->launches));
      CU(lsqr_launch_init_s2(sc, st, &s->launches));
      CU(lsqr_launch_init_vw(s->vv, s->w, s->x, n, sc, nullptr, nullptr, nullptr, st, &s->launches, n_sq));
      s->lsqr_ready = true;
      *status = GSR_SHARD_INIT_DONE;
      s->shard_next = SH_ITER_A;
      break;
    case SH_ITER_A: {  // the fused pass over this rank's rows                 exchange: tail of g, sum u^2, sum w^2
      CU(cudaMemsetAsync(s->g, 0, (size_t)n * sizeof(double), st));
      cudaError_t e = launch_lsqr_fused(s->v, s->side, s->tune, s->num_sms, s->vv, s->u, s->g, &sc->c0_u, &sc->usq,
                                        &sc->done, st, &s->launches);
      if (e == cudaSuccess && s->has_con)
        e = launch_lsqr_fused(s->con, s->con_side, s->tune, s->num_sms, s->vv, s->u + s->v.M, s->g, &sc->c0_u, &sc->usq,
                              &sc->done, st, &s->launches);
      if (e != cudaSuccess) return cuda_fail(e, "fused LSQR pass launch");
      CU(lsqr_launch_shard_xfer(s->g + oA, ns, sc, xb, SHARD_X_USQ_WSQ, 0, st, &s->launches));
      *xcount = ns + 2;
      s->shard_next = SH_ITER_B;
      break;
    }
    case SH_ITER_B:   // beta ; v <- g / beta - beta v ; partial ||v||^2                    exchange: one scalar
      CU(lsqr_launch_shard_xfer(s->g + oA, ns, sc, xb, SHARD_X_USQ_WSQ, 1, st, &s->launches));
      CU(lsqr_launch_vcombine(s->vv, s->g, n, sc, nullptr, st, &s->launches, n_sq));
      CU(lsqr_launch_shard_xfer(nullptr, 0, sc, xb, SHARD_X_VSQ, 0, st, &s->launches));
      *xcount = 1;
      s->shard_next = SH_ITER_C;
      break;
    case SH_ITER_C:   // scalars and stopping rule (identical on every rank) ; x, w, v update ; partial ||w||^2
      CU(lsqr_launch_shard_xfer(nullptr, 0, sc, xb, SHARD_X_VSQ, 1, st, &s->launches));
      CU(lsqr_launch_step_scalars(sc, s->shard_itnlim, s->shard_atol, s->shard_btol, s->shard_conlim, st, &s->launches));
      CU(lsqr_launch_update(s->vv, s->w, s->x, n, sc, nullptr, nullptr, nullptr, st, &s->launches, n_sq));
      *status = GSR_SHARD_ITER_DONE;
      s->shard_next = SH_ITER_A;
      break;
    default:
      return GSR_ESTATE;
  }
  return GSR_OK;
}

extern "C" int gsr_shard_poll(gsr_system* s, int32_t* stopped, gsr_lsqr_result* res, void* stream) {
  if (!s || !stopped) return GSR_EINVAL;
  if (s->shard_next < 0 || !s->lsqr_ready) return GSR_ESTATE;
  DevScalars h;
  int rc = fetch_scalars(s, &h, S(stream));
  if (rc) return rc;
  if (!h.done && s->shard_itnlim == 0) { h.done = 1; h.istop = 7; }   // as gsr_lsqr with itnlim = 0: no iteration is allowed
  *stopped = h.done ? 1 : 0;
  if (res) fill_result(h, res);
  return GSR_OK;
}

extern "C" int gsr_lsqr_host(const gsr_layout* L, const double* values_host, const int32_t* indices_host,
                             const double* b_host, double* x_host, int64_t itnlim, double atol, double btol,
                             double conlim, gsr_lsqr_result* res) {
  if (!x_host || !res || check_layout(L)) return GSR_EINVAL;   // (before any size is computed from the layout)
  if (L->n_rows > 0 && (!values_host || !indices_host || !b_host)) return GSR_EINVAL;
  const size_t M = (size_t)L->n_rows;
  const size_t n = (size_t)(5 * L->n_stars + 3 * L->n_knots + L->n_instr + L->n_glob);
  const size_t cpr = (L->flags & GSR_LAYOUT_COEFF23) ? NSLOT - 1 : NSLOT;
  double *dv = nullptr, *db = nullptr, *dx = nullptr;
  int32_t* di = nullptr;
  gsr_system* sys = nullptr;
  cudaStream_t st = nullptr;
  int rc = GSR_OK;
  cudaError_t e;
  auto cleanup = [&]() {
    gsr_destroy(sys);
    cudaFree(dv); cudaFree(di); cudaFree(db); cudaFree(dx);
    if (st) cudaStreamDestroy(st);
  };
  if ((e = cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking)) != cudaSuccess) return cuda_fail(e, "cudaStreamCreate");
  if ((e = cudaMalloc(&dv, (M ? M : 1) * cpr * sizeof(double))) != cudaSuccess ||
      (e = cudaMalloc(&di, (M ? M : 1) * NIDX * sizeof(int32_t))) != cudaSuccess ||
      (e = cudaMalloc(&db, (M ? M : 1) * sizeof(double))) != cudaSuccess ||
      (e = cudaMalloc(&dx, n * sizeof(double))) != cudaSuccess) {
    cleanup();
    cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? GSR_ENOMEM : cuda_fail(e, "cudaMalloc");
  }
  if (M) {
    if ((e = cudaMemcpyAsync(di, indices_host, M * NIDX * sizeof(int32_t), cudaMemcpyHostToDevice, st)) != cudaSuccess ||
        (e = cudaMemcpyAsync(dv, values_host, M * cpr * sizeof(double), cudaMemcpyHostToDevice, st)) != cudaSuccess ||
        (e = cudaMemcpyAsync(db, b_host, M * sizeof(double), cudaMemcpyHostToDevice, st)) != cudaSuccess) {
      cleanup();
      return cuda_fail(e, "cudaMemcpyAsync H2D");
    }
  }
  rc = gsr_create(&sys, L, dv, di, st);
  if (rc == GSR_OK) rc = gsr_lsqr(sys, db, dx, itnlim, atol, btol, conlim, res, st);
  if (rc == GSR_OK) {
    e = cudaMemcpyAsync(x_host, dx, n * sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) rc = cuda_fail(e, "cudaMemcpyAsync D2H");
  }
  cleanup();
  return rc;
}

// ---- diagnostics ---------------------------------------------------------------------------
extern "C" int gsr_launch_count(const gsr_system* s, int64_t* n) {
  if (!s || !n) return GSR_EINVAL;
  *n = s->launches;
  return GSR_OK;
}

extern "C" int gsr_profile(gsr_system* s, int enable) {
  if (!s) return GSR_EINVAL;
  s->profile = enable != 0;
  return GSR_OK;
}

extern "C" int gsr_profile_get(gsr_system* s, int which, double* mean_ms, int64_t* count) {
  if (!s || which < 1 || which > 3) return GSR_EINVAL;
  for (auto& p : s->pending) {
    float ms = 0.f;
    cudaError_t e = cudaEventSynchronize(p.b);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, p.a, p.b);
    if (e != cudaSuccess) return cuda_fail(e, "cudaEventElapsedTime");
    s->prof_ms[p.which] += ms;
    s->prof_n[p.which] += 1;
    s->pool.push_back(p);
  }
  s->pending.clear();
  if (mean_ms) *mean_ms = s->prof_n[which] ? s->prof_ms[which] / (double)s->prof_n[which] : 0.0;
  if (count) *count = s->prof_n[which];
  s->prof_ms[which] = 0.0;
  s->prof_n[which] = 0;
  return GSR_OK;
}

extern "C" int gsr_instr_acc_info(const gsr_system* s, int32_t* info) {
  if (!s || !info) return GSR_EINVAL;
  const InstrAcc& ia = s->side.ins;
  std::vector<int> d(SMID_SLOTS, -1);
  if (ia.sm_die && cudaMemcpy(d.data(), ia.sm_die, SMID_SLOTS * sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess)
    return cuda_fail(cudaGetLastError(), "cudaMemcpy sm_die");
  info[0] = ia.two_dies ? 1 : 0;
  info[1] = ia.copies_per_die;
  info[2] = ia.n_chunks;
  info[3] = info[4] = 0;
  for (int v : d) { if (v == 0) info[3]++; else if (v == 1) info[4]++; }
  return GSR_OK;
}

extern "C" int gsr_set_option(gsr_system* s, const char* name, int64_t value) {
  if (!s || !name) return GSR_EINVAL;
  if (!strcmp(name, "aprod1_variant")) s->tune.aprod1_variant = (int)value;
  else if (!strcmp(name, "aprod2_variant")) s->tune.aprod2_variant = (int)value;
  else if (!strcmp(name, "ctas_per_sm")) s->tune.ctas_per_sm = (int)value;
  else if (!strcmp(name, "warps")) s->tune.warps = (int)value;
  else if (!strcmp(name, "stages")) s->tune.stages = (int)value;
  else if (!strcmp(name, "instr_copies")) s->tune.instr_copies = (int)value;
  else if (!strcmp(name, "acc_smem")) s->tune.acc_smem = (int)value;
  else if (!strcmp(name, "die_local")) s->tune.die_local = (int)value;
  else if (!strcmp(name, "graph")) s->tune.graph = (int)value;
  else if (!strcmp(name, "gather_smem")) s->tune.gather_smem = (int)value;
  else if (!strcmp(name, "det_chunks")) { if (value < 0 || value > 65536) return GSR_EINVAL; s->tune.det_chunks = (int)value; }
  else if (!strcmp(name, "tab_private")) s->tune.tab_private = (int)value;
  else if (!strcmp(name, "acc_part")) s->tune.acc_part = (int)value;
  else if (!strcmp(name, "acc_part_fused")) s->tune.acc_part_fused = (int)value;
  else if (!strcmp(name, "fused")) s->tune.fused = (int)value;
  else if (!strcmp(name, "check_every")) s->tune.check_every = (int)value;
  else return GSR_EINVAL;
  return GSR_OK;
}
