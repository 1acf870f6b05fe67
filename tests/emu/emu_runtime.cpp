// tests/emu/emu_runtime.cpp -- the host emulator behind tests/emu/cuda_runtime.h (TEST INFRASTRUCTURE ONLY).
//
// A kernel launch runs its blocks one after the other; the threads of a block are OS threads from a pool (one per
// CUDA thread), so __syncthreads / __syncwarp / shuffles / the warp-wide DMMA are real rendezvous and a missing
// barrier in a kernel is a real data race here too (ThreadSanitizer can see it).  "Device" memory is the heap.
#include "cuda_runtime.h"

#include <algorithm>
#include <condition_variable>
#include <cstdio>
#include <map>
#include <mutex>
#include <set>
#include <string>
#include <thread>
#include <tuple>
#include <vector>

#if defined(__SANITIZE_ADDRESS__)
#include <sanitizer/asan_interface.h>
#define EMU_POISON(p, n) ASAN_POISON_MEMORY_REGION((p), (n))
#define EMU_UNPOISON(p, n) ASAN_UNPOISON_MEMORY_REGION((p), (n))
#else
#define EMU_POISON(p, n) ((void)0)
#define EMU_UNPOISON(p, n) ((void)0)
#endif

constexpr size_t SMEM_TOTAL = 228 * 1024;
extern "C" {
alignas(128) char smem_raw[SMEM_TOTAL];
}

namespace emu {

thread_local dim3 t_threadIdx, t_blockIdx, t_blockDim, t_gridDim;
constexpr int NUM_SMS = 3;          // what cudaDeviceGetAttribute reports: persistent kernels launch 3 CTAs
constexpr int MAX_THREADS = 1024;

// A barrier whose party may shrink: a thread that has left the kernel no longer takes part (as on the GPU).
struct Barrier {
  std::mutex m;
  int expected = 0, count = 0;
  std::atomic<unsigned> gen{0};
  void reset(int n) { expected = n; count = 0; }
  void release_locked() { count = 0; gen.fetch_add(1, std::memory_order_release); }
  void arrive_and_wait() {
    unsigned g;
    {
      std::lock_guard<std::mutex> lk(m);
      g = gen.load(std::memory_order_relaxed);
      if (++count >= expected) { release_locked(); return; }
    }
    int spins = 0;
    while (gen.load(std::memory_order_acquire) == g) {
      if (++spins > 64) std::this_thread::yield();
    }
  }
  void drop() {
    std::lock_guard<std::mutex> lk(m);
    --expected;
    if (expected > 0 && count >= expected) release_locked();
  }
};

struct WarpState {
  Barrier bar;
  uint64_t xch[32];
  double ma[32], mb[32];
};

static Barrier g_block_bar;
static WarpState g_warps[MAX_THREADS / 32];
thread_local WarpState* t_warp = nullptr;

// ---- request counting ---------------------------------------------------------------------------------------------
// Every hooked access of a thread is one record (kind, site = source line of the call, occurrence number of that site in
// this thread, address).  The lanes of a warp run the same code, so (site, occurrence) names one warp instruction; at
// the end of a block the records of each warp are grouped by it and the distinct 128-byte lines ("requests") and
// 32-byte sectors of every instruction are added to the totals of the class its addresses fall into.
bool g_counting = false;
struct Rec { unsigned kind, site, epoch, occ; uintptr_t addr; unsigned bytes; };
thread_local unsigned t_epoch = 0;      // warp rendezvous passed by this thread: the same for all lanes of a warp at any point of the code
static std::vector<Rec> g_logs[MAX_THREADS];
static std::map<unsigned long long, unsigned> g_occ[MAX_THREADS];
struct Region { uintptr_t lo, hi; std::string name; };
static std::vector<Region> g_regions;
struct Tot { unsigned long long instr = 0, lanes = 0, lines = 0, sectors = 0; };
static std::map<std::pair<int, std::string>, Tot> g_totals;       // (kind, class) -> totals
static std::mutex g_count_mutex;

void count_access(int kind, const void* addr, unsigned bytes, unsigned site) {
  const uintptr_t a = reinterpret_cast<uintptr_t>(addr);
  if (a >= reinterpret_cast<uintptr_t>(smem_raw) && a < reinterpret_cast<uintptr_t>(smem_raw) + SMEM_TOTAL) return;   // shared memory
  const unsigned tid = t_threadIdx.x;
  const unsigned long long key = ((unsigned long long)t_epoch << 32) | (site * 4u + (unsigned)kind);
  g_logs[tid].push_back(Rec{(unsigned)kind, site, t_epoch, g_occ[tid][key]++, a, bytes});
}
// every emuMalloc block is a region too; blocks of exactly n doubles are n-vectors and are split by parameter block
static unsigned long long g_n_bytes = 0, g_oA = 0, g_oI = 0, g_oG = 0, g_m_bytes = 0;
static std::vector<Region> g_allocs;
static std::string classify(uintptr_t a) {
  for (const Region& r : g_regions)
    if (a >= r.lo && a < r.hi) return r.name;
  for (const Region& r : g_allocs)
    if (a >= r.lo && a < r.hi) {
      const unsigned long long sz = r.hi - r.lo, off = a - r.lo;
      if (sz == g_n_bytes) return off < g_oA ? "n-vector: astrometric block" : off < g_oI ? "n-vector: attitude block"
                                  : off < g_oG ? "n-vector: instrumental block" : "n-vector: global";
      if (sz == g_m_bytes) return "M-vector";
      return "library buffer of " + std::to_string(sz) + " B";
    }
  return "other";
}
void note_alloc(void* p, size_t bytes) {
  std::lock_guard<std::mutex> lk(g_count_mutex);
  g_allocs.push_back(Region{reinterpret_cast<uintptr_t>(p), reinterpret_cast<uintptr_t>(p) + bytes, ""});
}
void note_free(void* p) {
  std::lock_guard<std::mutex> lk(g_count_mutex);
  for (size_t i = 0; i < g_allocs.size(); i++)
    if (g_allocs[i].lo == reinterpret_cast<uintptr_t>(p)) { g_allocs.erase(g_allocs.begin() + i); break; }
}
static void fold_block(unsigned block) {
  std::lock_guard<std::mutex> lk(g_count_mutex);
  for (unsigned w = 0; w * 32 < block; w++) {
    std::map<std::tuple<unsigned, unsigned, unsigned, unsigned>, std::vector<const Rec*>> by_instr;
    for (unsigned l = w * 32; l < std::min(block, w * 32 + 32); l++)
      for (const Rec& r : g_logs[l]) by_instr[{r.kind, r.site, r.epoch, r.occ}].push_back(&r);
    for (auto& [key, recs] : by_instr) {
      std::set<uintptr_t> lines, sectors;
      for (const Rec* r : recs) {
        for (uintptr_t b = r->addr; b < r->addr + r->bytes; b += 8) { lines.insert(b >> 7); sectors.insert(b >> 5); }
      }
      const bool in_row_loop = std::get<0>(key) == 2 || (std::get<1>(key) >> 20) != 0;
      Tot& t = g_totals[{(int)std::get<0>(key), (in_row_loop ? "" : "[outside the row loop] ") + classify(recs[0]->addr)}];
      t.instr += 1; t.lanes += recs.size(); t.lines += lines.size(); t.sectors += sectors.size();
    }
  }
  for (unsigned l = 0; l < block; l++) { g_logs[l].clear(); g_occ[l].clear(); }
}

// ---- thread pool ------------------------------------------------------------------------------------------------
struct Pool {
  std::mutex m;
  std::condition_variable cv_go, cv_done;
  std::vector<std::thread> workers;
  unsigned long long job = 0;
  int n_active = 0, n_done = 0;
  dim3 bidx, bdim, gdim;
  const std::function<void()>* body = nullptr;
  bool quit = false;

  void worker(int tid) {
    unsigned long long seen = 0;
    for (;;) {
      {
        std::unique_lock<std::mutex> lk(m);
        cv_go.wait(lk, [&] { return quit || (job != seen && tid < n_active); });
        if (quit) return;
        seen = job;
      }
      t_threadIdx = dim3{(unsigned)tid, 0, 0};
      t_blockIdx = bidx; t_blockDim = bdim; t_gridDim = gdim;
      t_warp = &g_warps[tid >> 5];
      t_epoch = 0;
      (*body)();
      t_warp->bar.drop();
      g_block_bar.drop();
      {
        std::lock_guard<std::mutex> lk(m);
        if (++n_done == n_active) cv_done.notify_one();
      }
    }
  }
  void ensure(int n) {
    while ((int)workers.size() < n) {
      const int tid = (int)workers.size();
      workers.emplace_back([this, tid] { worker(tid); });
    }
  }
  void run_block(unsigned b, unsigned grid, unsigned block, const std::function<void()>& f) {
    ensure((int)block);
    g_block_bar.reset((int)block);
    for (unsigned w = 0; w * 32 < block; w++) {
      const unsigned left = block - w * 32;
      g_warps[w].bar.reset((int)(left < 32 ? left : 32));
    }
    {
      std::lock_guard<std::mutex> lk(m);
      bidx = dim3{b, 0, 0}; bdim = dim3{block, 1, 1}; gdim = dim3{grid, 1, 1};
      body = &f;
      n_active = (int)block; n_done = 0;
      ++job;
    }
    cv_go.notify_all();
    std::unique_lock<std::mutex> lk(m);
    cv_done.wait(lk, [&] { return n_done == n_active; });
    n_active = 0;      // late wake-ups of idle workers must not pick the finished job up
    if (g_counting) fold_block(block);
  }
  ~Pool() {
    {
      std::lock_guard<std::mutex> lk(m);
      quit = true;
    }
    cv_go.notify_all();
    for (auto& t : workers) t.join();
  }
};
static Pool& pool() {
  static Pool* p = new Pool();      // leaked on purpose: no destructor races at interpreter exit
  return *p;
}

}  // namespace emu

// ---- streams, capture, graphs --------------------------------------------------------------------------------------
struct emuGraph { std::vector<std::function<void()>> ops; };
struct emuStream { emuGraph* capturing = nullptr; };
struct emuEvent { std::chrono::steady_clock::time_point t; };
static emuStream g_default_stream;
static emuStream* S(cudaStream_t st) { return st ? st : &g_default_stream; }
static void submit(cudaStream_t st, std::function<void()> op) {
  emuStream* s = S(st);
  if (s->capturing) s->capturing->ops.push_back(std::move(op));
  else op();
}

namespace emu {

void launch(unsigned grid, unsigned block, size_t smem_bytes, void* stream, std::function<void()> body) {
  if (grid == 0 || block == 0 || block > (unsigned)MAX_THREADS || smem_bytes > SMEM_TOTAL) {
    std::fprintf(stderr, "emu::launch: bad configuration grid %u block %u smem %zu\n", grid, block, smem_bytes);
    std::abort();
  }
  submit(static_cast<cudaStream_t>(stream), [=] {
    EMU_UNPOISON(smem_raw, SMEM_TOTAL);
    EMU_POISON(smem_raw + smem_bytes, SMEM_TOTAL - smem_bytes);     // only the requested dynamic shared memory exists
    for (unsigned b = 0; b < grid; b++) pool().run_block(b, grid, block, body);
    EMU_UNPOISON(smem_raw, SMEM_TOTAL);
  });
}

void syncthreads() { g_block_bar.arrive_and_wait(); }
void syncwarp() { ++t_epoch; t_warp->bar.arrive_and_wait(); }

uint64_t shfl(uint64_t v, int src_lane) {
  WarpState* w = t_warp;
  ++t_epoch;
  w->xch[t_threadIdx.x & 31] = v;
  w->bar.arrive_and_wait();
  const uint64_t r = w->xch[src_lane];
  w->bar.arrive_and_wait();
  return r;
}

// mma.sync.aligned.m8n8k4.row.col.f64: A is 8x4 (lane l holds A[l>>2][l&3]), B is 4x8 (lane l holds B[l&3][l>>2]),
// C/D is 8x8 (lane l holds C[l>>2][2*(l&3)] and C[l>>2][2*(l&3)+1]); fp64 FMAs over k.
void dmma884(double& c0, double& c1, double a, double b) {
  WarpState* w = t_warp;
  const int lane = (int)(t_threadIdx.x & 31);
  ++t_epoch;
  w->ma[lane] = a;
  w->mb[lane] = b;
  w->bar.arrive_and_wait();
  const int row = lane >> 2, col = 2 * (lane & 3);
  for (int k = 0; k < 4; k++) {
    const double av = w->ma[row * 4 + k];
    c0 = std::fma(av, w->mb[col * 4 + k], c0);
    c1 = std::fma(av, w->mb[(col + 1) * 4 + k], c1);
  }
  w->bar.arrive_and_wait();
}

unsigned smid() { return t_blockIdx.x % (unsigned)NUM_SMS; }

// cp.async.bulk.tensor.2d of an fp64 tensor encoded by the stand-in cuTensorMapEncodeTiled below: the box is written
// row by row, out-of-bounds elements as zeros (CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE fills with zeros).
void tensor_load_2d(void* dst, const CUtensorMap* map, int c0, int c1) {
  const double* base = reinterpret_cast<const double*>(map->opaque[0]);
  const long long d0 = (long long)map->opaque[1], d1 = (long long)map->opaque[2];
  const long long pitch = (long long)map->opaque[3] / 8;
  const int b0 = (int)map->opaque[4], b1 = (int)map->opaque[5];
  double* out = static_cast<double*>(dst);
  if (g_counting) {                                   // the in-bounds part of the box, one contiguous run of whole groups
    const long long rows = std::max(0LL, std::min((long long)b1, d1 - c1));
    if (rows > 0 && c0 == 0) count_access(2, base + (long long)c1 * pitch, (unsigned)(rows * pitch * 8), 2);
  }
  for (int j = 0; j < b1; j++)
    for (int i = 0; i < b0; i++) {
      const long long c = c0 + i, r = (long long)c1 + j;
      out[(size_t)j * b0 + i] = (c >= 0 && c < d0 && r >= 0 && r < d1) ? base[r * pitch + c] : 0.0;
    }
}
void bulk_copy(void* dst, const void* src, uint32_t bytes) {
  if (g_counting) count_access(2, src, bytes, 1);
  std::memcpy(dst, src, bytes);
}

}  // namespace emu

// ---- runtime API ------------------------------------------------------------------------------------------------------
cudaError_t emuMalloc(void** p, size_t bytes) {
  // exact-size heap blocks (AddressSanitizer then sees every out-of-bounds access of a kernel), 256-byte aligned
  void* q = nullptr;
  if (posix_memalign(&q, 256, bytes ? bytes : 1) != 0) { *p = nullptr; return cudaErrorMemoryAllocation; }
  std::memset(q, 0xCD, bytes);        // fresh device memory is not zero
  *p = q;
  emu::note_alloc(q, bytes);
  return cudaSuccess;
}
cudaError_t cudaFree(void* p) {
  if (p) emu::note_free(p);
  std::free(p);
  return cudaSuccess;
}
cudaError_t cudaMemset(void* p, int v, size_t bytes) { std::memset(p, v, bytes); return cudaSuccess; }
cudaError_t cudaMemsetAsync(void* p, int v, size_t bytes, cudaStream_t st) {
  submit(st, [=] { std::memset(p, v, bytes); });
  return cudaSuccess;
}
cudaError_t cudaMemcpy(void* dst, const void* src, size_t bytes, cudaMemcpyKind) { std::memmove(dst, src, bytes); return cudaSuccess; }
cudaError_t cudaMemcpyAsync(void* dst, const void* src, size_t bytes, cudaMemcpyKind, cudaStream_t st) {
  submit(st, [=] { std::memmove(dst, src, bytes); });
  return cudaSuccess;
}
cudaError_t cudaGetLastError() { return cudaSuccess; }
const char* cudaGetErrorString(cudaError_t e) { return e == cudaSuccess ? "no error (host emulation)" : "error (host emulation)"; }
cudaError_t cudaGetDevice(int* dev) { *dev = 0; return cudaSuccess; }
cudaError_t cudaDeviceGetAttribute(int* v, int attr, int) {
  *v = attr == cudaDevAttrMultiProcessorCount ? emu::NUM_SMS : 0;
  return cudaSuccess;
}
cudaError_t cudaStreamCreateWithFlags(cudaStream_t* st, unsigned) { *st = new emuStream(); return cudaSuccess; }
cudaError_t cudaStreamDestroy(cudaStream_t st) { delete st; return cudaSuccess; }
cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
cudaError_t cudaStreamBeginCapture(cudaStream_t st, cudaStreamCaptureMode) {
  emuStream* s = S(st);
  if (s->capturing) return cudaErrorUnknown;
  s->capturing = new emuGraph();
  return cudaSuccess;
}
cudaError_t cudaStreamEndCapture(cudaStream_t st, cudaGraph_t* graph) {
  emuStream* s = S(st);
  *graph = s->capturing;
  s->capturing = nullptr;
  return *graph ? cudaSuccess : cudaErrorUnknown;
}
cudaError_t cudaGraphInstantiate(cudaGraphExec_t* exec, cudaGraph_t graph, unsigned long long) {
  *exec = new emuGraph(*graph);
  return cudaSuccess;
}
cudaError_t cudaGraphLaunch(cudaGraphExec_t exec, cudaStream_t st) {
  for (auto& op : exec->ops) submit(st, op);
  return cudaSuccess;
}
cudaError_t cudaGraphDestroy(cudaGraph_t g) { delete g; return cudaSuccess; }
cudaError_t cudaGraphExecDestroy(cudaGraphExec_t g) { delete g; return cudaSuccess; }
cudaError_t cudaEventCreate(cudaEvent_t* e) { *e = new emuEvent(); return cudaSuccess; }
cudaError_t cudaEventDestroy(cudaEvent_t e) { delete e; return cudaSuccess; }
cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t) { e->t = std::chrono::steady_clock::now(); return cudaSuccess; }
cudaError_t cudaEventSynchronize(cudaEvent_t) { return cudaSuccess; }
cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t a, cudaEvent_t b) {
  *ms = std::chrono::duration<float, std::milli>(b->t - a->t).count();
  return cudaSuccess;
}

// cuTensorMapEncodeTiled stand-in: keeps what tensor_load_2d needs (rank 2, fp64, no swizzle / interleave)
static CUresult emu_encode_tiled(CUtensorMap* map, CUtensorMapDataType dt, cuuint32_t rank, void* base, const cuuint64_t* dims,
                                 const cuuint64_t* strides, const cuuint32_t* box, const cuuint32_t* estr,
                                 CUtensorMapInterleave il, CUtensorMapSwizzle sw, CUtensorMapL2promotion, CUtensorMapFloatOOBfill) {
  // the checks of the real encoder that matter for this library's views
  if (dt != CU_TENSOR_MAP_DATA_TYPE_FLOAT64 || rank != 2 || il != CU_TENSOR_MAP_INTERLEAVE_NONE || sw != CU_TENSOR_MAP_SWIZZLE_NONE)
    return 1;
  if (reinterpret_cast<uintptr_t>(base) % 16 || strides[0] % 16 || box[0] > 256 || box[1] > 256 || estr[0] != 1 || estr[1] != 1)
    return 1;
  if (dims[0] == 0 || dims[1] == 0 || (box[0] * 8) % 16) return 1;
  std::memset(map, 0, sizeof(*map));
  map->opaque[0] = reinterpret_cast<unsigned long long>(base);
  map->opaque[1] = dims[0];
  map->opaque[2] = dims[1];
  map->opaque[3] = strides[0];
  map->opaque[4] = box[0];
  map->opaque[5] = box[1];
  return CUDA_SUCCESS;
}
cudaError_t cudaGetDriverEntryPoint(const char* name, void** fn, int, cudaDriverEntryPointQueryResult* res) {
  if (std::strcmp(name, "cuTensorMapEncodeTiled") == 0) {
    *fn = reinterpret_cast<void*>(&emu_encode_tiled);
    *res = cudaDriverEntryPointSuccess;
    return cudaSuccess;
  }
  *fn = nullptr;
  *res = cudaDriverEntryPointSymbolNotFound;
  return cudaSuccess;
}

// ---- request counting: control (tests/emu/count_requests.py) -----------------------------------------------------------
extern "C" void emu_count_enable(int on) { emu::g_counting = on != 0; }
extern "C" void emu_count_layout(unsigned long long n_bytes, unsigned long long oA_bytes, unsigned long long oI_bytes,
                                 unsigned long long oG_bytes, unsigned long long m_bytes) {
  emu::g_n_bytes = n_bytes; emu::g_oA = oA_bytes; emu::g_oI = oI_bytes; emu::g_oG = oG_bytes; emu::g_m_bytes = m_bytes;
}
extern "C" void emu_count_reset() { std::lock_guard<std::mutex> lk(emu::g_count_mutex); emu::g_totals.clear(); emu::g_regions.clear(); }
extern "C" void emu_count_region(const char* name, const void* p, unsigned long long bytes) {
  std::lock_guard<std::mutex> lk(emu::g_count_mutex);
  emu::g_regions.push_back(emu::Region{reinterpret_cast<uintptr_t>(p), reinterpret_cast<uintptr_t>(p) + bytes, name});
}
// "kind class instructions lanes lines sectors" per line
extern "C" int emu_count_report(char* out, int cap) {
  std::lock_guard<std::mutex> lk(emu::g_count_mutex);
  std::string s;
  for (auto& [k, t] : emu::g_totals)
    s += std::to_string(k.first) + " " + k.second + " " + std::to_string(t.instr) + " " + std::to_string(t.lanes) + " " +
         std::to_string(t.lines) + " " + std::to_string(t.sectors) + "\n";
  if ((int)s.size() + 1 > cap) return -(int)s.size() - 1;
  std::memcpy(out, s.c_str(), s.size() + 1);
  return (int)s.size();
}
