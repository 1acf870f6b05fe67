// tests/emu/cuda_runtime.h -- a HOST stand-in for the CUDA runtime and device intrinsics that csrc/*.cu use, so that
// the kernels' own C++ (everything but their inline PTX, which has host branches under GSR_HOST_EMULATION) can be
// compiled by g++ and run on the CPU with one OS thread per CUDA thread.
//
// TEST INFRASTRUCTURE ONLY.  tests/emu/build_emu.py compiles csrc/*.cu against this header into
// tests/emu/libgsr_emu.so, which only tests/test_emulated_kernels.py loads.  The product (paper_2503_22863_b200/)
// never loads it and has no CPU fallback.  It exists because the code paths added in round 2 could not run on
// hardware (the GPU pool was closed): here they run against the CPU oracle, under AddressSanitizer if wanted
// (device buffers are heap blocks of their exact size, the unused tail of dynamic shared memory is poisoned).
// What it cannot show: anything about timing, the async proxy, the memory model or the real TMA / tensor-core units.
#pragma once
#include <atomic>
#include <chrono>
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <source_location>

// ---- qualifiers ---------------------------------------------------------------------------------------------
#define __global__
#define __device__
#define __host__
#define __forceinline__ inline __attribute__((always_inline))
#define __restrict__ __restrict
#define __launch_bounds__(...)
#define __grid_constant__
#define __shared__ static            // one block runs at a time, so block-shared statics are plain statics

// ---- vector types -------------------------------------------------------------------------------------------
struct alignas(16) int4 { int x, y, z, w; };
struct alignas(16) double2 { double x, y; };
static inline int4 make_int4(int x, int y, int z, int w) { return int4{x, y, z, w}; }
static inline double2 make_double2(double x, double y) { return double2{x, y}; }
struct dim3 { unsigned x = 1, y = 1, z = 1; };

// ---- the emulator (emu_runtime.cpp) ---------------------------------------------------------------------------
struct CUtensorMap_st { alignas(64) unsigned long long opaque[16]; };
typedef CUtensorMap_st CUtensorMap;
namespace emu {
extern thread_local dim3 t_threadIdx, t_blockIdx, t_blockDim, t_gridDim;
void launch(unsigned grid, unsigned block, size_t smem_bytes, void* stream, std::function<void()> body);
void syncthreads();
void syncwarp();
uint64_t shfl(uint64_t v, int src_lane);          // value held by src_lane of the caller's warp (all 32 lanes call)
void dmma884(double& c0, double& c1, double a, double b);   // mma.sync.m8n8k4.f64 of the caller's warp
unsigned smid();
void tensor_load_2d(void* dst, const CUtensorMap* map, int c0, int c1);
void bulk_copy(void* dst, const void* src, uint32_t bytes);
// request counting (tests/emu/count_requests.py): every hooked global access is logged per thread and grouped per warp
// instruction afterwards.  kind: 0 = read-only gather (__ldg), 1 = fp64 reduction / atomic, 2 = TMA / bulk copy
extern bool g_counting;
void count_access(int kind, const void* addr, unsigned bytes, unsigned site);
// site = source line + (1 << 20) when the access is made by the per-tile device routines (aprod_device.cuh), i.e. inside
// the row loop of a matrix kernel, as opposed to a kernel prologue / epilogue or an n-length kernel
static inline unsigned site_of(const std::source_location& loc) {
  const char* f = loc.file_name();
  const char* e = f;
  while (*e) e++;
  const char tail[] = "aprod_device.cuh";
  const int n = (int)sizeof(tail) - 1;
  bool tile = (e - f) >= n;
  for (int i = 0; tile && i < n; i++) tile = e[i - n] == tail[i];
  return loc.line() + (tile ? (1u << 20) : 0u);
}
}  // namespace emu
#define threadIdx emu::t_threadIdx
#define blockIdx emu::t_blockIdx
#define blockDim emu::t_blockDim
#define gridDim emu::t_gridDim

extern "C" char smem_raw[];          // extern __shared__ char smem_raw[] of the kernels

// ---- device intrinsics ----------------------------------------------------------------------------------------
static inline void __syncthreads() { emu::syncthreads(); }
static inline void __syncwarp(unsigned = 0xffffffffu) { emu::syncwarp(); }
template <class T> static inline T __shfl_sync(unsigned, T v, int src) {
  static_assert(sizeof(T) <= 8, "shfl");
  uint64_t b = 0;
  std::memcpy(&b, &v, sizeof(T));
  b = emu::shfl(b, src & 31);
  T r;
  std::memcpy(&r, &b, sizeof(T));
  return r;
}
template <class T> static inline T __shfl_xor_sync(unsigned m, T v, int lane_mask) {
  return __shfl_sync(m, v, (int)((emu::t_threadIdx.x & 31u) ^ (unsigned)lane_mask));
}
template <class T> static inline T __ldg(const T* p, const std::source_location loc = std::source_location::current()) {
  if (emu::g_counting) emu::count_access(0, p, sizeof(T), emu::site_of(loc));
  return *p;
}
template <class T> static inline T __ldcs(const T* p) { return *p; }
static inline size_t __cvta_generic_to_shared(const void* p) { return reinterpret_cast<size_t>(p); }
static inline long long clock64() {
  return (long long)std::chrono::steady_clock::now().time_since_epoch().count();
}
static inline double atomicAdd(double* p, double v, const std::source_location loc = std::source_location::current()) {
  if (emu::g_counting) emu::count_access(1, p, 8, emu::site_of(loc));
  std::atomic_ref<double> a(*p);
  double old = a.load(std::memory_order_relaxed);
  while (!a.compare_exchange_weak(old, old + v, std::memory_order_relaxed)) {}
  return old;
}
static inline int atomicAdd(int* p, int v) { return __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
static inline int atomicOr(int* p, int v) { return __atomic_fetch_or(p, v, __ATOMIC_RELAXED); }
static inline int atomicAnd(int* p, int v) { return __atomic_fetch_and(p, v, __ATOMIC_RELAXED); }
static inline double __dmul_rn(double a, double b) { return a * b; }   // (built with -ffp-contract=off)
static inline double __dadd_rn(double a, double b) { return a + b; }
using std::fma;
using std::sqrt;
using std::fabs;

// ---- runtime API ------------------------------------------------------------------------------------------------
typedef int cudaError_t;
enum { cudaSuccess = 0, cudaErrorInvalidValue = 1, cudaErrorMemoryAllocation = 2, cudaErrorUnknown = 999 };
typedef struct emuStream* cudaStream_t;
typedef struct emuEvent* cudaEvent_t;
typedef struct emuGraph* cudaGraph_t;
typedef struct emuGraph* cudaGraphExec_t;
enum cudaMemcpyKind { cudaMemcpyHostToHost, cudaMemcpyHostToDevice, cudaMemcpyDeviceToHost, cudaMemcpyDeviceToDevice };
enum { cudaStreamNonBlocking = 1 };
enum cudaStreamCaptureMode { cudaStreamCaptureModeGlobal, cudaStreamCaptureModeThreadLocal, cudaStreamCaptureModeRelaxed };
enum { cudaFuncAttributeMaxDynamicSharedMemorySize = 8 };
enum { cudaDevAttrMultiProcessorCount = 16 };
enum { cudaEnableDefault = 0 };
enum cudaDriverEntryPointQueryResult { cudaDriverEntryPointSuccess = 0, cudaDriverEntryPointSymbolNotFound = 1 };

cudaError_t emuMalloc(void** p, size_t bytes);
template <class T> static inline cudaError_t cudaMalloc(T** p, size_t bytes) { return emuMalloc(reinterpret_cast<void**>(p), bytes); }
cudaError_t cudaFree(void* p);
cudaError_t cudaMemset(void* p, int v, size_t bytes);
cudaError_t cudaMemsetAsync(void* p, int v, size_t bytes, cudaStream_t st);
cudaError_t cudaMemcpy(void* dst, const void* src, size_t bytes, cudaMemcpyKind k);
cudaError_t cudaMemcpyAsync(void* dst, const void* src, size_t bytes, cudaMemcpyKind k, cudaStream_t st);
cudaError_t cudaGetLastError();
const char* cudaGetErrorString(cudaError_t e);
cudaError_t cudaGetDevice(int* dev);
cudaError_t cudaDeviceGetAttribute(int* v, int attr, int dev);
cudaError_t cudaStreamCreateWithFlags(cudaStream_t* st, unsigned flags);
cudaError_t cudaStreamDestroy(cudaStream_t st);
cudaError_t cudaStreamSynchronize(cudaStream_t st);
cudaError_t cudaStreamBeginCapture(cudaStream_t st, cudaStreamCaptureMode mode);
cudaError_t cudaStreamEndCapture(cudaStream_t st, cudaGraph_t* graph);
cudaError_t cudaGraphInstantiate(cudaGraphExec_t* exec, cudaGraph_t graph, unsigned long long flags);
cudaError_t cudaGraphLaunch(cudaGraphExec_t exec, cudaStream_t st);
cudaError_t cudaGraphDestroy(cudaGraph_t g);
cudaError_t cudaGraphExecDestroy(cudaGraphExec_t g);
cudaError_t cudaEventCreate(cudaEvent_t* e);
cudaError_t cudaEventDestroy(cudaEvent_t e);
cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t st);
cudaError_t cudaEventSynchronize(cudaEvent_t e);
cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t a, cudaEvent_t b);
cudaError_t cudaGetDriverEntryPoint(const char* name, void** fn, int flags, cudaDriverEntryPointQueryResult* res);
template <class F> static inline cudaError_t cudaFuncSetAttribute(F, int, int) { return cudaSuccess; }

// ---- driver-API names gsr_api.cu needs for cuTensorMapEncodeTiled ----------------------------------------------------
typedef int CUresult;
enum { CUDA_SUCCESS = 0 };
typedef unsigned int cuuint32_t;
typedef unsigned long long cuuint64_t;
enum CUtensorMapDataType { CU_TENSOR_MAP_DATA_TYPE_FLOAT64 = 9 };
enum CUtensorMapInterleave { CU_TENSOR_MAP_INTERLEAVE_NONE = 0 };
enum CUtensorMapSwizzle { CU_TENSOR_MAP_SWIZZLE_NONE = 0 };
enum CUtensorMapL2promotion { CU_TENSOR_MAP_L2_PROMOTION_L2_256B = 3 };
enum CUtensorMapFloatOOBfill { CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE = 0 };
