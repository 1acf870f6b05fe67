// Device side of the seeded generator (inputs only -- none of the method's arithmetic).
// Same counter-based hash as gaia_synth/host.py: all integer outputs (index records) are
// bit-identical to the host generator; N(0,1) values agree to a few ulp.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -shared -Xcompiler -fPIC device.cu -o libgaia_synth.so
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

constexpr uint64_t GOLD = 0x9E3779B97F4A7C15ull;

__host__ __device__ inline uint64_t mix64(uint64_t z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
__host__ __device__ inline uint64_t key_of(uint64_t seed, uint64_t stream) { return mix64(seed + stream * GOLD); }
__device__ inline uint64_t rnd64(uint64_t key, uint64_t ctr) { return mix64(key + ctr * GOLD); }
__device__ inline int64_t bounded(uint64_t u32, uint64_t n) { return (int64_t)((u32 * n) >> 32); }

__device__ inline void normal_pair(uint64_t key, uint64_t ctr, double* z0, double* z1) {
  const uint64_t h = rnd64(key, ctr);
  const double u1 = ((double)(h >> 32) + 1.0) * 2.3283064365386963e-10;      // (0,1]
  const double u2 = (double)(h & 0xFFFFFFFFull) * 2.3283064365386963e-10;    // [0,1)
  const double rad = sqrt(-2.0 * log(u1));
  double s, c;
  sincos(6.283185307179586 * u2, &s, &c);
  *z0 = rad * c;
  *z1 = rad * s;
}

struct GenParams {
  uint64_t seed;
  int64_t r0, nrows, M_obs, n_constraint, S, K, I;
  int32_t G, obs_per_star, hot, wlen, n_hot;
  const int64_t* star_ptr;   // S+1, or null (uniform obs_per_star)
  const int64_t* hot_starts; // n_hot, or null
  uint32_t hot_thresh;       // HOT_PROB * 2^32
};

// one thread per (row, coefficient pair): 12 threads per row write the values; thread 0 of a row
// also writes the index record
__global__ void __launch_bounds__(256) k_fill_rows(GenParams p, double* __restrict__ vals, int32_t* __restrict__ idx) {
  const uint64_t kv = key_of(p.seed, 1), ka = key_of(p.seed, 2), ki = key_of(p.seed, 3);
  const int64_t total = p.nrows * 12;
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < total; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t lr = t / 12;
    const int q = (int)(t - lr * 12);
    const int64_t r = p.r0 + lr;
    double z0, z1;
    normal_pair(kv, (uint64_t)(r * 12 + q), &z0, &z1);
    const bool constraint = r >= p.M_obs;
    if (constraint) {
      const bool is_att = r < p.M_obs + p.n_constraint / 2;
      const int k0 = 2 * q, k1 = 2 * q + 1;
      z0 = is_att ? ((k0 >= 5 && k0 < 17) ? 1.0 : 0.0) : ((k0 >= 17 && k0 < 23) ? 1.0 : 0.0);
      z1 = is_att ? ((k1 >= 5 && k1 < 17) ? 1.0 : 0.0) : ((k1 >= 17 && k1 < 23) ? 1.0 : 0.0);
    }
    if (q == 11 && p.G == 0) z1 = 0.0;
    reinterpret_cast<double2*>(vals)[lr * 12 + q] = make_double2(z0, z1);
    if (q != 0) continue;
    // ---- index record
    int64_t star;
    if (constraint) star = p.S - 1;
    else if (p.star_ptr == nullptr) star = r / p.obs_per_star;
    else {  // last s with star_ptr[s] <= r
      int64_t lo = 0, hi = p.S;
      while (hi - lo > 1) { const int64_t mid = (lo + hi) >> 1; if (p.star_ptr[mid] <= r) lo = mid; else hi = mid; }
      star = lo;
    }
    if (star > p.S - 1) star = p.S - 1;
    const int64_t span = p.K - 4;
    const uint64_t h1 = rnd64(ka, (uint64_t)(2 * r));
    int64_t att = bounded(h1 >> 32, (uint64_t)span);
    if (p.hot) {
      const uint64_t h2 = rnd64(ka, (uint64_t)(2 * r + 1));
      if ((uint32_t)(h1 & 0xFFFFFFFFull) < p.hot_thresh) {
        const int64_t w = bounded(h2 >> 32, (uint64_t)p.n_hot);
        att = p.hot_starts[w] + bounded(h2 & 0xFFFFFFFFull, (uint64_t)p.wlen);
      }
    }
    int32_t rec[8];
    rec[0] = (int32_t)star;
    rec[1] = (int32_t)att;
    int64_t srt[6];
    for (int s = 0; s < 6; s++) {
      const uint64_t h = rnd64(ki, (uint64_t)(8 * r + s));
      int64_t d = bounded(h >> 32, (uint64_t)(p.I - s));
      for (int j = 0; j < s; j++) d += (d >= srt[j]);
      rec[2 + s] = (int32_t)d;
      int pos = 0;
      for (int j = 0; j < s; j++) pos += (srt[j] < d);
      for (int j = s; j > pos; j--) srt[j] = srt[j - 1];
      srt[pos] = d;
    }
    int4* o = reinterpret_cast<int4*>(idx + lr * 8);
    o[0] = make_int4(rec[0], rec[1], rec[2], rec[3]);
    o[1] = make_int4(rec[4], rec[5], rec[6], rec[7]);
  }
}

// out[i - i0] = scale * N(0,1) for element counters i0 .. i0+count-1 (element e: pair e/2, part e%2)
__global__ void __launch_bounds__(256) k_fill_normal(double* __restrict__ out, int64_t i0, int64_t count,
                                                     uint64_t key, double scale) {
  for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < count; t += (int64_t)gridDim.x * blockDim.x) {
    const int64_t e = i0 + t;
    double z0, z1;
    normal_pair(key, (uint64_t)(e >> 1), &z0, &z1);
    out[t] = scale * ((e & 1) ? z1 : z0);
  }
}

}  // namespace

extern "C" int gs_fill_rows(double* vals, int32_t* idx, uint64_t seed, int64_t r0, int64_t nrows, int64_t M_obs,
                            int64_t n_constraint, int64_t S, int64_t K, int64_t I, int32_t G, int32_t obs_per_star,
                            const int64_t* star_ptr_dev, int32_t hot, const int64_t* hot_starts_dev, int32_t n_hot,
                            int32_t wlen, double hot_prob, void* stream) {
  if (nrows <= 0) return 0;
  GenParams p;
  p.seed = seed; p.r0 = r0; p.nrows = nrows; p.M_obs = M_obs; p.n_constraint = n_constraint;
  p.S = S; p.K = K; p.I = I; p.G = G; p.obs_per_star = obs_per_star; p.hot = hot; p.wlen = wlen; p.n_hot = n_hot;
  p.star_ptr = star_ptr_dev; p.hot_starts = hot_starts_dev;
  p.hot_thresh = (uint32_t)(hot_prob * 4294967296.0);
  int64_t blocks = (nrows * 12 + 255) / 256;
  if (blocks > 148 * 32) blocks = 148 * 32;
  k_fill_rows<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(p, vals, idx);
  return (int)cudaGetLastError();
}

extern "C" int gs_fill_normal(double* out, int64_t i0, int64_t count, uint64_t seed, int32_t stream_id, double scale,
                              void* stream) {
  if (count <= 0) return 0;
  int64_t blocks = (count + 255) / 256;
  if (blocks > 148 * 32) blocks = 148 * 32;
  k_fill_normal<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(out, i0, count, key_of(seed, (uint64_t)stream_id), scale);
  return (int)cudaGetLastError();
}
