// Keyed LRU cache of hierarchies (NEXT-4; "an LRU cache of solver handles keyed by a
// hash of the sparsity pattern ... on a cache hit the matrix coefficients are updated in place";
// :121, :287 reuse_setup).  A host-side map around amg_setup / amg_resetup_values: the key is a
// 64-bit hash of (n, nnz, rowptr, col, options) computed on the device (one pass over the pattern,
// order-independent sum of mixed words, so no ordering of the atomics matters).
#include <cstring>
#include <list>
#include <mutex>

#include "amg_internal.cuh"

namespace {

__device__ __forceinline__ unsigned long long cache_mix(unsigned long long z) {
  z += 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}

// sum over k of mix(k, a[k]) in wrap-around arithmetic: commutative, so the result is unique
__global__ void k_pattern_hash(int64_t m, const int* __restrict__ a, unsigned long long tag,
                               unsigned long long* __restrict__ out) {
  unsigned long long s = 0;
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < m; k += (int64_t)gridDim.x * blockDim.x)
    s += cache_mix(((unsigned long long)k << 32) ^ (unsigned long long)(unsigned)a[k] ^ tag);
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0 && s != 0) atomicAdd(out, s);
}

struct Entry {
  unsigned long long key;
  int64_t n, nnz;
  amg_handle h;
};

}  // namespace

struct amg_cache_s {
  int capacity = 4;
  std::list<Entry> lru;  // front = most recently used
  std::mutex mu;
  unsigned long long* d_hash = nullptr;
  int64_t hits = 0, misses = 0, evictions = 0;
};

extern "C" {

amg_status amg_cache_create(amg_cache* out, int32_t capacity) {
  if (!out || capacity < 1) return AMG_ERR_INVALID_ARG;
  *out = new amg_cache_s;
  (*out)->capacity = capacity;
  return AMG_OK;
}

amg_status amg_cache_destroy(amg_cache c) {
  if (!c) return AMG_OK;
  for (Entry& e : c->lru) amg_destroy(e.h);
  if (c->d_hash) cudaFree(c->d_hash);
  delete c;
  return AMG_OK;
}

amg_status amg_cache_get(amg_cache c, int64_t n, int64_t nnz, const int32_t* d_rowptr, const int32_t* d_col,
                         const double* d_val, const amg_options* opt, int32_t on_hit, amg_handle* out, int32_t* hit,
                         void* cuda_stream) {
  if (!c || !out || n <= 0 || nnz <= 0 || !d_rowptr || !d_col || !d_val || on_hit < 0 || on_hit > 2)
    return AMG_ERR_INVALID_ARG;
  *out = nullptr;
  std::lock_guard<std::mutex> lk(c->mu);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (!c->d_hash && cudaMalloc(&c->d_hash, sizeof(unsigned long long)) != cudaSuccess) return AMG_ERR_OOM;
  // ---- key: pattern + options ----
  unsigned long long opt_tag = 0x243F6A8885A308D3ULL;
  if (opt) {
    const unsigned char* p = reinterpret_cast<const unsigned char*>(opt);
    const int m = opt->struct_size > 0 && opt->struct_size <= (int)sizeof(amg_options) ? opt->struct_size : 0;
    for (int i = 0; i < m; ++i) opt_tag = (opt_tag ^ p[i]) * 0x100000001B3ULL;
  }
  if (cudaMemsetAsync(c->d_hash, 0, sizeof(unsigned long long), st) != cudaSuccess) return AMG_ERR_CUDA;
  k_pattern_hash<<<296, 256, 0, st>>>(n + 1, d_rowptr, 1ULL, c->d_hash);
  k_pattern_hash<<<592, 256, 0, st>>>(nnz, d_col, 2ULL, c->d_hash);
  unsigned long long key = 0;
  if (cudaMemcpyAsync(&key, c->d_hash, sizeof(key), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaStreamSynchronize(st) != cudaSuccess)
    return AMG_ERR_CUDA;
  key ^= opt_tag + (unsigned long long)n * 0x9E3779B97F4A7C15ULL + (unsigned long long)nnz;
  // ---- hit: move to the front; values updated per on_hit ----
  for (auto it = c->lru.begin(); it != c->lru.end(); ++it) {
    if (it->key != key || it->n != n || it->nnz != nnz) continue;
    c->lru.splice(c->lru.begin(), c->lru, it);
    ++c->hits;
    if (hit) *hit = 1;
    *out = it->h;
    if (on_hit == 0) return AMG_OK;  // reuse_setup: same values, nothing to do
    return amg_resetup_values(it->h, d_val, on_hit == 2 ? 1 : 0, cuda_stream);
  }
  // ---- miss: set up, insert, evict the least recently used beyond the capacity ----
  ++c->misses;
  if (hit) *hit = 0;
  amg_handle h = nullptr;
  const amg_status s = amg_setup(&h, n, nnz, d_rowptr, d_col, d_val, opt, cuda_stream);
  if (s != AMG_OK) return s;
  c->lru.push_front(Entry{key, n, nnz, h});
  while ((int)c->lru.size() > c->capacity) {
    amg_destroy(c->lru.back().h);
    c->lru.pop_back();
    ++c->evictions;
  }
  *out = h;
  return AMG_OK;
}

amg_status amg_cache_stats(amg_cache c, int64_t* entries, int64_t* hits, int64_t* misses, int64_t* evictions) {
  if (!c) return AMG_ERR_INVALID_ARG;
  std::lock_guard<std::mutex> lk(c->mu);
  if (entries) *entries = (int64_t)c->lru.size();
  if (hits) *hits = c->hits;
  if (misses) *misses = c->misses;
  if (evictions) *evictions = c->evictions;
  return AMG_OK;
}

}  // extern "C"
