// extern "C" entry points of amg_b200 (include/amg_b200.h): argument checks, handle lifetime,
// allocator hook.  All numerical work is in amg_setup.cu / amg_solve.cu.
#include <algorithm>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "amg_internal.cuh"

namespace {

constexpr int AMG_BATCH_MIN = 4;  // fewer right-hand sides than this: a loop of single solves is cheaper

thread_local std::string g_thread_error;

std::mutex g_alloc_mutex;  // guards the three words below (handles copy them at creation)
void* (*g_alloc_fn)(size_t, void*, void*) = nullptr;
void (*g_free_fn)(void*, void*) = nullptr;
void* g_alloc_user = nullptr;

// Every entry point that takes a handle: the handle's device is made current for the call (and
// restored), and the stream is remembered (amg_destroy waits for the last one only).
struct Enter {
  int prev = -1;
  Enter(amg_handle_s* h, void* st, bool has_stream = true) {
    int cur = 0;
    if (cudaGetDevice(&cur) == cudaSuccess && cur != h->device) {
      prev = cur;
      cudaSetDevice(h->device);
    }
    if (has_stream) h->last_stream = (cudaStream_t)st;
  }
  ~Enter() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

}  // namespace

void amg_set_thread_error(const std::string& s) { g_thread_error = s; }

// Library-owned device memory.  A handle uses the allocator that was installed when it was created
// (amg_set_allocator) for its whole life, else the device's default stream-ordered pool.
void* amg_dev_alloc(amg_handle_s* H, size_t bytes, cudaStream_t st) {
  bytes += VEC_PAD * sizeof(double);  // slack for the 16-byte-rounded bulk copies of the row-tile kernels
  void* p = nullptr;
  if (H->alloc_fn) {
    p = H->alloc_fn(bytes, (void*)st, H->alloc_user);
  } else if (cudaMallocAsync(&p, bytes, st) != cudaSuccess) {
    // stream-ordered pool: the setup allocates and frees hundreds of temporaries; cudaMalloc /
    // cudaFree would each synchronise the device and map / unmap memory (hundreds of ms per setup)
    cudaGetLastError();
    p = nullptr;
  }
  if (p) H->allocs.push_back(p);
  return p;
}

static void raw_free(amg_handle_s* H, void* p) {
  if (H->free_fn)
    H->free_fn(p, H->alloc_user);
  else
    cudaFreeAsync(p, H->last_stream);  // stream-ordered after the last work of the handle
}

void amg_dev_free(amg_handle_s* H, void* p) {
  if (!p) return;
  auto it = std::find(H->allocs.rbegin(), H->allocs.rend(), p);
  if (it == H->allocs.rend()) return;  // not ours (e.g. the caller's val array)
  H->allocs.erase(std::next(it).base());
  raw_free(H, p);
}

void amg_free_all(amg_handle_s* H) {
  for (void* p : H->allocs) raw_free(H, p);
  H->allocs.clear();
}

namespace {

amg_status create_handle(amg_handle* out, int64_t n, int64_t nnz, const int32_t* d_rowptr, const int32_t* d_col,
                         const double* d_val, const amg_options* opt, int32_t nagg, const int32_t* const* h_d_aggs,
                         void* cuda_stream) {
  if (!out) return AMG_ERR_INVALID_ARG;
  *out = nullptr;
  if (n <= 0 || nnz <= 0 || !d_rowptr || !d_col || !d_val) {
    amg_set_thread_error("amg_setup: null pointer or empty matrix");
    return AMG_ERR_INVALID_ARG;
  }
  if (n >= (int64_t)1 << 31 || nnz >= (int64_t)1 << 31) {
    amg_set_thread_error("amg_setup: n and nnz must be below 2^31 (int32 indices)");
    return AMG_ERR_UNSUPPORTED;
  }
  amg_options o;
  amg_options_default(&o);
  if (opt) {
    if (opt->struct_size <= 0 || opt->struct_size > (int32_t)sizeof(amg_options)) {
      amg_set_thread_error("amg_setup: bad amg_options.struct_size");
      return AMG_ERR_INVALID_ARG;
    }
    memcpy(&o, opt, (size_t)opt->struct_size);
    o.struct_size = (int32_t)sizeof(amg_options);
  }
  if (o.pre_sweeps < 0 || o.post_sweeps < 0 || o.max_levels < 1 || o.coarse_max_rows < 1 ||
      o.smoother < 0 || o.smoother > 2 || !(o.cheby_ratio > 1.0) || o.pre_sweeps + o.post_sweeps > AMG_MAX_SWEEPS || (o.krylov != 0 && o.krylov != 1) || !(o.strong_beta >= 0.0) ||
      o.symmetric < -1 || o.symmetric > 1 || o.agg_passes < 1 || o.agg_passes > 4 || nagg < 0) {
    amg_set_thread_error("amg_setup: option out of range");
    return AMG_ERR_INVALID_ARG;
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  amg_handle_s* H = new amg_handle_s;
  H->opt = o;
  H->n = n;
  H->nnz = nnz;
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
    amg_set_thread_error(std::string("amg_setup: no CUDA device: ") + cudaGetErrorString(cudaGetLastError()));
    delete H;
    return AMG_ERR_CUDA;
  }
  H->device = dev;
  H->last_stream = st;
  H->sm_count = prop.multiProcessorCount;
  H->l2_bytes = (size_t)prop.l2CacheSize;
  {
    std::lock_guard<std::mutex> lk(g_alloc_mutex);
    H->alloc_fn = g_alloc_fn, H->free_fn = g_free_fn, H->alloc_user = g_alloc_user;
  }
  if (!H->alloc_fn) {  // per device, idempotent: freed blocks stay in the pool, repeated setups reuse them
    cudaMemPool_t pool;
    if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
      uint64_t keep = ~0ULL;
      cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
  }
  amg_configure_kernels();  // per-device function attributes (dynamic shared memory opt-in)

  auto fail = [&](amg_status s) {
    amg_set_thread_error(H->err.empty() ? "amg_setup failed" : H->err);
    cudaStreamSynchronize(st);
    amg_destroy_graphs(H);
    amg_batch_release(H);
    for (auto& e : H->ev)
      if (e) cudaEventDestroy(e);
    if (H->h_ctl) cudaFreeHost(H->h_ctl);
    amg_free_all(H);
    delete H;
    cudaGetLastError();
    return s;
  };

  amg_status s = amg_build_hierarchy(H, d_rowptr, d_col, d_val, nagg, h_d_aggs, st);
  if (s != AMG_OK) return fail(s);

  // Krylov workspace
  auto setup_ws = [&]() -> amg_status {
    const int n0 = H->lv[0].n;
    for (int i = 0; i < 9; ++i) AMG_ALLOC(H, H->kv[i], double, n0, st);
    AMG_ALLOC(H, H->io_tmp, double, n0, st);
    AMG_ALLOC(H, H->io_tmp2, double, n0, st);
    AMG_ALLOC(H, H->io_tmp3, double, n0, st);
    AMG_ALLOC(H, H->ctl, KrylovCtl, 1, st);
    int cap = H->sm_count * 8;
    for (const Level& L : H->lv) cap = std::max(cap, L.nblk);
    cap = std::max(cap, 4096);
    H->partials_cap = cap;
    AMG_ALLOC(H, H->partials, double, 2 * (size_t)cap, st);
    AMG_ALLOC(H, H->counter, unsigned, 1, st);
    AMG_CUDA_TRY(H, cudaMemsetAsync(H->counter, 0, sizeof(unsigned), st));
    AMG_TRY(amg_setup_tail(H, 0, st));
    if (!H->symmetric) AMG_TRY(amg_ensure_transposed(H, st));
    AMG_CUDA_TRY(H, cudaMemsetAsync(H->ctl, 0, sizeof(KrylovCtl), st));
    AMG_CUDA_TRY(H, cudaMallocHost((void**)&H->h_ctl, sizeof(KrylovCtl) * 8));
    for (auto& e : H->ev) AMG_CUDA_TRY(H, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
    return AMG_OK;
  };
  s = setup_ws();
  if (s != AMG_OK) return fail(s);
  *out = H;
  return AMG_OK;
}

}  // namespace

extern "C" {

amg_status amg_options_default(amg_options* o) {
  if (!o) return AMG_ERR_INVALID_ARG;
  memset(o, 0, sizeof(*o));
  o->struct_size = (int32_t)sizeof(amg_options);
  o->krylov = 0;
  o->symmetric = -1;
  o->agg_passes = 1;
  o->pre_sweeps = 2;
  o->post_sweeps = 2;
  o->smoother = 0;
  o->coarse_max_rows = 64;
  o->max_levels = 32;
  o->max_match_rounds = 0;
  o->force_generic = 0;
  o->use_graph = 1;
  o->tail_dense_rows = 2304;
  o->use_pdl = 1;
  o->split_prolong_rows = 800000;
  o->use_while = 1;
  o->omega = 2.0 / 3.0;
  o->strong_beta = 0.25;
  o->coarse_scale = 1.0;
  o->hash_seed = 0;
  o->hierarchy_fp32 = 0;
  o->value_dict = 1;
  o->cheby_ratio = 6.0;
  return AMG_OK;
}

amg_status amg_set_allocator(void* (*alloc_fn)(size_t, void*, void*), void (*free_fn)(void*, void*), void* user) {
  if ((alloc_fn == nullptr) != (free_fn == nullptr)) return AMG_ERR_INVALID_ARG;
  std::lock_guard<std::mutex> lk(g_alloc_mutex);
  g_alloc_fn = alloc_fn;
  g_free_fn = free_fn;
  g_alloc_user = user;
  return AMG_OK;
}

amg_status amg_setup(amg_handle* out, int64_t n, int64_t nnz, const int32_t* d_rowptr, const int32_t* d_col,
                     const double* d_val, const amg_options* opt, void* cuda_stream) {
  return create_handle(out, n, nnz, d_rowptr, d_col, d_val, opt, 0, nullptr, cuda_stream);
}

amg_status amg_setup_with_aggregates(amg_handle* out, int64_t n, int64_t nnz, const int32_t* d_rowptr,
                                     const int32_t* d_col, const double* d_val, const amg_options* opt,
                                     int32_t nagg, const int32_t* const* h_d_aggs, void* cuda_stream) {
  static const int32_t* const none[1] = {nullptr};
  if (nagg < 0 || (nagg > 0 && !h_d_aggs)) {
    if (out) *out = nullptr;
    amg_set_thread_error("amg_setup_with_aggregates: bad aggregate list");
    return AMG_ERR_INVALID_ARG;
  }
  return create_handle(out, n, nnz, d_rowptr, d_col, d_val, opt, nagg, nagg > 0 ? h_d_aggs : none, cuda_stream);
}

// NEXT-1: the paper's cache-hit path -- "matrix coefficients are updated in place
// and the setup is repeated on the new values", the operation its Fig. 3 times
// ("warm resetup-and-solve", :285).  The handle keeps its identity; its hierarchy is rebuilt from
// the stored pattern and the new values, with the matching skipped when the aggregates are kept.
// All memory cycles through the stream-ordered pool, so no device allocation reaches the driver.
amg_status amg_resetup_values(amg_handle h, const double* d_val, int32_t keep_aggregates, void* cuda_stream) {
  if (!h) return AMG_ERR_INVALID_ARG;
  if (!d_val) {
    h->err = "amg_resetup_values: null values";
    return AMG_ERR_INVALID_ARG;
  }
  Enter e(h, cuda_stream);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (keep_aggregates) {
    // warm: values only, on the kept hierarchy (patterns, partitions, blobs' index sections, graphs stay)
    int fallback = 0;
    const amg_status sw = amg_resetup_values_warm(h, d_val, &fallback, st);
    if (sw != AMG_OK || !fallback) return sw;
  }
  cudaStreamSynchronize(st);
  std::vector<const int32_t*> aggs;
  if (keep_aggregates)
    for (size_t l = 0; l + 1 < h->lv.size(); ++l) aggs.push_back(h->lv[l].nat_agg);
  amg_handle fresh = nullptr;
  amg_options o = h->opt;  // symmetric = -1 repeats the device check on the new values
  const amg_status s = create_handle(&fresh, h->n, h->nnz, h->nat_rowptr, h->nat_col, d_val, &o,
                                     keep_aggregates ? (int32_t)aggs.size() : 0,
                                     keep_aggregates ? aggs.data() : nullptr, cuda_stream);
  if (s != AMG_OK) {
    h->err = "amg_resetup_values: " + g_thread_error;  // the old hierarchy stays usable
    return s;
  }
  std::swap(*h, *fresh);  // the caller's handle now owns the new hierarchy
  return amg_destroy(fresh);
}

amg_status amg_destroy(amg_handle h) {
  if (!h) return AMG_OK;
  {
    Enter e(h, nullptr, false);
    cudaStreamSynchronize(h->last_stream);  // the handle runs one call at a time: its last stream is enough
    amg_destroy_graphs(h);
    amg_batch_release(h);
    for (auto& ev : h->ev)
      if (ev) cudaEventDestroy(ev);
    if (h->h_ctl) cudaFreeHost(h->h_ctl);
    amg_free_all(h);
  }
  delete h;
  return AMG_OK;
}

amg_status amg_solve_ex(amg_handle h, const double* d_b, double* d_x, double rtol, int32_t maxit, int32_t krylov,
                        int32_t precond, amg_info* info, void* cuda_stream) {
  if (!h) return AMG_ERR_INVALID_ARG;
  if (!d_b || !d_x || maxit < 0 || !(rtol >= 0.0) || (krylov != 0 && krylov != 1)) {
    h->err = "amg_solve: bad argument";
    return AMG_ERR_INVALID_ARG;
  }
  Enter e(h, cuda_stream);
  return amg_krylov_solve(h, d_b, d_x, rtol, maxit, krylov, precond ? 1 : 0, 0, info, (cudaStream_t)cuda_stream);
}

amg_status amg_solve(amg_handle h, const double* d_b, double* d_x, double rtol, int32_t maxit, amg_info* info,
                     void* cuda_stream) {
  if (!h) return AMG_ERR_INVALID_ARG;
  // PCG needs A = A^T: a nonsymmetric handle solves with BiCGSTAB (the paper's default)
  return amg_solve_ex(h, d_b, d_x, rtol, maxit, h->symmetric ? h->opt.krylov : 1, 1, info, cuda_stream);
}

amg_status amg_solve_transpose(amg_handle h, const double* d_g, double* d_lambda, double rtol, int32_t maxit,
                               amg_info* info, void* cuda_stream) {
  if (!h) return AMG_ERR_INVALID_ARG;
  // symmetric: the transposition is skipped, A lambda = g is solved on the same hierarchy
  if (h->symmetric) return amg_solve(h, d_g, d_lambda, rtol, maxit, info, cuda_stream);
  if (!d_g || !d_lambda || maxit < 0 || !(rtol >= 0.0)) {
    h->err = "amg_solve_transpose: bad argument";
    return AMG_ERR_INVALID_ARG;
  }
  // nonsymmetric: operator A^T, preconditioner B^T (transposed level operators on the same aggregates,
  // same smoother diagonals), right-preconditioned BiCGSTAB
  Enter e(h, cuda_stream);
  AMG_TRY(amg_ensure_transposed(h, (cudaStream_t)cuda_stream));
  return amg_krylov_solve(h, d_g, d_lambda, rtol, maxit, 1, 1, 1, info, (cudaStream_t)cuda_stream);
}

amg_status amg_solve_batched(amg_handle h, int32_t transpose, const double* d_B, double* d_X, int32_t nrhs,
                             int64_t ld, double rtol, int32_t maxit, amg_info* infos, void* cuda_stream) {
  if (!h) return AMG_ERR_INVALID_ARG;
  if (nrhs < 0 || ld < h->n || !d_B || !d_X) {
    h->err = "amg_solve_batched: bad argument";
    return AMG_ERR_INVALID_ARG;
  }
  int32_t s0 = 0;
  if (h->opt.krylov == 0 && h->symmetric && nrhs >= AMG_BATCH_MIN) {
    // NEXT-3: one operator pass serves 8 right-hand sides (PCG + AMG on a symmetric handle; the transposed
    // systems are the same systems).  Chunks of 8; a remainder of fewer than AMG_BATCH_MIN columns is looped.
    Enter e(h, cuda_stream);
    if (amg_batch_prepare(h, (cudaStream_t)cuda_stream)) {
      h->last_launches = 0;
      while (nrhs - s0 >= AMG_BATCH_MIN) {
        const int32_t m = nrhs - s0 < 8 ? nrhs - s0 : 8;
        AMG_TRY(amg_solve_batch_chunk(h, d_B + (size_t)s0 * ld, d_X + (size_t)s0 * ld, m, ld, rtol, maxit,
                                      infos ? infos + s0 : nullptr, (cudaStream_t)cuda_stream));
        s0 += m;
      }
    }
  }
  for (int32_t s = s0; s < nrhs; ++s) {
    amg_info* inf = infos ? infos + s : nullptr;
    amg_status st = transpose ? amg_solve_transpose(h, d_B + (size_t)s * ld, d_X + (size_t)s * ld, rtol, maxit, inf,
                                                    cuda_stream)
                              : amg_solve(h, d_B + (size_t)s * ld, d_X + (size_t)s * ld, rtol, maxit, inf,
                                          cuda_stream);
    if (st != AMG_OK) return st;
  }
  return AMG_OK;
}

amg_status amg_solve_host(amg_handle h, const double* h_b, double* h_x, double rtol, int32_t maxit, amg_info* info,
                          void* cuda_stream) {
  if (!h) return AMG_ERR_INVALID_ARG;
  if (!h_b || !h_x) {
    h->err = "amg_solve_host: null pointer";
    return AMG_ERR_INVALID_ARG;
  }
  Enter e(h, cuda_stream);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t bytes = sizeof(double) * (size_t)h->n;
  AMG_CUDA_TRY(h, cudaMemcpyAsync(h->io_tmp, h_b, bytes, cudaMemcpyHostToDevice, st));
  AMG_TRY(amg_solve(h, h->io_tmp, h->io_tmp2, rtol, maxit, info, cuda_stream));
  AMG_CUDA_TRY(h, cudaMemcpyAsync(h_x, h->io_tmp2, bytes, cudaMemcpyDeviceToHost, st));
  AMG_CUDA_TRY(h, cudaStreamSynchronize(st));
  return AMG_OK;
}

amg_status amg_grad_values(amg_handle h, const double* d_lambda, const double* d_x, int32_t nrhs, int64_t ld,
                           double* d_gA, int32_t accumulate, void* cuda_stream) {
  if (!h) return AMG_ERR_INVALID_ARG;
  if (!d_lambda || !d_x || !d_gA || nrhs < 0 || (nrhs > 1 && ld < h->n)) {
    h->err = "amg_grad_values: bad argument";
    return AMG_ERR_INVALID_ARG;
  }
  Enter e(h, cuda_stream);
  return amg_grad_values_impl(h, d_lambda, d_x, nrhs, ld, d_gA, accumulate, (cudaStream_t)cuda_stream);
}

amg_status amg_apply_preconditioner(amg_handle h, const double* d_r, double* d_z, void* cuda_stream) {
  if (!h) return AMG_ERR_INVALID_ARG;
  if (!d_r || !d_z) return AMG_ERR_INVALID_ARG;
  Enter e(h, cuda_stream);
  return amg_level_op_impl(h, 0, 5, nullptr, d_r, d_z, 1, (cudaStream_t)cuda_stream);
}

amg_status amg_get_num_levels(amg_handle h, int32_t* num_levels) {
  if (!h || !num_levels) return AMG_ERR_INVALID_ARG;
  *num_levels = (int32_t)h->lv.size();
  return AMG_OK;
}

amg_status amg_get_level_info(amg_handle h, int32_t level, int64_t* rows, int64_t* nnz) {
  if (!h || level < 0 || level >= (int32_t)h->lv.size()) return AMG_ERR_INVALID_ARG;
  if (rows) *rows = h->lv[level].n;
  if (nnz) *nnz = h->lv[level].nnz;
  return AMG_OK;
}

amg_status amg_get_aggregates(amg_handle h, int32_t level, int32_t* d_agg_out, void* cuda_stream) {
  if (!h || level < 0 || level >= (int32_t)h->lv.size() - 1 || !d_agg_out) return AMG_ERR_INVALID_ARG;
  Enter e(h, cuda_stream);
  AMG_CUDA_TRY(h, cudaMemcpyAsync(d_agg_out, h->lv[level].nat_agg, sizeof(int) * (size_t)h->lv[level].n,
                                  cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream));
  return AMG_OK;
}

amg_status amg_get_level_csr(amg_handle h, int32_t level, int32_t* d_rowptr, int32_t* d_col, double* d_val,
                             void* cuda_stream) {
  if (!h || level < 0 || level >= (int32_t)h->lv.size() || !d_rowptr || !d_col || !d_val)
    return AMG_ERR_INVALID_ARG;
  Enter e(h, cuda_stream);
  return amg_natural_level_csr(h, level, d_rowptr, d_col, d_val, (cudaStream_t)cuda_stream);
}

amg_status amg_get_setup_stats(amg_handle h, amg_setup_stats* stats) {
  if (!h || !stats) return AMG_ERR_INVALID_ARG;
  *stats = h->stats;
  return AMG_OK;
}

amg_status amg_get_level_path(amg_handle h, int32_t level, int32_t* fast_path) {
  if (!h || level < 0 || level >= (int32_t)h->lv.size() || !fast_path) return AMG_ERR_INVALID_ARG;
  *fast_path = h->lv[level].fast;
  return AMG_OK;
}

amg_status amg_get_algorithmic_bytes(amg_handle h, int32_t which, double* bytes) {
  if (!h || !bytes || which < 0 || (which > 4 && (which < 10 || which > 12))) return AMG_ERR_INVALID_ARG;
  *bytes = amg_algorithmic_bytes(h, which);
  return AMG_OK;
}

amg_status amg_get_last_launches(amg_handle h, int64_t* launches) {
  if (!h || !launches) return AMG_ERR_INVALID_ARG;
  *launches = h->last_launches;
  return AMG_OK;
}

amg_status amg_get_residual_history(amg_handle h, double* h_out, int32_t cap, int32_t* count, void* cuda_stream) {
  if (!h || !count || cap < 0 || (cap > 0 && !h_out)) return AMG_ERR_INVALID_ARG;
  Enter e(h, cuda_stream);
  *count = h->hist_len;
  const int m = h->hist_len < cap ? h->hist_len : cap;
  if (m > 0) {
    cudaStream_t st = (cudaStream_t)cuda_stream;
    AMG_CUDA_TRY(h, cudaMemcpyAsync(h_out, h->hist, sizeof(double) * (size_t)m, cudaMemcpyDeviceToHost, st));
    AMG_CUDA_TRY(h, cudaStreamSynchronize(st));
  }
  return AMG_OK;
}

amg_status amg_write_report(amg_handle h, const char* path, void* cuda_stream) {
  if (!h || !path) return AMG_ERR_INVALID_ARG;
  Enter e(h, cuda_stream);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  std::vector<double> hist((size_t)(h->hist_len > 0 ? h->hist_len : 0));
  if (!hist.empty())
    AMG_CUDA_TRY(h, cudaMemcpyAsync(hist.data(), h->hist, sizeof(double) * hist.size(), cudaMemcpyDeviceToHost, st));
  AMG_CUDA_TRY(h, cudaStreamSynchronize(st));
  FILE* f = fopen(path, "w");
  if (!f) {
    h->err = std::string("amg_write_report: cannot open ") + path;
    return AMG_ERR_INVALID_ARG;
  }
  const amg_options& o = h->opt;
  fprintf(f, "amg_b200 hierarchy report\n");
  fprintf(f, "rows %lld  nonzeros %lld  symmetric %d  levels %d\n", (long long)h->n, (long long)h->nnz, h->symmetric,
          (int)h->lv.size());
  fprintf(f, "options: krylov %d  agg_passes %d  sweeps %d+%d  smoother %d (omega %.6g, cheby_ratio %.6g)  strong_beta %.6g  "
             "coarse_scale %.6g  coarse_max_rows %d  hierarchy_fp32 %d  value_dict %d  tail_dense_rows %d  use_graph %d  use_pdl %d  use_while %d\n",
          o.krylov, o.agg_passes, o.pre_sweeps, o.post_sweeps, o.smoother, o.omega, o.cheby_ratio, o.strong_beta,
          o.coarse_scale, o.coarse_max_rows, o.hierarchy_fp32, o.value_dict, o.tail_dense_rows, o.use_graph, o.use_pdl, o.use_while);
  double sn = 0.0, sz = 0.0;
  fprintf(f, "%5s %12s %14s %9s %7s %6s %8s %12s %11s\n", "level", "rows", "nonzeros", "nnz/row", "rounds", "tiles", "kernels",
          "blob MB", "dict values");
  for (size_t l = 0; l < h->lv.size(); ++l) {
    const Level& L = h->lv[l];
    sn += L.n, sz += L.nnz;
    fprintf(f, "%5d %12d %14d %9.2f %7d %6d %8s %12.2f %11d\n", (int)l, L.n, L.nnz, L.n ? (double)L.nnz / L.n : 0.0,
            L.match_rounds, L.nblk, L.fast ? "row-tile" : "row-vec", L.blob_bytes / 1e6, L.ndict);
  }
  fprintf(f, "grid complexity %.4f  operator complexity %.4f  coarsest dense LU %d x %d  dense tail from level %d\n",
          h->n ? sn / (double)h->n : 0.0, h->nnz ? sz / (double)h->nnz : 0.0, h->nL, h->nL, h->tail_dense_level);
  fprintf(f, "setup ms: total %.3f  aggregation %.3f  galerkin %.3f  renumbering+packing %.3f  lu %.3f  (max rounds %d)\n",
          h->stats.total_ms, h->stats.aggregate_ms, h->stats.galerkin_ms, h->stats.reorder_ms, h->stats.lu_ms,
          h->stats.match_rounds_max);
  fprintf(f, "residual history of the last reporting solve (%d iterations): ||r_k|| / ||b||\n", (int)hist.size());
  for (size_t k = 0; k < hist.size(); ++k) fprintf(f, "%5d %.17g\n", (int)k + 1, hist[k]);
  fclose(f);
  return AMG_OK;
}

amg_status amg_get_symmetric(amg_handle h, int32_t* symmetric) {
  if (!h || !symmetric) return AMG_ERR_INVALID_ARG;
  *symmetric = h->symmetric;
  return AMG_OK;
}

amg_status amg_level_op(amg_handle h, int32_t level, int32_t op, const double* d_in0, const double* d_in1,
                        double* d_out, int32_t reps, void* cuda_stream) {
  if (!h || level < 0 || level >= (int32_t)h->lv.size() || !d_out) return AMG_ERR_INVALID_ARG;
  Enter e(h, cuda_stream);
  return amg_level_op_impl(h, level, op, d_in0, d_in1, d_out, reps, (cudaStream_t)cuda_stream);
}

const char* amg_last_error(amg_handle h) { return h ? h->err.c_str() : g_thread_error.c_str(); }

}  // extern "C"
