// amg_grad_values_noalloc: the batched matrix-value gradient (G2, Eq. 2) for callers that
// must not allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// The existing path (amg_grad_values, amg_solve.cu) interleaves X to XT[column][rhs] in a scratch buffer that
// it allocates on the handle and grows on demand.  This variant keeps that scratch in a file-scope device
// array of a fixed, modest size, needs no handle (the caller passes the sparsity pattern), and calls no
// cudaMalloc / cudaFree / allocating library routine.  Nothing of the existing path is changed; the kernels
// are the same templates (amg_kernels.cuh), instantiated again in this translation unit.
//
// The array is part of the library image: every GPU that loads the library holds its 8 MiB until the process
// exits.  All calls share it and it keeps the last call's contents; the interleave pass overwrites every
// element the gradient pass reads (n * nrhs of them), so nothing has to start at zero.  Two calls that overlap
// on the GPU (different streams, or different host threads on one device) race on it.
#include <mutex>
#include <string>

#include "amg_kernels.cuh"

namespace {

// AMG_NOALLOC_MAX_DOUBLES (include/amg_b200.h): most n * nrhs values of one call; 1 Mi doubles = 8 MiB
static __device__ __align__(256) double g_noalloc_xt[AMG_NOALLOC_MAX_DOUBLES];

// In host code `g_noalloc_xt` is a host-side stand-in, not a device address: the device address is looked up
// once per device, with that device current, and cached.
constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
double* g_scratch[MAX_DEVICES] = {};

amg_status fail(amg_status st, const std::string& msg) {
  amg_set_thread_error(msg);
  return st;
}

amg_status scratch_for_current_device(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(AMG_ERR_CUDA, std::string("amg_grad_values_noalloc: cudaGetDevice: ") + cudaGetErrorString(e));
  if (dev < 0 || dev >= MAX_DEVICES) return fail(AMG_ERR_UNSUPPORTED, "amg_grad_values_noalloc: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_noalloc_xt);  // `dev` is current: its copy of the array
    if (e != cudaSuccess || !p)
      return fail(AMG_ERR_CUDA, std::string("amg_grad_values_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
    g_scratch[dev] = p;
  }
  *out = g_scratch[dev];
  return AMG_OK;
}

}  // namespace

extern "C" AMG_API amg_status amg_grad_values_noalloc(int64_t n, int64_t nnz, const int32_t* d_rowptr,
                                                      const int32_t* d_col, const double* d_lambda,
                                                      const double* d_x, int32_t nrhs, int64_t ld, double* d_gA,
                                                      int32_t accumulate, void* cuda_stream) {
  if (!d_rowptr || !d_col || !d_lambda || !d_x || !d_gA) return fail(AMG_ERR_INVALID_ARG, "amg_grad_values_noalloc: null pointer");
  if (n < 0 || nnz < 0 || n > 0x7fffffff || nnz > 0x7fffffff || nrhs < 1 || ld < n)
    return fail(AMG_ERR_INVALID_ARG, "amg_grad_values_noalloc: bad argument (need 0 <= n, nnz < 2^31, nrhs >= 1, ld >= n)");
  const size_t sm = sizeof(double) * (size_t)nrhs * (GT_ROWS + 1);
  if (sm > 48 * 1024)
    return fail(AMG_ERR_UNSUPPORTED, "amg_grad_values_noalloc: nrhs too large (at most 94 right-hand sides per call; accumulate over calls)");
  if (n * (int64_t)nrhs > (int64_t)AMG_NOALLOC_MAX_DOUBLES)
    return fail(AMG_ERR_UNSUPPORTED, "amg_grad_values_noalloc: n * nrhs = " + std::to_string(n * (int64_t)nrhs) +
                                         " exceeds the static scratch of AMG_NOALLOC_MAX_DOUBLES = " +
                                         std::to_string((long long)AMG_NOALLOC_MAX_DOUBLES) +
                                         " values; use amg_grad_values (handle-owned scratch) or fewer right-hand sides per call");
  if (n == 0 || nnz == 0) return AMG_OK;
  double* XT = nullptr;
  const amg_status ss = scratch_for_current_device(&XT);
  if (ss != AMG_OK) return ss;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int ni = (int)n;
  // pass 1: XT[j][s] = X[s * ld + j] (overwrites all n * nrhs values pass 2 reads)
  k_interleave_rhs<<<div_up(ni, GT_ROWS), 256, sm, st>>>(ni, nrhs, ld, d_x, XT);
  // pass 2: one contiguous gather of nrhs values per stored entry, one write of gA
  const double mean = (double)nnz / (double)n;
  const int g8 = div_up((int64_t)n * 8, 256), g32 = div_up((int64_t)n * 32, 256);
  const bool wide = mean > 12.0;
#define AMG_GRAD_CASE(NR)                                                                                            \
  if (wide)                                                                                                         \
    k_grad_values_batched<32, NR><<<g32, 256, 0, st>>>(ni, d_rowptr, d_col, d_lambda, ld, XT, nrhs, d_gA, accumulate); \
  else                                                                                                              \
    k_grad_values_batched<8, NR><<<g8, 256, 0, st>>>(ni, d_rowptr, d_col, d_lambda, ld, XT, nrhs, d_gA, accumulate);
  switch (nrhs) {
    case 2: AMG_GRAD_CASE(2) break;
    case 4: AMG_GRAD_CASE(4) break;
    case 8: AMG_GRAD_CASE(8) break;
    case 16: AMG_GRAD_CASE(16) break;
    default: AMG_GRAD_CASE(0) break;
  }
#undef AMG_GRAD_CASE
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(AMG_ERR_CUDA, std::string("amg_grad_values_noalloc: launch: ") + cudaGetErrorString(e));
  return AMG_OK;
}
