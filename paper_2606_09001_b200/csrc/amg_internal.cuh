// Internal definitions of the amg_b200 library (sm_100a).  Not part of the C ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <vector>

#include "amg_b200.h"

// ------------------------------------------------------------------------------------------
// tuning constants of the row-tile streaming kernels
// ------------------------------------------------------------------------------------------
constexpr int RT_CONSUMERS = 256;     // consumer threads per CTA (8 warps walk the ELL slices)
constexpr int RT_GATHERERS = 192;     // gather threads (6 warps) that assemble the x slots ahead of the row walk
constexpr int RT_GATHER_UNROLL = 4;   // halo columns per gather thread held in registers
constexpr int RT_GGROUPS = 2;         // groups of gather warps working on alternate tiles
constexpr int RT_GATHER_ROWS = 2;     // own rows per gather thread held in registers
constexpr int RT_THREADS = RT_CONSUMERS + 32 + RT_GATHERERS;  // + one producer warp (issues the bulk copies)
constexpr int RT_STAGES = 3;          // tiles in the bulk-async ring of a CTA
constexpr int RT_CTAS = 2;            // persistent CTAs per SM
constexpr int RT_STAGE_BYTES = 29696; // shared memory of one ring stage (descriptor + operands of one tile)
constexpr int RT_XSLOTS = 4;          // x slots (side ring): how many tiles the gather warps run ahead
constexpr int RT_XSLOT_BYTES = 5632;  // one x slot: 8 bytes x (rows + halo columns of a tile)
// Ring geometry of the row-tile kernel per kind of level: 0 = fp64 / fp32 values (the constants above), 1 = levels
// stored as 8-bit codes into a value dictionary (4 bytes per entry: a tile of the same bytes holds ~2 x the rows,
// so the x slots grow and the stages shrink; one more stage keeps as many bytes in flight)
template <int GEO> struct RtGeo;
template <> struct RtGeo<0> {
  static constexpr int STAGES = RT_STAGES, STAGE_BYTES = RT_STAGE_BYTES, XSLOTS = RT_XSLOTS, XSLOT_BYTES = RT_XSLOT_BYTES;
  static constexpr int GATHER_UNROLL = RT_GATHER_UNROLL, GATHER_ROWS = RT_GATHER_ROWS;
  static constexpr int CONSUMERS = RT_CONSUMERS, GATHERERS = RT_GATHERERS, THREADS = RT_THREADS;
};
template <> struct RtGeo<1> {
  static constexpr int STAGES = 4, STAGE_BYTES = 19456, XSLOTS = 4, XSLOT_BYTES = 8192;
  static constexpr int GATHER_UNROLL = 4, GATHER_ROWS = 4;
  static constexpr int CONSUMERS = 256, GATHERERS = 256, THREADS = CONSUMERS + 32 + GATHERERS;  // 8 + 8 warps: the gather bounds these levels
};
template <int GEO> constexpr int rt_smem_bytes() {
  return 256 + RtGeo<GEO>::STAGES * RtGeo<GEO>::STAGE_BYTES + RtGeo<GEO>::XSLOTS * RtGeo<GEO>::XSLOT_BYTES;
}
inline int rt_stage_bytes(int geo) { return geo ? RtGeo<1>::STAGE_BYTES : RtGeo<0>::STAGE_BYTES; }
inline int rt_xslot_bytes(int geo) { return geo ? RtGeo<1>::XSLOT_BYTES : RtGeo<0>::XSLOT_BYTES; }
constexpr int RT_MAX_NNZ = 4096;                   // most entries / halo columns of a tile (packer scratch)
constexpr int RT_MAX_ROWS = 1024;                  // most rows of a tile
constexpr int VEC_PAD = 8;        // every vector / index array is over-allocated by this many elements:
                                  // the bulk copies round their slices out to 16-byte boundaries
constexpr int RB_THREADS = 256;   // row-vector fallback kernels
constexpr int RED_THREADS = 256;  // BLAS-1 kernels
constexpr int AMG_MAX_SWEEPS = 12; // most pre + post sweeps of a cycle
constexpr int MAX_DENSE = 4096;   // largest coarsest level accepted

#include "amg_tilepack.cuh"

// ------------------------------------------------------------------------------------------
// device-resident Krylov scalars and loop control (S7-S9: no host round trip inside the loop)
// ------------------------------------------------------------------------------------------
struct KrylovCtl {
  double rho, rho_new, sigma, alpha, beta, omega;
  double rr, ss, ts, tt, rv;
  double bnorm2, rtol;
  int iter, status, done, maxit;
  int first, halfstep, hist_cap, pad1;
  double* hist;  // [hist_cap] ||r_k|| / ||b|| of iteration k = 1.. (the value its convergence test saw), or null
};

enum FinalizeId {
  FIN_NONE = 0,
  FIN_INIT_PCG,    // sum0 = ||b||^2
  FIN_INIT_BICG,   // sum0 = ||b||^2
  FIN_RZ,          // sum0 = r.z          -> beta, rho
  FIN_PQ,          // sum0 = p.q          -> alpha (or breakdown)
  FIN_RR,          // sum0 = ||r||^2      -> iter++, convergence
  FIN_RV,          // sum0 = rhat.v       -> alpha (or breakdown)
  FIN_SS,          // sum0 = ||s||^2      -> iter++, half-step convergence
  FIN_TS_TT,       // sum0 = t.s, sum1 = t.t -> omega
  FIN_RR_RHO,      // sum0 = ||r||^2, sum1 = rhat.r -> convergence, beta, rho
};

// ------------------------------------------------------------------------------------------
// one level of the hierarchy, stored in aggregate-contiguous ("permuted") numbering
// ------------------------------------------------------------------------------------------
// transposed operator A_l^T of a level (nonsymmetric adjoint): same rows, same
// aggregates, same permuted numbering, its own tile partition and blobs
struct LevelOpT {
  int* rowptr = nullptr;
  int* col = nullptr;
  double* val = nullptr;
  int* src = nullptr;       // [nnz] position in the level's own val[] every entry came from (value-only resetup)
  int* blk_ptr = nullptr;
  TileDesc* tiles = nullptr;
  unsigned char* blob = nullptr;
  int* halo_idx = nullptr;
  int* halo_cagg = nullptr;
  size_t blob_bytes = 0;
  int nblk = 0;
  int fast = 0;
};

struct Level {
  int n = 0;        // rows
  int nc = 0;       // rows of the next level (0 on the coarsest)
  int nnz = 0;
  int nnz_alloc = 0;  // padded to a multiple of 4 (+4) for 128-bit loads
  // operator A_l
  int* rowptr = nullptr;
  int* col = nullptr;
  double* val = nullptr;
  double* dinv = nullptr;   // smoother diagonal (null on the coarsest)
  // diagonal of every sweep of a cycle: pre-sweep s -> dsw[s], post-sweep s -> dsw[nu1 + s].  All equal to dinv unless
  // the smoother is the Chebyshev-accelerated L1-Jacobi (smoother = 2): then tau * dinv with the sweep's weight
  double* dsw[AMG_MAX_SWEEPS] = {nullptr};
  int* agg = nullptr;       // [n]  coarse id of every row, non-decreasing
  int* agg_ptr = nullptr;   // [nc+1] first row of every aggregate
  // row-tile partition (boundaries aligned to aggregate starts)
  int* blk_ptr = nullptr;   // [nblk+1]
  TileDesc* tiles = nullptr;  // [nblk]
  unsigned char* blob = nullptr;  // tile-packed operator (amg_tilepack.cuh), fast levels only
  int* halo_idx = nullptr;        // halo lists of all tiles, concatenated
  int* halo_cagg = nullptr;       // coarse index of every halo entry
  size_t blob_bytes = 0;
  int nblk = 0;
  int fast = 0;             // 1: row-tile streaming kernels; 0: row-vector fallback
  LevelOpT T;               // A_l^T (only when the handle is nonsymmetric)
  // mixed-precision hierarchy: the blobs above (and T's) hold fp32 values; level 0 keeps fp64 blobs of A_0 (K) and
  // A_0^T (KT) for the Krylov method's own SpMV
  LevelOpT K, KT;
  int v32 = 0;              // 1: this level's V-cycle operator is the fp64 one rounded to fp32
  double* vdict = nullptr;  // [256] value dictionary of the level (ascending distinct values, [255] = 0 for padding
  int ndict = 0;            //   slots); ndict > 0: the tile blobs hold 8-bit codes (TileDesc::vb = 1)
  unsigned long long* vd_table = nullptr;  // hash set of the distinct values (kept for warm resetups)
  int* vd_count = nullptr;                 // {distinct values, overflow}
  int lpr = 8;              // lanes per row of the fallback kernels
  int stream_hint = 0;      // 1: matrix larger than half of L2 -> evict-first loads
  // natural numbering (the caller's / oracle's): hooks and the ABI boundary
  int* nat_agg = nullptr;   // [n] aggregate ids in natural numbering of levels l, l+1
  int* pos = nullptr;       // [n] natural index -> permuted position
  int* inv = nullptr;       // [n] permuted position -> natural index
  // work vectors (permuted numbering)
  double* b = nullptr;      // right-hand side of this level (levels > 0)
  double* x = nullptr;      // iterate / ping
  double* x2 = nullptr;     // pong
  double* rtmp = nullptr;   // fine residual (fallback path only)
  int match_rounds = 0;
  // value-only (warm) resetup maps, built on the first amg_resetup_values(keep_aggregates = 1):
  int* src0 = nullptr;         // level 0 only: [nnz] position in the caller's val[] of every permuted entry
  int* contrib_ptr = nullptr;  // [nnz_{l+1} + 1] per entry of A_{l+1}: its fine contributions ...
  int* contrib_idx = nullptr;  // [nnz_l] ... as ascending positions in this level's val[] (fixed summation order)
};

struct AmgBatch;  // batched multi-RHS state (amg_batched.cu)

struct amg_handle_s {
  amg_options opt;
  int64_t n = 0, nnz = 0;
  std::vector<Level> lv;
  // natural level-0 pattern for amg_grad_values
  int* nat_rowptr = nullptr;
  int* nat_col = nullptr;
  // coarsest dense LU (of A_L; luT / pivT: of A_L^T, nonsymmetric handles only)
  int nL = 0;
  double* lu = nullptr;
  int* piv = nullptr;
  double* luT = nullptr;
  int* pivT = nullptr;
  bool have_T = false;
  bool have_maps = false;  // warm-resetup maps built
  // Krylov work vectors (level-0 size, permuted numbering)
  double* kv[10] = {nullptr};
  double* io_tmp = nullptr;  // staging for amg_solve_host / hooks
  double* io_tmp2 = nullptr;
  double* io_tmp3 = nullptr;
  KrylovCtl* ctl = nullptr;       // device
  KrylovCtl* h_ctl = nullptr;     // pinned host mirror
  double* partials = nullptr;     // [2 * partials_cap]
  int partials_cap = 0;
  unsigned* counter = nullptr;
  // coarse tail of the V-cycle: the cycle from level tail_dense_level down is one dense operator (amg_tail.cuh)
  int tail_grid = 0;
  int tail_dense_level = -1;         // -1: off
  double* tail_dense_B = nullptr;
  double* tail_dense_BT = nullptr;   // the same for the transposed hierarchy
  // CUDA graph of one Krylov iteration (keyed by krylov/precond)
  // [krylov * 2 + precond]: one iteration; [4]: the start of an AMG-PCG solve (first V-cycle + p = z)
  // [5]: one BiCGSTAB + AMG iteration on the transposed hierarchy; [6]: one V-cycle (amg_apply_preconditioner)
  cudaGraphExec_t graph_exec[7] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  int64_t graph_launches[7] = {0, 0, 0, 0, 0, 0, 0};  // kernel nodes per replay
  // the Krylov loop as one graph with a conditional WHILE node ([krylov * 2 + precond], [4]: transposed BiCGSTAB)
  cudaGraphExec_t while_exec[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
  int64_t while_launches[5] = {0, 0, 0, 0, 0};  // kernel nodes of the body
  bool while_failed = false, while_used = false;
  double* apply_out = nullptr;               // result buffer of the captured V-cycle
  double* vcycle_final_out = nullptr;        // if set: the last post-sweep of a cycle started at level 0 writes here
  int64_t last_launches = 0;                 // kernels enqueued by the last solve / hook / gradient call
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
  cudaStream_t cap_stream = nullptr;  // graphs are captured here (the legacy stream cannot capture)
  int device = 0;                     // the device the handle lives on
  cudaStream_t last_stream = nullptr; // stream of the last call (amg_destroy waits for it)
  void* (*alloc_fn)(size_t, void*, void*) = nullptr;  // allocator captured at creation (amg_set_allocator)
  void (*free_fn)(void*, void*) = nullptr;
  void* alloc_user = nullptr;
  double* hist = nullptr;             // residual history of the last solve (device), hist_cap entries
  int hist_cap = 0;
  int hist_len = 0;                   // iterations of the last solve that reported (info != NULL)
  AmgBatch* batch = nullptr;          // work vectors / graphs of the batched solve, built on first use
  double* grad_xt = nullptr;          // interleaved right-hand sides of amg_grad_values (grown on demand)
  size_t grad_xt_cap = 0;
  int sm_count = 148;
  size_t l2_bytes = 0;
  int symmetric = 1;
  amg_setup_stats stats{};
  std::vector<void*> allocs;
  std::string err;
};

// ------------------------------------------------------------------------------------------
// host helpers
// ------------------------------------------------------------------------------------------
void amg_set_thread_error(const std::string& s);
void* amg_dev_alloc(amg_handle_s* H, size_t bytes, cudaStream_t st);  // tracked; nullptr on failure
void amg_dev_free(amg_handle_s* H, void* p);                           // early release of a tracked block
void amg_free_all(amg_handle_s* H);

#define AMG_CUDA_TRY(H, expr)                                                              \
  do {                                                                                     \
    cudaError_t _e = (expr);                                                               \
    if (_e != cudaSuccess) {                                                               \
      (H)->err = std::string(#expr) + ": " + cudaGetErrorString(_e);                        \
      return AMG_ERR_CUDA;                                                                 \
    }                                                                                      \
  } while (0)

#define AMG_TRY(expr)                    \
  do {                                   \
    amg_status _s = (expr);              \
    if (_s != AMG_OK) return _s;         \
  } while (0)

#define AMG_ALLOC(H, ptr, type, count, st)                                         \
  do {                                                                             \
    (ptr) = (type*)amg_dev_alloc((H), sizeof(type) * (size_t)(count), (st));        \
    if (!(ptr)) {                                                                  \
      (H)->err = "device allocation failed: " #ptr;                                \
      return AMG_ERR_OOM;                                                          \
    }                                                                              \
  } while (0)

static inline int div_up(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

// setup.cu
amg_status amg_build_hierarchy(amg_handle_s* H, const int32_t* d_rowptr, const int32_t* d_col,
                               const double* d_val, int32_t nagg, const int32_t* const* h_d_aggs,
                               cudaStream_t st);
amg_status amg_natural_level_csr(amg_handle_s* H, int level, int32_t* d_rowptr, int32_t* d_col,
                                 double* d_val, cudaStream_t st);
amg_status amg_exclusive_scan(amg_handle_s* H, const int* d_in, int* d_out, int n, cudaStream_t st);

// solve.cu
amg_status amg_vcycle(amg_handle_s* H, int level, const double* b, double** x_out, KrylovCtl* ctl,
                      bool fuse_rz, cudaStream_t st, bool x1_ready = false);
amg_status amg_krylov_solve(amg_handle_s* H, const double* d_b, double* d_x, double rtol, int maxit,
                            int krylov, int precond, int transposed, amg_info* info, cudaStream_t st);
amg_status amg_level_op_impl(amg_handle_s* H, int level, int op, const double* d_in0,
                             const double* d_in1, double* d_out, int reps, cudaStream_t st);
amg_status amg_grad_values_impl(amg_handle_s* H, const double* d_lambda, const double* d_x, int nrhs,
                                int64_t ld, double* d_gA, int accumulate, cudaStream_t st);
double amg_algorithmic_bytes(amg_handle_s* H, int which);
void amg_destroy_graphs(amg_handle_s* H);
amg_status amg_setup_tail(amg_handle_s* H, int transposed, cudaStream_t st);
void amg_configure_kernels();
// batched.cu (NEXT-3)
int amg_batch_prepare(amg_handle_s* H, cudaStream_t st);
amg_status amg_solve_batch_chunk(amg_handle_s* H, const double* d_B, double* d_X, int ncols, int64_t ld, double rtol,
                                 int maxit, amg_info* infos, cudaStream_t st);
void amg_batch_release(amg_handle_s* H);
// setup.cu: transposed level operators, their tile blobs, LU of A_L^T, dense tail of B^T
amg_status amg_ensure_transposed(amg_handle_s* H, cudaStream_t st);
// setup.cu: NEXT-1 value-only resetup on the kept hierarchy; *fallback = 1: the caller has to rebuild (symmetry changed)
amg_status amg_ensure_src0(amg_handle_s* H, cudaStream_t st);
amg_status amg_build_sweep_diagonals(amg_handle_s* H, cudaStream_t st);  // Level::dsw from Level::dinv
amg_status amg_resetup_values_warm(amg_handle_s* H, const double* d_val, int* fallback, cudaStream_t st);
