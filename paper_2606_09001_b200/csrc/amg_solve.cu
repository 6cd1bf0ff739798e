// Solve-phase host drivers: kernel dispatch, V-cycle (S6), PCG / BiCGSTAB (S7-S9) with the
// iteration replayed as a CUDA graph and the convergence test on the device, per-level hooks,
// gradient (G2), algorithmic byte counts.
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "amg_kernels.cuh"
#include "amg_tail.cuh"

namespace {

thread_local int64_t g_nlaunch = 0;  // kernel launches enqueued by this thread (amg_get_last_launches)

thread_local bool g_pdl = false;     // true while an iteration is being captured with programmatic edges
thread_local cudaGraphConditionalHandle g_loop = 0;  // != 0 while the body of a WHILE node is being captured
thread_local int g_kop = 0;          // 1: the Krylov method's own SpMV (mixed-precision hierarchy: the fp64 blobs of level 0)
thread_local int g_tr = 0;           // 1: the level operators are the transposed ones (A_l^T, nonsymmetric adjoint)

// kernel launch; with g_pdl the kernel may become resident while its predecessor drains
// (programmatic dependent launch: every kernel of the solve calls griddepcontrol.wait first)
template <typename... KArgs>
struct Launcher {
  void (*k)(KArgs...);
  dim3 g, b;
  size_t sm;
  cudaStream_t st;
  template <typename... A>
  void operator()(A&&... a) const {
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = g, cfg.blockDim = b, cfg.dynamicSmemBytes = sm, cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = g_pdl ? 1 : 0;
    cudaLaunchKernelEx(&cfg, k, KArgs(a)...);
  }
};
template <typename... KArgs>
Launcher<KArgs...> launch(void (*k)(KArgs...), dim3 g, dim3 b, size_t sm, cudaStream_t st) {
  return Launcher<KArgs...>{k, g, b, sm, st};
}

constexpr int TPB = 256;
inline int grid_for(int n) { return n > 0 ? div_up(n, TPB) : 1; }

inline int red_grid(const amg_handle_s* H, int n) {
  int g = div_up(n, RED_THREADS * 4);
  int cap = H->sm_count * 8;
  if (g > cap) g = cap;
  if (g > H->partials_cap) g = H->partials_cap;
  return g < 1 ? 1 : g;
}

// ---- dispatch of the row kernels ---------------------------------------------------------
inline const LevelOpT* lv_kop(const Level& L) {  // fp64 blobs for the Krylov SpMV of a mixed-precision hierarchy
  if (!g_kop) return nullptr;
  const LevelOpT* K = g_tr ? &L.KT : &L.K;
  return K->fast ? K : nullptr;
}
inline int lv_fast(const Level& L) {
  if (g_kop && L.v32) return lv_kop(L) != nullptr;  // no fp64 blobs: the row-vector kernels on the fp64 CSR
  return g_tr ? L.T.fast : L.fast;
}
inline int lv_nblk(const Level& L) {
  if (const LevelOpT* K = lv_kop(L)) return K->nblk;
  return g_tr ? L.T.nblk : L.nblk;
}

inline int lv_geo(const Level& L) {  // ring geometry of the blobs about to be streamed (RtGeo)
  return (lv_kop(L) == nullptr && L.ndict > 0) ? 1 : 0;
}
template <int OP, int NDOT, bool STREAM>
void launch_tile(const amg_handle_s* H, const Level& L, const RowArgs& a, cudaStream_t st) {
  int grid = H->sm_count * RT_CTAS;
  if (grid > lv_nblk(L)) grid = lv_nblk(L);
  if (lv_geo(L))
    ++g_nlaunch, launch(k_rowtile<OP, NDOT, STREAM, 1>, grid, RtGeo<1>::THREADS, rt_smem_bytes<1>(), st)(a);
  else
    ++g_nlaunch, launch(k_rowtile<OP, NDOT, STREAM, 0>, grid, RT_THREADS, rt_smem_bytes<0>(), st)(a);
}

template <int OP, int NDOT>
void launch_row(const amg_handle_s* H, const Level& L, const RowArgs& a, cudaStream_t st) {
  if (lv_fast(L)) {
    if (L.stream_hint)
      launch_tile<OP, NDOT, true>(H, L, a, st);
    else
      launch_tile<OP, NDOT, false>(H, L, a, st);
  } else {
    const int64_t threads = (int64_t)L.n * L.lpr;
    int g = div_up(threads, RB_THREADS);
    if (NDOT > 0 && g > 4096) g = 4096;  // bounded partials; the kernel strides over rows
    if (g < 1) g = 1;
    switch (L.lpr) {
      case 4: ++g_nlaunch; launch(k_rowvec<OP, NDOT, 4>, g, RB_THREADS, 0, st)(a); break;
      case 8: ++g_nlaunch; launch(k_rowvec<OP, NDOT, 8>, g, RB_THREADS, 0, st)(a); break;
      case 16: ++g_nlaunch; launch(k_rowvec<OP, NDOT, 16>, g, RB_THREADS, 0, st)(a); break;
      default: ++g_nlaunch; launch(k_rowvec<OP, NDOT, 32>, g, RB_THREADS, 0, st)(a); break;
    }
  }
}

template <int OP, int NDOT>
void set_tile_attr() {
  cudaFuncSetAttribute(k_rowtile<OP, NDOT, true, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, rt_smem_bytes<0>());
  cudaFuncSetAttribute(k_rowtile<OP, NDOT, false, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, rt_smem_bytes<0>());
  cudaFuncSetAttribute(k_rowtile<OP, NDOT, true, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, rt_smem_bytes<1>());
  cudaFuncSetAttribute(k_rowtile<OP, NDOT, false, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, rt_smem_bytes<1>());
}

RowArgs base_args(const amg_handle_s* H, const Level& L, KrylovCtl* ctl) {
  RowArgs a;
  memset(&a, 0, sizeof(a));
  a.n = L.n;
  a.v32 = (L.v32 && !g_kop) ? 1 : 0;
  if (const LevelOpT* K = lv_kop(L)) {
    a.rowptr = g_tr ? L.T.rowptr : L.rowptr, a.col = g_tr ? L.T.col : L.col, a.val = g_tr ? L.T.val : L.val;
    a.tiles = K->tiles, a.ntiles = K->nblk, a.blob = K->blob, a.halo_idx = K->halo_idx, a.halo_cagg = K->halo_cagg;
  } else if (g_tr) {
    a.rowptr = L.T.rowptr, a.col = L.T.col, a.val = L.T.val;
    a.tiles = L.T.tiles, a.ntiles = L.T.nblk, a.blob = L.T.blob;
    a.halo_idx = L.T.halo_idx, a.halo_cagg = L.T.halo_cagg;
  } else {
    a.rowptr = L.rowptr, a.col = L.col, a.val = L.val;
    a.tiles = L.tiles, a.ntiles = L.nblk, a.blob = L.blob;
    a.halo_idx = L.halo_idx, a.halo_cagg = L.halo_cagg;
  }
  a.vdict = L.ndict > 0 ? L.vdict : nullptr;  // (A_l^T holds the same values: the same dictionary)
  a.dinv = L.dinv;
  a.dinv_x1 = L.dinv;
  a.agg = L.agg;
  a.agg_ptr = L.agg_ptr;
  a.gamma = H->opt.coarse_scale;
  a.partials = H->partials;
  a.counter = H->counter;
  a.ctl = ctl;
  a.fin = FIN_NONE;
  return a;
}

// y = A x  [+ dots]
void op_spmv(amg_handle_s* H, const Level& L, const double* x, double* y, int ndot, const double* d0, int fin,
             KrylovCtl* ctl, cudaStream_t st) {
  RowArgs a = base_args(H, L, ctl);
  a.x = x;
  a.out = y;
  a.d0 = d0;
  a.fin = fin;
  if (ndot == 0)
    launch_row<OP_SPMV, 0>(H, L, a, st);
  else if (ndot == 1)
    launch_row<OP_SPMV, 1>(H, L, a, st);
  else
    launch_row<OP_SPMV, 2>(H, L, a, st);
}

void op_jacobi(amg_handle_s* H, const Level& L, const double* b, const double* x, double* out, bool dot,
               KrylovCtl* ctl, cudaStream_t st, const double* dinv = nullptr) {
  RowArgs a = base_args(H, L, ctl);
  if (dinv) a.dinv = dinv;  // the diagonal of this sweep (Chebyshev weights), or a copy of it (timing hook)
  a.x = x;
  a.b = b;
  a.out = out;
  a.fin = FIN_RZ;
  if (dot)
    launch_row<OP_JACOBI, 1>(H, L, a, st);
  else
    launch_row<OP_JACOBI, 0>(H, L, a, st);
}

void op_jacobi0(amg_handle_s* H, const Level& L, const double* b, double* out, KrylovCtl* ctl, cudaStream_t st,
                const double* d0 = nullptr, const double* d1 = nullptr) {
  RowArgs a = base_args(H, L, ctl);
  if (d0) a.dinv_x1 = d0;  // diagonals of the first and the second sweep
  if (d1) a.dinv = d1;
  a.b = b;
  a.out = out;
  launch_row<OP_JACOBI0, 0>(H, L, a, st);
}

void op_jacobi_prolong(amg_handle_s* H, const Level& L, const double* b, const double* x, const double* ec,
                       double* out, bool dot, KrylovCtl* ctl, cudaStream_t st, const double* dinv = nullptr) {
  RowArgs a = base_args(H, L, ctl);
  if (dinv) a.dinv = dinv;
  a.x = x;
  a.b = b;
  a.ec = ec;
  a.out = out;
  a.fin = FIN_RZ;
  if (dot)
    launch_row<OP_JACOBI_PROLONG, 1>(H, L, a, st);
  else
    launch_row<OP_JACOBI_PROLONG, 0>(H, L, a, st);
}

// rc = R (b - A x); with dinv_c / x1c also x1c = dinv_c o rc, the first sweep of the coarse level from zero
// (row-tile path only)
void op_residual_restrict(amg_handle_s* H, const Level& L, const double* b, const double* x, double* rc,
                          KrylovCtl* ctl, cudaStream_t st, const double* dinv_c = nullptr, double* x1c = nullptr) {
  RowArgs a = base_args(H, L, ctl);
  a.x = x;
  a.b = b;
  if (lv_fast(L)) {
    a.out = rc;
    a.dinv_c = x1c ? dinv_c : nullptr;
    a.out2 = dinv_c ? x1c : nullptr;
    if (L.stream_hint)
      launch_tile<OP_RESTRICT, 0, true>(H, L, a, st);
    else
      launch_tile<OP_RESTRICT, 0, false>(H, L, a, st);
  } else {
    a.out = L.rtmp;
    launch_row<OP_RESID, 0>(H, L, a, st);
    ++g_nlaunch, launch(k_restrict_rows, grid_for(L.nc), TPB, 0, st)(L.nc, L.agg_ptr, L.rtmp, rc, ctl);
  }
}

void op_coarse_solve(amg_handle_s* H, const double* b, double* x, KrylovCtl* ctl, cudaStream_t st) {
  const int n = H->nL;
  if (n <= LU_SMALL_MAX) {
    const size_t sm = sizeof(double) * ((size_t)n * (n + 1) + n);
    ++g_nlaunch, launch(k_lu_solve_small, 1, 256, sm, st)(n, g_tr ? H->luT : H->lu, g_tr ? H->pivT : H->piv, b, x, ctl);
    return;
  }
  int T = n <= 32 ? 32 : (n <= 64 ? 64 : (n <= 256 ? 256 : 1024));
  ++g_nlaunch, launch(k_lu_solve, 1, T, sizeof(double) * n, st)(n, g_tr ? H->luT : H->lu, g_tr ? H->pivT : H->piv, b, x, ctl);
}

// V-cycle from level D down as the dense collapsed operator (amg_tail.cuh); returns the result buffer
double* op_tail(amg_handle_s* H, const double* b, double* out, KrylovCtl* ctl, int fin, cudaStream_t st) {
  Level& L = H->lv[H->tail_dense_level];
  if (!out) out = L.x;
  TailArgs a;
  memset(&a, 0, sizeof(a));
  a.n = L.n;
  a.dense_B = g_tr ? H->tail_dense_BT : H->tail_dense_B;
  a.b = b;
  a.z = out;
  a.partials = H->partials;
  a.counter = H->counter;
  a.ctl = ctl;
  a.fin = fin;
  ++g_nlaunch, launch(k_dense_tail, H->tail_grid, TAIL_THREADS, 0, st)(a);
  return out;
}

}  // namespace

// Dense collapsed operator of the coarse tail: column j = V-cycle of levels D.. on e_j
// (transposed = 1: the same for the transposed hierarchy, after the forward one)
amg_status amg_setup_tail(amg_handle_s* H, int transposed, cudaStream_t st) {
  if (!transposed) H->tail_dense_level = -1;
  const int nlev = (int)H->lv.size();
  const int Lc = nlev - 1;
  if (H->opt.tail_dense_rows <= 0 || H->opt.force_generic || nlev > TAIL_MAX_LEVELS) return AMG_OK;
  int D = -1;
  for (int l = 0; l < nlev; ++l)
    if (H->lv[l].n <= H->opt.tail_dense_rows && H->lv[l].n <= MAX_DENSE) {
      D = l;
      break;
    }
  if (D < 0) return AMG_OK;
  const int nD = H->lv[D].n;
  const size_t lu_smem = (tail_smem_bytes(H->nL) + 127) & ~(size_t)127;
  size_t vec_bytes = 0;
  for (int l = D; l < nlev; ++l) vec_bytes += 3 * sizeof(double) * (size_t)H->lv[l].n;
  const size_t smem = lu_smem + vec_bytes;
  if (smem > 200 * 1024) return AMG_OK;
  if (transposed && H->tail_dense_level != D) return AMG_OK;  // no forward operator: levels are visited
  std::vector<TailLevel> h(nlev);
  for (int l = 0; l < nlev; ++l) {
    const Level& L = H->lv[l];
    TailLevel& T = h[l];
    T.n = L.n;
    T.nc = L.nc;
    T.nnz = L.nnz;
    const double mean = L.n > 0 ? (double)L.nnz / L.n : 1.0;
    T.lpr = mean <= 6.0 ? 4 : (mean <= 24.0 ? 8 : 16);
    T.rowptr = transposed ? L.T.rowptr : L.rowptr;
    T.col = transposed ? L.T.col : L.col;
    T.val = transposed ? L.T.val : L.val;
    T.dinv = L.dinv;
    for (int q = 0; q < AMG_MAX_SWEEPS; ++q) T.dsw[q] = L.dsw[q];
    T.agg = L.agg;
    T.agg_ptr = L.agg_ptr;
    T.v32 = L.v32;
  }
  TailLevel* d;
  AMG_ALLOC(H, d, TailLevel, nlev, st);
  AMG_CUDA_TRY(H, cudaMemcpyAsync(d, h.data(), sizeof(TailLevel) * nlev, cudaMemcpyHostToDevice, st));
  double*& Bd = transposed ? H->tail_dense_BT : H->tail_dense_B;
  if (!Bd) AMG_ALLOC(H, Bd, double, (size_t)nD * nD, st);
  TailBuildArgs ba;
  memset(&ba, 0, sizeof(ba));
  ba.lv = d;
  ba.D = D;
  ba.last = Lc;
  ba.nu1 = H->opt.pre_sweeps;
  ba.nu2 = H->opt.post_sweeps;
  ba.gamma = H->opt.coarse_scale;
  ba.nL = H->nL;
  ba.lu = transposed ? H->luT : H->lu;
  ba.piv = transposed ? H->pivT : H->piv;
  ba.B = Bd;
  ba.lu_smem = (int)lu_smem;
  launch(k_tail_dense_build, nD, TAILB_THREADS, smem, st)(ba);
  AMG_CUDA_TRY(H, cudaGetLastError());
  AMG_CUDA_TRY(H, cudaStreamSynchronize(st));  // h goes out of scope
  amg_dev_free(H, d);
  H->tail_dense_level = D;
  H->tail_grid = H->sm_count;
  return AMG_OK;
}

// ------------------------------------------------------------------------------------------
// S6: V-cycle from a zero guess.  *x_out points at the level's result buffer.
// fuse_rz: the last smoother sweep of level 0 also produces r.z (FIN_RZ).
// ------------------------------------------------------------------------------------------
amg_status amg_vcycle(amg_handle_s* H, int l, const double* b, double** x_out, KrylovCtl* ctl, bool fuse_rz,
                      cudaStream_t st, bool x1_ready) {
  const int Lc = (int)H->lv.size() - 1;
  Level& L = H->lv[l];
  // the caller may ask for the result of a level-0 cycle in a buffer of its own (BiCGSTAB keeps phat
  // across the second V-cycle of an iteration: no copy)
  double* const fo = (l == 0) ? H->vcycle_final_out : nullptr;
  if (l == H->tail_dense_level) {
    *x_out = op_tail(H, b, fo, ctl, (fuse_rz && l == 0) ? FIN_RZ : FIN_NONE, st);
    AMG_CUDA_TRY(H, cudaGetLastError());
    return AMG_OK;
  }
  if (l == Lc) {
    double* out = fo ? fo : L.x;
    op_coarse_solve(H, b, out, ctl, st);
    *x_out = out;
    if (fuse_rz && l == 0)
      ++g_nlaunch, launch(k_dot, red_grid(H, L.n), RED_THREADS, 0, st)(L.n, b, out, H->partials, H->counter, ctl, FIN_RZ);
    AMG_CUDA_TRY(H, cudaGetLastError());
    return AMG_OK;
  }
  const int nu1 = H->opt.pre_sweeps, nu2 = H->opt.post_sweeps;
  double* cur = L.x;
  double* oth = L.x2;
  int done_sweeps = 0;
  if (nu1 >= 2 && x1_ready) {
    // the restriction of the level above left x1 = dinv o b in L.x2: the second sweep is a plain one
    // (one gather per halo column instead of the two of the fused pair)
    op_jacobi(H, L, b, L.x2, cur, false, ctl, st, L.dsw[1]);
    done_sweeps = 2;
  } else if (nu1 >= 2) {
    op_jacobi0(H, L, b, cur, ctl, st, L.dsw[0], L.dsw[1]);
    done_sweeps = 2;
  } else if (nu1 == 1) {
    ++g_nlaunch, launch(k_scale_dinv, grid_for(L.n), TPB, 0, st)(L.n, L.dsw[0], b, cur, ctl);
    done_sweeps = 1;
  } else {
    ++g_nlaunch, launch(k_zero, grid_for(L.n), TPB, 0, st)(L.n, cur, ctl);
  }
  for (int s = done_sweeps; s < nu1; ++s) {
    op_jacobi(H, L, b, cur, oth, false, ctl, st, L.dsw[s]);
    std::swap(cur, oth);
  }
  Level& C = H->lv[l + 1];
  // the coarse level starts with two sweeps from zero on the row-tile path: hand it its first one
  const bool give_x1 = lv_fast(L) && lv_fast(C) && nu1 >= 2 && l + 1 < Lc && l + 1 != H->tail_dense_level;
  op_residual_restrict(H, L, b, cur, C.b, ctl, st, give_x1 ? C.dsw[0] : nullptr, give_x1 ? C.x2 : nullptr);
  double* ec = nullptr;
  AMG_TRY(amg_vcycle(H, l + 1, C.b, &ec, ctl, false, st, give_x1));
  const bool want_dot = fuse_rz && l == 0;
  if (nu2 >= 1) {
    double* out = (fo && nu2 == 1) ? fo : oth;
    if (lv_fast(L) && L.n >= H->opt.split_prolong_rows && H->opt.split_prolong_rows > 0) {
      // Two scattered loads per halo column make the fused sweep L1-bound on the largest levels
      // (level 0 of cfg 3: 53 us against 33 us for a plain sweep); there a separate unit-stride
      // correction pass (8 us) followed by the plain sweep is cheaper.
      ++g_nlaunch, launch(k_prolong_add, grid_for((L.n + 1) / 2), TPB, 0, st)(L.n, L.agg, ec, H->opt.coarse_scale, cur, cur, ctl);
      op_jacobi(H, L, b, cur, out, want_dot && nu2 == 1, ctl, st, L.dsw[nu1]);
    } else {
      op_jacobi_prolong(H, L, b, cur, ec, out, want_dot && nu2 == 1, ctl, st, L.dsw[nu1]);
    }
    if (out == oth)
      std::swap(cur, oth);
    else
      cur = out;
    for (int s = 1; s < nu2; ++s) {
      out = (fo && s == nu2 - 1) ? fo : oth;
      op_jacobi(H, L, b, cur, out, want_dot && s == nu2 - 1, ctl, st, L.dsw[nu1 + s]);
      if (out == oth)
        std::swap(cur, oth);
      else
        cur = out;
    }
  } else {
    double* out = fo ? fo : oth;
    ++g_nlaunch, launch(k_prolong_add, grid_for((L.n + 1) / 2), TPB, 0, st)(L.n, L.agg, ec, H->opt.coarse_scale, cur, out, ctl);
    cur = out;
    if (want_dot) ++g_nlaunch, launch(k_dot, red_grid(H, L.n), RED_THREADS, 0, st)(L.n, b, cur, H->partials, H->counter, ctl, FIN_RZ);
  }
  *x_out = cur;
  AMG_CUDA_TRY(H, cudaGetLastError());
  return AMG_OK;
}

// ------------------------------------------------------------------------------------------
// Krylov drivers.  Work vectors: kv[0]=x kv[1]=r kv[2]=p kv[3]=q/v kv[4]=rhat kv[5]=s kv[6]=t
// kv[7]=phat (copy when the V-cycle result buffer is reused) kv[8]=shat
// ------------------------------------------------------------------------------------------
namespace {

// buffer that receives x1 = dinv o b of level 0 from the kernel that produces b (so that the first two
// sweeps of the V-cycle are one plain sweep on x1), or null when the cycle does not start that way
double* l0_x1(amg_handle_s* H, int precond) {
  Level& L0 = H->lv[0];
  const int Lc = (int)H->lv.size() - 1;
  if (!precond || Lc == 0 || H->tail_dense_level == 0 || H->opt.pre_sweeps < 2 || !lv_fast(L0)) return nullptr;
  return L0.x2;
}

// one PCG iteration: q = A p, sigma; x,r update; z = B r, rho; p = z + beta p
amg_status enqueue_pcg_iteration(amg_handle_s* H, int precond, cudaStream_t st) {
  Level& L0 = H->lv[0];
  const int n = L0.n;
  double *x = H->kv[0], *r = H->kv[1], *p = H->kv[2], *q = H->kv[3];
  g_kop = 1;
  op_spmv(H, L0, p, q, 1, p, FIN_PQ, H->ctl, st);
  g_kop = 0;
  ++g_nlaunch, launch(k_pcg_xr, red_grid(H, n), RED_THREADS, 0, st)(n, p, q, x, r, L0.dsw[0], l0_x1(H, precond), H->partials,
                                                                        H->counter, H->ctl);
  double* z = r;
  if (precond) {
    AMG_TRY(amg_vcycle(H, 0, r, &z, H->ctl, true, st, l0_x1(H, precond) != nullptr));
  } else {
    ++g_nlaunch, launch(k_dot, red_grid(H, n), RED_THREADS, 0, st)(n, r, r, H->partials, H->counter, H->ctl, FIN_RZ);
  }
  ++g_nlaunch, launch(k_pcg_p, red_grid(H, n), RED_THREADS, 0, st)(n, z, p, H->ctl, g_loop);
  AMG_CUDA_TRY(H, cudaGetLastError());
  return AMG_OK;
}

amg_status enqueue_bicg_iteration(amg_handle_s* H, int precond, cudaStream_t st) {
  Level& L0 = H->lv[0];
  const int n = L0.n;
  double *x = H->kv[0], *r = H->kv[1], *p = H->kv[2], *v = H->kv[3], *rhat = H->kv[4], *s = H->kv[5],
         *t = H->kv[6], *ph = H->kv[7];
  ++g_nlaunch, launch(k_bicg_p, red_grid(H, n), RED_THREADS, 0, st)(n, r, v, p, L0.dsw[0], l0_x1(H, precond), H->ctl);
  double* phat = p;
  if (precond) {
    double* zz = nullptr;
    H->vcycle_final_out = ph;
    const amg_status sv = amg_vcycle(H, 0, p, &zz, H->ctl, false, st, l0_x1(H, precond) != nullptr);
    H->vcycle_final_out = nullptr;
    AMG_TRY(sv);
    phat = zz;  // == ph on every path of the cycle: the second V-cycle of this iteration may overwrite the level-0 buffers
  }
  g_kop = 1;
  op_spmv(H, L0, phat, v, 1, rhat, FIN_RV, H->ctl, st);
  g_kop = 0;
  ++g_nlaunch, launch(k_bicg_s, red_grid(H, n), RED_THREADS, 0, st)(n, r, v, s, L0.dsw[0], l0_x1(H, precond), H->partials,
                                                                        H->counter, H->ctl);
  double* shat = s;
  if (precond) AMG_TRY(amg_vcycle(H, 0, s, &shat, H->ctl, false, st, l0_x1(H, precond) != nullptr));
  g_kop = 1;
  op_spmv(H, L0, shat, t, 2, s, FIN_TS_TT, H->ctl, st);
  g_kop = 0;
  ++g_nlaunch, launch(k_bicg_xr, red_grid(H, n), RED_THREADS, 0, st)(n, phat, shat, s, t, rhat, x, r, H->partials, H->counter,
                                                   H->ctl);
  if (g_loop) ++g_nlaunch, launch(k_while_ctl, 1, 1, 0, st)((const KrylovCtl*)H->ctl, g_loop);
  AMG_CUDA_TRY(H, cudaGetLastError());
  return AMG_OK;
}

amg_status enqueue_iteration(amg_handle_s* H, int krylov, int precond, cudaStream_t st) {
  return krylov == 0 ? enqueue_pcg_iteration(H, precond, st) : enqueue_bicg_iteration(H, precond, st);
}

// the start of an AMG-PCG solve after k_krylov_init: z = B r (r.z on the last sweep), p = z
amg_status enqueue_pcg_start(amg_handle_s* H, cudaStream_t st) {
  double* z = nullptr;
  AMG_TRY(amg_vcycle(H, 0, H->kv[1], &z, H->ctl, true, st, l0_x1(H, 1) != nullptr));
  ++g_nlaunch, launch(k_pcg_p, red_grid(H, H->lv[0].n), RED_THREADS, 0, st)(H->lv[0].n, z, H->kv[2], H->ctl, (cudaGraphConditionalHandle)0);
  AMG_CUDA_TRY(H, cudaGetLastError());
  return AMG_OK;
}

// one V-cycle from level 0 on io_tmp2 (amg_apply_preconditioner): x1 = dinv o r, then the cycle
amg_status enqueue_apply(amg_handle_s* H, cudaStream_t st) {
  Level& L0 = H->lv[0];
  double* x1 = l0_x1(H, 1);
  if (x1) ++g_nlaunch, launch(k_scale_dinv, grid_for(L0.n), TPB, 0, st)(L0.n, L0.dsw[0], H->io_tmp2, x1, nullptr);
  AMG_TRY(amg_vcycle(H, 0, H->io_tmp2, &H->apply_out, nullptr, false, st, x1 != nullptr));
  return AMG_OK;
}

// krylov == -1: the start graph (slot 4); -2: amg_apply_preconditioner (slot 6); g_tr: the transposed BiCGSTAB +
// AMG iteration (slot 5)
inline int graph_slot(int krylov, int precond) {
  return krylov == -2 ? 6 : (krylov < 0 ? 4 : (g_tr ? 5 : krylov * 2 + precond));
}

amg_status get_iteration_graph(amg_handle_s* H, int krylov, int precond, cudaStream_t st, cudaGraphExec_t* out) {
  const int slot = graph_slot(krylov, precond);
  if (H->graph_exec[slot]) {
    *out = H->graph_exec[slot];
    return AMG_OK;
  }
  cudaGraph_t g = nullptr;
  (void)st;
  if (!H->cap_stream) AMG_CUDA_TRY(H, cudaStreamCreateWithFlags(&H->cap_stream, cudaStreamNonBlocking));
  AMG_CUDA_TRY(H, cudaStreamBeginCapture(H->cap_stream, cudaStreamCaptureModeThreadLocal));
  const int64_t launches0 = g_nlaunch;
  g_pdl = H->opt.use_pdl != 0;
  amg_status s = krylov == -2 ? enqueue_apply(H, H->cap_stream)
                 : krylov < 0 ? enqueue_pcg_start(H, H->cap_stream)
                              : enqueue_iteration(H, krylov, precond, H->cap_stream);
  g_pdl = false;
  H->graph_launches[slot] = g_nlaunch - launches0;  // kernel nodes of one replay
  g_nlaunch = launches0;                            // capturing enqueues nothing
  cudaError_t e = cudaStreamEndCapture(H->cap_stream, &g);
  if (s != AMG_OK) {
    if (g) cudaGraphDestroy(g);
    return s;
  }
  AMG_CUDA_TRY(H, e);
  cudaGraphExec_t ex = nullptr;
  e = cudaGraphInstantiate(&ex, g, 0);
  cudaGraphDestroy(g);
  AMG_CUDA_TRY(H, e);
  H->graph_exec[slot] = ex;
  *out = ex;
  return AMG_OK;
}

// The whole Krylov loop as ONE graph: a conditional WHILE node whose body is one iteration (PDL-chained
// kernels); the body's last kernel sets the condition from the device-side convergence flag.  No host polling,
// no copy between iterations, no surplus iteration.  Returns AMG_ERR_UNSUPPORTED (once, remembered) if the driver
// refuses any step: the caller falls back to replaying the iteration graph under host control.
amg_status get_while_graph(amg_handle_s* H, int krylov, int precond, cudaGraphExec_t* out) {
  const int slot = g_tr ? 4 : krylov * 2 + precond;
  if (H->while_exec[slot]) {
    *out = H->while_exec[slot];
    return AMG_OK;
  }
  if (H->while_failed) return AMG_ERR_UNSUPPORTED;
  if (!H->cap_stream && cudaStreamCreateWithFlags(&H->cap_stream, cudaStreamNonBlocking) != cudaSuccess) return AMG_ERR_CUDA;
  cudaGraph_t g = nullptr;
  cudaGraphExec_t ex = nullptr;
  bool ok = cudaGraphCreate(&g, 0) == cudaSuccess;
  cudaGraphConditionalHandle hd = 0;
  ok = ok && cudaGraphConditionalHandleCreate(&hd, g, 1, cudaGraphCondAssignDefault) == cudaSuccess;
  cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
  np.type = cudaGraphNodeTypeConditional;
  np.conditional.handle = hd;
  np.conditional.type = cudaGraphCondTypeWhile;
  np.conditional.size = 1;
  cudaGraphNode_t node = nullptr;
  ok = ok && cudaGraphAddNode(&node, g, nullptr, 0, &np) == cudaSuccess;
  amg_status s = AMG_OK;
  if (ok) {
    cudaGraph_t body = np.conditional.phGraph_out[0];
    ok = cudaStreamBeginCaptureToGraph(H->cap_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal) ==
         cudaSuccess;
    if (ok) {
      const int64_t launches0 = g_nlaunch;
      g_pdl = H->opt.use_pdl != 0;
      g_loop = hd;
      s = enqueue_iteration(H, krylov, precond, H->cap_stream);
      g_loop = 0;
      g_pdl = false;
      H->while_launches[slot] = g_nlaunch - launches0;
      g_nlaunch = launches0;
      cudaGraph_t cap = nullptr;
      ok = cudaStreamEndCapture(H->cap_stream, &cap) == cudaSuccess && s == AMG_OK;
    }
  }
  ok = ok && cudaGraphInstantiate(&ex, g, 0) == cudaSuccess;
  if (g) cudaGraphDestroy(g);
  if (!ok) {
    cudaGetLastError();
    H->while_failed = true;
    return s != AMG_OK ? s : AMG_ERR_UNSUPPORTED;
  }
  H->while_exec[slot] = ex;
  *out = ex;
  return AMG_OK;
}

}  // namespace

void amg_destroy_graphs(amg_handle_s* H) {
  for (auto& g : H->while_exec)
    if (g) {
      cudaGraphExecDestroy(g);
      g = nullptr;
    }
  for (auto& g : H->graph_exec)
    if (g) {
      cudaGraphExecDestroy(g);
      g = nullptr;
    }
  if (H->cap_stream) {
    cudaStreamDestroy(H->cap_stream);
    H->cap_stream = nullptr;
  }
}

amg_status amg_krylov_solve(amg_handle_s* H, const double* d_b, double* d_x, double rtol, int maxit, int krylov,
                            int precond, int transposed, amg_info* info, cudaStream_t st) {
  struct TrScope {  // the enqueue helpers read g_tr
    TrScope(int t) { g_tr = t; }
    ~TrScope() { g_tr = 0; }
  } tr_scope(transposed);
  Level& L0 = H->lv[0];
  const int n = L0.n;
  double *x = H->kv[0], *r = H->kv[1], *p = H->kv[2], *v = H->kv[3], *rhat = H->kv[4];
  const int64_t launches0 = g_nlaunch;
  // loop control: rtol / maxit / the history buffer go to the device as arguments of the init kernel
  if (H->hist_cap < maxit) {  // residual history (PAPER.md:125 diagnostics): one entry per iteration
    if (H->hist) {
      AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
      amg_dev_free(H, H->hist);
    }
    H->hist_cap = maxit < 256 ? 256 : maxit;
    H->hist = (double*)amg_dev_alloc(H, sizeof(double) * (size_t)H->hist_cap, st);
    if (!H->hist) {
      H->hist_cap = 0;
      H->err = "device allocation failed: residual history";
      return AMG_ERR_OOM;
    }
  }
  CtlInit ci;
  ci.rtol = rtol, ci.maxit = maxit, ci.hist = H->hist, ci.hist_cap = H->hist_cap;
  H->hist_len = 0;
  if (krylov == 0) {
    ++g_nlaunch, launch(k_krylov_init, red_grid(H, n), RED_THREADS, 0, st)(n, d_b, L0.inv, r, x, p, nullptr, nullptr, L0.dsw[0],
                                                         l0_x1(H, precond), H->partials, H->counter, H->ctl, FIN_INIT_PCG, ci);
    if (precond && H->opt.use_graph && maxit > 0) {
      cudaGraphExec_t gstart = nullptr;
      AMG_TRY(get_iteration_graph(H, -1, 1, st, &gstart));
      AMG_CUDA_TRY(H, cudaGraphLaunch(gstart, st));
      g_nlaunch += H->graph_launches[4];
    } else if (precond) {
      AMG_TRY(enqueue_pcg_start(H, st));
    } else {
      ++g_nlaunch, launch(k_dot, red_grid(H, n), RED_THREADS, 0, st)(n, r, r, H->partials, H->counter, H->ctl, FIN_RZ);
      ++g_nlaunch, launch(k_pcg_p, red_grid(H, n), RED_THREADS, 0, st)(n, r, p, H->ctl, (cudaGraphConditionalHandle)0);
    }
  } else {
    ++g_nlaunch, launch(k_krylov_init, red_grid(H, n), RED_THREADS, 0, st)(n, d_b, L0.inv, r, x, p, v, rhat, nullptr, nullptr,
                                                         H->partials, H->counter, H->ctl, FIN_INIT_BICG, ci);
  }
  AMG_CUDA_TRY(H, cudaGetLastError());

  // the loop: one graph with a conditional WHILE node (device-side loop control), else the iteration graph
  // replayed under host control
  cudaGraphExec_t gwhile = nullptr;
  if (H->opt.use_graph && H->opt.use_while && maxit > 0) {
    const amg_status sw = get_while_graph(H, krylov, precond, &gwhile);
    if (sw != AMG_OK && sw != AMG_ERR_UNSUPPORTED) return sw;
  }
  if (gwhile) {
    AMG_CUDA_TRY(H, cudaGraphLaunch(gwhile, st));
    H->while_used = true;
  } else {
    cudaGraphExec_t gexec = nullptr;
    if (H->opt.use_graph && maxit > 0) AMG_TRY(get_iteration_graph(H, krylov, precond, st, &gexec));
    // The host runs at most LAG iterations ahead of the device's convergence flag; iterations
    // enqueued after convergence return at their first instruction.
    constexpr int NSLOT = 4, LAG = 1;
    for (int it = 0; it < maxit; ++it) {
      if (gexec) {
        AMG_CUDA_TRY(H, cudaGraphLaunch(gexec, st));
        g_nlaunch += H->graph_launches[graph_slot(krylov, precond)];
      } else
        AMG_TRY(enqueue_iteration(H, krylov, precond, st));
      const int slot = it % NSLOT;
      AMG_CUDA_TRY(H, cudaMemcpyAsync(&H->h_ctl[slot], H->ctl, sizeof(KrylovCtl), cudaMemcpyDeviceToHost, st));
      AMG_CUDA_TRY(H, cudaEventRecord(H->ev[slot], st));
      if (it >= LAG) {
        const int old = (it - LAG) % NSLOT;
        AMG_CUDA_TRY(H, cudaEventSynchronize(H->ev[old]));
        if (H->h_ctl[old].done) break;
      }
    }
  }
  const bool half = (krylov == 1);
  const double* phat = half ? (precond ? H->kv[7] : p) : nullptr;
  ++g_nlaunch, launch(k_krylov_output, grid_for(n), TPB, 0, st)(n, x, phat, L0.inv, d_x, H->ctl);
  AMG_CUDA_TRY(H, cudaGetLastError());
  H->last_launches = g_nlaunch - launches0;
  // info == NULL: the call returns here, with the last iteration and the output kernel still in the
  // stream (x is valid in stream order; nothing is reported)
  if (!info) return AMG_OK;
  AMG_CUDA_TRY(H, cudaMemcpyAsync(&H->h_ctl[4], H->ctl, sizeof(KrylovCtl), cudaMemcpyDeviceToHost, st));
  AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
  const KrylovCtl& c = H->h_ctl[4];
  if (gwhile) {  // kernels the device-side loop launched: iterations passed x kernel nodes of the body
    const int slot = g_tr ? 4 : krylov * 2 + precond;
    g_nlaunch += (int64_t)(c.iter > 0 ? c.iter : 1) * H->while_launches[slot];
    H->last_launches = g_nlaunch - launches0;
  }
  H->hist_len = c.iter < H->hist_cap ? c.iter : H->hist_cap;
  info->iterations = c.iter;
  info->status = c.status;
  info->b_norm = sqrt(c.bnorm2);
  info->rel_residual = c.bnorm2 > 0.0 ? sqrt(c.rr) / sqrt(c.bnorm2) : 0.0;
  if (c.status == AMG_MAXIT && c.iter == 0) info->rel_residual = c.bnorm2 > 0.0 ? 1.0 : 0.0;
  return AMG_OK;
}

void amg_configure_kernels() {
  // opt in to > 48 KB of dynamic shared memory: a per-device attribute of every instantiation in use
  set_tile_attr<OP_SPMV, 0>(), set_tile_attr<OP_SPMV, 1>(), set_tile_attr<OP_SPMV, 2>();
  set_tile_attr<OP_JACOBI, 0>(), set_tile_attr<OP_JACOBI, 1>();
  set_tile_attr<OP_JACOBI0, 0>();
  set_tile_attr<OP_JACOBI_PROLONG, 0>(), set_tile_attr<OP_JACOBI_PROLONG, 1>();
  set_tile_attr<OP_RESTRICT, 0>();
  cudaFuncSetAttribute(k_tail_dense_build, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
}

// ------------------------------------------------------------------------------------------
// per-level hooks (natural numbering at the boundary)
// ------------------------------------------------------------------------------------------
amg_status amg_level_op_impl(amg_handle_s* H, int level, int op, const double* d_in0, const double* d_in1,
                             double* d_out, int reps, cudaStream_t st) {
  const int Lc = (int)H->lv.size() - 1;
  Level& L = H->lv[level];
  if (reps < 1) reps = 1;
  const int64_t launches0 = g_nlaunch;
  double *t0 = H->io_tmp, *t1 = H->io_tmp2, *t2 = H->io_tmp3;
  const bool needs_coarse = (op >= 1 && op <= 4) || op == 6;
  if (needs_coarse && level >= Lc) {
    H->err = "level op needs a level below the coarsest";
    return AMG_ERR_INVALID_ARG;
  }
  auto perm_in = [&](const Level& Lv, const double* nat, double* out) {
    ++g_nlaunch, launch(k_permute_in, grid_for(Lv.n), TPB, 0, st)(Lv.n, nat, Lv.inv, out);
  };
  auto perm_out = [&](const Level& Lv, const double* in, double* nat) {
    ++g_nlaunch, launch(k_permute_out, grid_for(Lv.n), TPB, 0, st)(Lv.n, in, Lv.inv, nat);
  };
  switch (op) {
    case 0:
      if (!d_in0) return AMG_ERR_INVALID_ARG;
      perm_in(L, d_in0, t0);
      for (int r = 0; r < reps; ++r) op_spmv(H, L, t0, t2, 0, nullptr, FIN_NONE, nullptr, st);
      perm_out(L, t2, d_out);
      break;
    case 1:
      if (!d_in0 || !d_in1) return AMG_ERR_INVALID_ARG;
      perm_in(L, d_in0, t0);
      perm_in(L, d_in1, t1);
      if (level == 0 && reps > 1) {
        // timing of back-to-back sweeps: the launches rotate over three operand sets (x, b, dinv, out:
        // 12 level-0 vectors) so that no operand of a launch can still sit in L2 from the launch before
        double* set[3][4] = {{t0, t1, H->kv[0], t2}, {H->kv[1], H->kv[2], H->kv[3], H->kv[4]},
                             {H->kv[5], H->kv[6], H->kv[7], H->kv[8]}};
        const size_t bytes = sizeof(double) * (size_t)L.n;
        for (int q = 0; q < 3; ++q) {
          if (q > 0) {
            AMG_CUDA_TRY(H, cudaMemcpyAsync(set[q][0], t0, bytes, cudaMemcpyDeviceToDevice, st));
            AMG_CUDA_TRY(H, cudaMemcpyAsync(set[q][1], t1, bytes, cudaMemcpyDeviceToDevice, st));
          }
          AMG_CUDA_TRY(H, cudaMemcpyAsync(set[q][2], L.dinv, bytes, cudaMemcpyDeviceToDevice, st));
        }
        for (int r = 0; r < reps; ++r) {
          double** q = set[(reps - 1 - r) % 3];  // the last launch works on set 0: its result goes out
          op_jacobi(H, L, q[1], q[0], q[3], false, nullptr, st, q[2]);
        }
      } else {
        for (int r = 0; r < reps; ++r) op_jacobi(H, L, t1, t0, t2, false, nullptr, st);
      }
      perm_out(L, t2, d_out);
      break;
    case 2: {
      if (!d_in0 || !d_in1) return AMG_ERR_INVALID_ARG;
      Level& C = H->lv[level + 1];
      perm_in(L, d_in0, t0);
      perm_in(L, d_in1, t1);
      for (int r = 0; r < reps; ++r) op_residual_restrict(H, L, t1, t0, t2, nullptr, st);
      perm_out(C, t2, d_out);
    } break;
    case 3: {
      if (!d_in0 || !d_in1) return AMG_ERR_INVALID_ARG;
      Level& C = H->lv[level + 1];
      perm_in(L, d_in0, t0);
      perm_in(C, d_in1, t1);
      for (int r = 0; r < reps; ++r)
        ++g_nlaunch, launch(k_prolong_add, grid_for((L.n + 1) / 2), TPB, 0, st)(L.n, L.agg, t1, H->opt.coarse_scale, t0, t2, nullptr);
      perm_out(L, t2, d_out);
    } break;
    case 4:
      if (!d_in1) return AMG_ERR_INVALID_ARG;
      perm_in(L, d_in1, t1);
      for (int r = 0; r < reps; ++r) op_jacobi0(H, L, t1, t2, nullptr, st);
      perm_out(L, t2, d_out);
      break;
    case 5: {
      if (!d_in1) return AMG_ERR_INVALID_ARG;
      perm_in(L, d_in1, t1);
      double* z = nullptr;
      if (level == 0 && H->opt.use_graph && !g_tr) {
        // the preconditioner itself: the cycle replayed as a PDL-chained graph, like inside a solve
        cudaGraphExec_t gx = nullptr;
        AMG_TRY(get_iteration_graph(H, -2, 1, st, &gx));
        for (int r = 0; r < reps; ++r) {
          AMG_CUDA_TRY(H, cudaGraphLaunch(gx, st));
          g_nlaunch += H->graph_launches[6];
        }
        z = H->apply_out;
      } else {
        for (int r = 0; r < reps; ++r) AMG_TRY(amg_vcycle(H, level, t1, &z, nullptr, false, st));
      }
      perm_out(L, z, d_out);
    } break;
    case 6: {  // prolongation-fused sweep: d_in1 = [b (rows of this level) | e_c (rows of the next)]
      if (!d_in0 || !d_in1) return AMG_ERR_INVALID_ARG;
      Level& C = H->lv[level + 1];
      perm_in(L, d_in0, t0);
      perm_in(L, d_in1, t1);
      perm_in(C, d_in1 + L.n, C.x2);
      for (int r = 0; r < reps; ++r) op_jacobi_prolong(H, L, t1, t0, C.x2, t2, false, nullptr, st);
      perm_out(L, t2, d_out);
    } break;
    case 7:  // y = A_l^T x (nonsymmetric handles)
    case 8: {  // V-cycle of the transposed hierarchy started at this level: z = B_l^T b
      if (!H->have_T) {
        H->err = "level op 7 / 8: the handle has no transposed hierarchy (symmetric matrix)";
        return AMG_ERR_INVALID_ARG;
      }
      const double* in = op == 7 ? d_in0 : d_in1;
      if (!in) return AMG_ERR_INVALID_ARG;
      perm_in(L, in, t1);
      g_tr = 1;
      amg_status sv = AMG_OK;
      double* z = t2;
      for (int r = 0; r < reps && sv == AMG_OK; ++r) {
        if (op == 7)
          op_spmv(H, L, t1, t2, 0, nullptr, FIN_NONE, nullptr, st);
        else
          sv = amg_vcycle(H, level, t1, &z, nullptr, false, st);
      }
      g_tr = 0;
      AMG_TRY(sv);
      perm_out(L, z, d_out);
    } break;
    default:
      H->err = "unknown level op";
      return AMG_ERR_INVALID_ARG;
  }
  AMG_CUDA_TRY(H, cudaGetLastError());
  H->last_launches = g_nlaunch - launches0;  // stream-ordered: no synchronisation
  return AMG_OK;
}

// ------------------------------------------------------------------------------------------
// G2
// ------------------------------------------------------------------------------------------
amg_status amg_grad_values_impl(amg_handle_s* H, const double* d_lambda, const double* d_x, int nrhs, int64_t ld,
                                double* d_gA, int accumulate, cudaStream_t st) {
  const int n = (int)H->n;
  const double mean = n > 0 ? (double)H->nnz / n : 1.0;
  if (nrhs > 1) {
    // interleave X once, then one contiguous gather of nrhs values per stored entry; the scratch stays on
    // the handle (grown on demand), so that a call allocates nothing and does not synchronise
    const size_t need = sizeof(double) * (size_t)n * nrhs;
    if (H->grad_xt_cap < need) {
      if (H->grad_xt) {
        AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
        amg_dev_free(H, H->grad_xt);
        H->grad_xt = nullptr, H->grad_xt_cap = 0;
      }
      H->grad_xt = (double*)amg_dev_alloc(H, need, st);
      if (!H->grad_xt) {
        H->err = "device allocation failed: interleaved right-hand sides";
        return AMG_ERR_OOM;
      }
      H->grad_xt_cap = need;
    }
    double* XT = H->grad_xt;
    const size_t sm = sizeof(double) * (size_t)nrhs * (GT_ROWS + 1);
    if (sm > 48 * 1024) {
      H->err = "amg_grad_values: nrhs too large (at most 94 right-hand sides per call; accumulate over calls)";
      return AMG_ERR_UNSUPPORTED;
    }
    ++g_nlaunch, launch(k_interleave_rhs, div_up(n, GT_ROWS), 256, sm, st)(n, nrhs, ld, d_x, XT);
    const int g8 = div_up((int64_t)n * 8, 256), g32 = div_up((int64_t)n * 32, 256);
    const bool wide = mean > 12.0;
#define AMG_GRAD_CASE(NR)                                                                                          \
  if (wide)                                                                                                       \
    ++g_nlaunch, launch(k_grad_values_batched<32, NR>, g32, 256, 0, st)(n, H->nat_rowptr, H->nat_col, d_lambda, ld, \
                                                                        XT, nrhs, d_gA, accumulate);                \
  else                                                                                                            \
    ++g_nlaunch, launch(k_grad_values_batched<8, NR>, g8, 256, 0, st)(n, H->nat_rowptr, H->nat_col, d_lambda, ld,   \
                                                                      XT, nrhs, d_gA, accumulate);
    switch (nrhs) {
      case 2: AMG_GRAD_CASE(2) break;
      case 4: AMG_GRAD_CASE(4) break;
      case 8:  // nrhs / 2 lanes per stored entry: one coalesced request per entry
        ++g_nlaunch, launch(k_grad_values_coop<8>, div_up((int64_t)n * 4, 256), 256, 0, st)(n, H->nat_rowptr, H->nat_col, d_lambda, ld, XT, d_gA, accumulate);
        break;
      case 16:
        ++g_nlaunch, launch(k_grad_values_coop<16>, div_up((int64_t)n * 8, 256), 256, 0, st)(n, H->nat_rowptr, H->nat_col, d_lambda, ld, XT, d_gA, accumulate);
        break;
      default: AMG_GRAD_CASE(0) break;
    }
#undef AMG_GRAD_CASE
    AMG_CUDA_TRY(H, cudaGetLastError());
    H->last_launches = 2;
    return AMG_OK;
  }
  if (nrhs == 1 && H->opt.force_generic == 0) {
    ++g_nlaunch, launch(k_grad_values_entries, div_up(n, 256), 256, 0, st)(n, H->nat_rowptr, H->nat_col, d_lambda, d_x, d_gA, accumulate);
  } else if (mean <= 12.0 && nrhs == 1) {
    ++g_nlaunch, launch(k_grad_values_rows, div_up(n, 256), 256, 0, st)(n, H->nat_rowptr, H->nat_col, d_lambda, d_x, d_gA, accumulate);
  } else if (mean <= 12.0) {
    const int64_t threads = (int64_t)n * 8;
    ++g_nlaunch, launch(k_grad_values<8>, div_up(threads, 256), 256, 0, st)(n, H->nat_rowptr, H->nat_col, d_lambda, d_x, nrhs, ld,
                                                          d_gA, accumulate);
  } else {
    const int64_t threads = (int64_t)n * 32;
    ++g_nlaunch, launch(k_grad_values<32>, div_up(threads, 256), 256, 0, st)(n, H->nat_rowptr, H->nat_col, d_lambda, d_x, nrhs, ld,
                                                           d_gA, accumulate);
  }
  AMG_CUDA_TRY(H, cudaGetLastError());
  H->last_launches = 1;
  return AMG_OK;
}

// ------------------------------------------------------------------------------------------
// algorithmic bytes
// ------------------------------------------------------------------------------------------
double amg_algorithmic_bytes(amg_handle_s* H, int which) {
  const int Lc = (int)H->lv.size() - 1;
  auto M = [&](int l) { return 12.0 * H->lv[l].nnz + 4.0 * (H->lv[l].n + 1); };
  auto V = [&](int l) { return 8.0 * H->lv[l].n; };
  auto vcycle = [&]() {
    // per level l < L with V(2,2): 4 matrix passes + 13 vector passes + 2 index passes + 2 coarse vectors
    const int nu1 = H->opt.pre_sweeps, nu2 = H->opt.post_sweeps;
    double tot = 0.0;
    for (int l = 0; l < Lc; ++l) {
      const double Ml = M(l), Vl = V(l), Cl = 4.0 * H->lv[l].n, Vc = V(l + 1);
      double b = 0.0;
      if (nu1 >= 2) b += Ml + 3 * Vl;                       // fused first two sweeps: b, dinv -> x
      else if (nu1 == 1) b += 3 * Vl;
      else b += Vl;
      for (int s = 2; s < nu1; ++s) b += Ml + 4 * Vl;       // x, b, dinv -> x'
      b += Ml + 2 * Vl + Cl + Vc;                           // residual + restriction: x, b, agg_ptr -> r_c
      if (nu2 >= 1) b += Ml + 4 * Vl + Cl + Vc;             // prolongation fused into the first post sweep
      else b += 2 * Vl + Cl + Vc;
      for (int s = 1; s < nu2; ++s) b += Ml + 4 * Vl;
      tot += b;
    }
    tot += 8.0 * H->nL * H->nL + 16.0 * H->nL;
    return tot;
  };
  switch (which) {
    case 0: return M(0) + 2 * V(0);
    case 1: return vcycle();
    case 2: return (M(0) + 2 * V(0)) + 6 * V(0) + 3 * V(0) + vcycle();
    case 3: return 2 * (M(0) + 2 * V(0)) + 2 * vcycle() + (4 + 3 + 8) * V(0) + 2 * V(0);
    case 4: return M(0) + 4 * V(0);
    case 10: {  // bytes the V-cycle's operators occupy as stored: tile blobs + halo index lists (else the CSR)
      double tot = 0.0;
      for (int l = 0; l < Lc; ++l) tot += H->lv[l].fast ? (double)H->lv[l].blob_bytes : M(l);
      return tot;
    }
    case 11: return H->lv[0].fast ? (double)H->lv[0].blob_bytes : M(0);  // level 0 alone
    case 12: {  // levels stored as 8-bit codes into a value dictionary
      double cnt = 0.0;
      for (int l = 0; l < Lc; ++l) cnt += H->lv[l].ndict > 0 ? 1.0 : 0.0;
      return cnt;
    }
    default: return 0.0;
  }
}
