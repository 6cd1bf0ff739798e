// Host driver of the batched multi-right-hand-side AMG-PCG solve (NEXT-3; kernels in
// amg_batched.cuh): work vectors for NB interleaved right-hand sides, ring geometry per level,
// batched V-cycle, the iteration replayed as a PDL-chained CUDA graph, per-column results.
#include <algorithm>
#include <cstring>

#include "amg_batched.cuh"

struct LevelGeomB {
  int stages = 0, xslots = 0, stage_bytes = 0, xslot_bytes = 0, smem = 0;
};

struct AmgBatch {
  int eligible = -1;  // -1: not examined yet
  std::vector<double*> x, x2, b;  // per level, [n_l][NB]
  std::vector<LevelGeomB> geom;
  LevelGeomB geomK;  // level 0's fp64 blobs of a mixed-precision hierarchy (the Krylov SpMV)
  double* kv[4] = {nullptr, nullptr, nullptr, nullptr};  // x, r, p, q
  KrylovCtlB* ctl = nullptr;
  KrylovCtlB* h_ctl = nullptr;  // pinned, 6 slots
  double* partials = nullptr;
  int partials_cap = 0;
  unsigned* counter = nullptr;
  cudaGraphExec_t g_start = nullptr, g_iter = nullptr, g_while = nullptr;  // g_while: the loop as one WHILE-node graph
  int64_t nl_start = 0, nl_iter = 0;
  bool while_failed = false;
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
};

namespace {

thread_local int64_t gb_nlaunch = 0;
thread_local bool gb_pdl = false;
thread_local cudaGraphConditionalHandle gb_loop = 0;  // != 0 while the body of a WHILE node is captured

template <typename... KArgs, typename... A>
void launch_b(void (*k)(KArgs...), dim3 g, dim3 b, size_t sm, cudaStream_t st, A&&... a) {
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = g, cfg.blockDim = b, cfg.dynamicSmemBytes = sm, cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = gb_pdl ? 1 : 0;
  cudaLaunchKernelEx(&cfg, k, KArgs(a)...);
  ++gb_nlaunch;
}

inline int red_grid_b(const amg_handle_s* H, int64_t units) {
  int g = div_up(units, RED_THREADS * 4);
  const int cap = H->sm_count * 8;
  return g > cap ? cap : (g < 1 ? 1 : g);
}

template <int OP, int NDOT>
void set_attr_b() {
  cudaFuncSetAttribute(k_rowtile_b<OP, NDOT, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, RTB_SMEM_MAX);
  cudaFuncSetAttribute(k_rowtile_b<OP, NDOT, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, RTB_SMEM_MAX);
  cudaFuncSetAttribute(k_rowtile_b<OP, NDOT, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, RTB_SMEM_MAX_VD);
  cudaFuncSetAttribute(k_rowtile_b<OP, NDOT, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, RTB_SMEM_MAX_VD);
}

template <int OP, int NDOT>
void launch_rowtile_b(amg_handle_s* H, const Level& L, const LevelGeomB& G, RowArgsB& a, cudaStream_t st,
                      const LevelOpT* K = nullptr) {
  a.n = L.n, a.tiles = L.tiles, a.ntiles = L.nblk, a.blob = L.blob, a.halo_idx = L.halo_idx;
  if (K) a.tiles = K->tiles, a.ntiles = K->nblk, a.blob = K->blob, a.halo_idx = K->halo_idx;
  a.vdict = (L.ndict > 0 && !K) ? L.vdict : nullptr;
  if (!a.dinv) a.dinv = L.dinv;  // (the sweeps pass the diagonal of their own sweep index: Chebyshev weights)
  a.agg_ptr = L.agg_ptr;
  a.partials = H->batch->partials, a.counter = H->batch->counter;
  a.stages = G.stages, a.xslots = G.xslots, a.stage_bytes = G.stage_bytes, a.xslot_bytes = G.xslot_bytes;
  int grid = H->sm_count;  // one CTA per SM
  if (grid > a.ntiles) grid = a.ntiles;
  const bool vd = a.vdict != nullptr;
  if (L.stream_hint) {
    if (vd) launch_b(k_rowtile_b<OP, NDOT, true, true>, grid, RTB_THREADS, G.smem, st, a);
    else launch_b(k_rowtile_b<OP, NDOT, true, false>, grid, RTB_THREADS, G.smem, st, a);
  } else {
    if (vd) launch_b(k_rowtile_b<OP, NDOT, false, true>, grid, RTB_THREADS, G.smem, st, a);
    else launch_b(k_rowtile_b<OP, NDOT, false, false>, grid, RTB_THREADS, G.smem, st, a);
  }
}

RowArgsB args_b(KrylovCtlB* ctl) {
  RowArgsB a;
  memset(&a, 0, sizeof(a));
  a.ctl = ctl;
  a.fin = FIN_NONE;
  return a;
}

void op_jacobi_b(amg_handle_s* H, int l, const double* b, const double* x, double* out, bool dot, KrylovCtlB* ctl,
                 cudaStream_t st, int sweep) {
  RowArgsB a = args_b(ctl);
  a.x = x, a.b = b, a.out = out, a.fin = FIN_RZ, a.dinv = H->lv[l].dsw[sweep];
  if (dot)
    launch_rowtile_b<OP_JACOBI, 1>(H, H->lv[l], H->batch->geom[l], a, st);
  else
    launch_rowtile_b<OP_JACOBI, 0>(H, H->lv[l], H->batch->geom[l], a, st);
}

// V-cycle from a zero guess for NB right-hand sides.  The first sweep x1 = dinv o b of level l is in
// x2[l] already (written by the kernel that produced b).  Returns the result buffer.
amg_status vcycle_b(amg_handle_s* H, int l, const double* b, double** out, KrylovCtlB* ctl, bool fuse_rz,
                    cudaStream_t st) {
  AmgBatch& Bt = *H->batch;
  Level& L = H->lv[l];
  if (l == H->tail_dense_level) {
    TailArgsB a;
    memset(&a, 0, sizeof(a));
    a.n = L.n, a.dense_B = H->tail_dense_B, a.b = b, a.z = Bt.x[l];
    a.partials = Bt.partials, a.counter = Bt.counter, a.ctl = ctl;
    a.fin = (fuse_rz && l == 0) ? FIN_RZ : FIN_NONE;
    launch_b(k_dense_tail_b, H->sm_count, TAILB_T, 0, st, a);
    *out = Bt.x[l];
    AMG_CUDA_TRY(H, cudaGetLastError());
    return AMG_OK;
  }
  const int nu1 = H->opt.pre_sweeps, nu2 = H->opt.post_sweeps;
  double *cur = Bt.x2[l], *oth = Bt.x[l];  // cur = x1 (one sweep from zero)
  for (int s = 1; s < nu1; ++s) {
    op_jacobi_b(H, l, b, cur, oth, false, ctl, st, s);
    std::swap(cur, oth);
  }
  const int lc = l + 1;
  {
    RowArgsB a = args_b(ctl);
    a.x = cur, a.b = b, a.out = Bt.b[lc];
    if (lc != H->tail_dense_level) a.dinv_c = H->lv[lc].dsw[0], a.out2 = Bt.x2[lc];  // x1 of the coarse level
    launch_rowtile_b<OP_RESTRICT, 0>(H, L, Bt.geom[l], a, st);
  }
  double* ec = nullptr;
  AMG_TRY(vcycle_b(H, lc, Bt.b[lc], &ec, ctl, false, st));
  const bool want_dot = fuse_rz && l == 0;
  // the coarse correction x += gamma P e_c is its own unit-stride pass, then a plain sweep: the fused variant
  // needs two gathers per column and keeps the own rows off the bulk copies (level 0 of cfg 3, 8 right-hand
  // sides: 337 us fused against 143 + 45 us)
  launch_b(k_prolong_add_b, red_grid_b(H, (int64_t)L.n * NB2), RED_THREADS, 0, st, L.n, (const int*)L.agg,
           (const double*)ec, H->opt.coarse_scale, cur, (const KrylovCtlB*)ctl);
  op_jacobi_b(H, l, b, cur, oth, want_dot && nu2 == 1, ctl, st, nu1);
  std::swap(cur, oth);
  for (int s = 1; s < nu2; ++s) {
    op_jacobi_b(H, l, b, cur, oth, want_dot && s == nu2 - 1, ctl, st, nu1 + s);
    std::swap(cur, oth);
  }
  *out = cur;
  AMG_CUDA_TRY(H, cudaGetLastError());
  return AMG_OK;
}

amg_status enqueue_start_b(amg_handle_s* H, cudaStream_t st) {
  AmgBatch& Bt = *H->batch;
  double* z = nullptr;
  AMG_TRY(vcycle_b(H, 0, Bt.kv[1], &z, Bt.ctl, true, st));
  const int n = H->lv[0].n;
  launch_b(k_pcg_p_b, red_grid_b(H, (int64_t)n * NB2), RED_THREADS, 0, st, n, (const double*)z, Bt.kv[2],
           (const KrylovCtlB*)Bt.ctl, (cudaGraphConditionalHandle)0);
  AMG_CUDA_TRY(H, cudaGetLastError());
  return AMG_OK;
}

amg_status enqueue_iteration_b(amg_handle_s* H, cudaStream_t st) {
  AmgBatch& Bt = *H->batch;
  Level& L0 = H->lv[0];
  const int n = L0.n;
  double *x = Bt.kv[0], *r = Bt.kv[1], *p = Bt.kv[2], *q = Bt.kv[3];
  const bool l0_dense = H->tail_dense_level == 0;
  if (l0_dense) {
    H->err = "internal: batched solve on a hierarchy whose level 0 is the dense tail";
    return AMG_ERR_UNSUPPORTED;
  }
  {
    RowArgsB a = args_b(Bt.ctl);
    a.x = p, a.out = q, a.fin = FIN_PQ;
    if (L0.K.fast)  // mixed-precision hierarchy: the Krylov operator stays fp64
      launch_rowtile_b<OP_SPMV, 1>(H, L0, Bt.geomK, a, st, &L0.K);
    else
      launch_rowtile_b<OP_SPMV, 1>(H, L0, Bt.geom[0], a, st);
  }
  launch_b(k_pcg_xr_b, red_grid_b(H, (int64_t)n * NB2), RED_THREADS, 0, st, n, (const double*)p, (const double*)q, x, r,
           (const double*)L0.dsw[0], Bt.x2[0], Bt.partials, Bt.counter, Bt.ctl);
  double* z = nullptr;
  AMG_TRY(vcycle_b(H, 0, r, &z, Bt.ctl, true, st));
  launch_b(k_pcg_p_b, red_grid_b(H, (int64_t)n * NB2), RED_THREADS, 0, st, n, (const double*)z, p,
           (const KrylovCtlB*)Bt.ctl, gb_loop);
  AMG_CUDA_TRY(H, cudaGetLastError());
  return AMG_OK;
}

amg_status capture_b(amg_handle_s* H, bool start, cudaGraphExec_t* out, int64_t* nl) {
  if (!H->cap_stream) AMG_CUDA_TRY(H, cudaStreamCreateWithFlags(&H->cap_stream, cudaStreamNonBlocking));
  AMG_CUDA_TRY(H, cudaStreamBeginCapture(H->cap_stream, cudaStreamCaptureModeThreadLocal));
  const int64_t l0 = gb_nlaunch;
  gb_pdl = H->opt.use_pdl != 0;
  const amg_status s = start ? enqueue_start_b(H, H->cap_stream) : enqueue_iteration_b(H, H->cap_stream);
  gb_pdl = false;
  *nl = gb_nlaunch - l0;
  gb_nlaunch = l0;
  cudaGraph_t g = nullptr;
  cudaError_t e = cudaStreamEndCapture(H->cap_stream, &g);
  if (s != AMG_OK) {
    if (g) cudaGraphDestroy(g);
    return s;
  }
  AMG_CUDA_TRY(H, e);
  e = cudaGraphInstantiate(out, g, 0);
  cudaGraphDestroy(g);
  AMG_CUDA_TRY(H, e);
  return AMG_OK;
}

// the whole loop as one graph: conditional WHILE node, body = one batched iteration (see get_while_graph)
bool capture_while_b(amg_handle_s* H, cudaGraphExec_t* out) {
  if (!H->cap_stream && cudaStreamCreateWithFlags(&H->cap_stream, cudaStreamNonBlocking) != cudaSuccess) return false;
  cudaGraph_t g = nullptr;
  bool ok = cudaGraphCreate(&g, 0) == cudaSuccess;
  cudaGraphConditionalHandle hd = 0;
  ok = ok && cudaGraphConditionalHandleCreate(&hd, g, 1, cudaGraphCondAssignDefault) == cudaSuccess;
  cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
  np.conditional.handle = hd;
  np.conditional.type = cudaGraphCondTypeWhile;
  np.conditional.size = 1;
  cudaGraphNode_t node = nullptr;
  ok = ok && cudaGraphAddNode(&node, g, nullptr, 0, &np) == cudaSuccess;
  if (ok) {
    ok = cudaStreamBeginCaptureToGraph(H->cap_stream, np.conditional.phGraph_out[0], nullptr, nullptr, 0,
                                       cudaStreamCaptureModeThreadLocal) == cudaSuccess;
    if (ok) {
      const int64_t l0 = gb_nlaunch;
      gb_pdl = H->opt.use_pdl != 0;
      gb_loop = hd;
      const amg_status s = enqueue_iteration_b(H, H->cap_stream);
      gb_loop = 0;
      gb_pdl = false;
      gb_nlaunch = l0;
      cudaGraph_t cap = nullptr;
      ok = cudaStreamEndCapture(H->cap_stream, &cap) == cudaSuccess && s == AMG_OK;
    }
  }
  ok = ok && cudaGraphInstantiate(out, g, 0) == cudaSuccess;
  if (g) cudaGraphDestroy(g);
  if (!ok) cudaGetLastError();
  return ok;
}

}  // namespace

void amg_batch_release(amg_handle_s* H) {  // device memory is tracked by the handle (amg_free_all)
  AmgBatch* B = H->batch;
  if (!B) return;
  if (B->g_start) cudaGraphExecDestroy(B->g_start);
  if (B->g_iter) cudaGraphExecDestroy(B->g_iter);
  if (B->g_while) cudaGraphExecDestroy(B->g_while);
  for (auto& e : B->ev)
    if (e) cudaEventDestroy(e);
  if (B->h_ctl) cudaFreeHost(B->h_ctl);
  delete B;
  H->batch = nullptr;
}

// 1 if the batched kernels can run this hierarchy (work vectors, ring geometry and graphs are set up on
// the first call), 0 if amg_solve_batched has to loop over single solves
int amg_batch_prepare(amg_handle_s* H, cudaStream_t st) {
  if (!H->batch) H->batch = new AmgBatch;
  AmgBatch& B = *H->batch;
  if (B.eligible >= 0) return B.eligible;
  B.eligible = 0;
  const int D = H->tail_dense_level;
  if (!H->symmetric || H->opt.force_generic || D < 1 || H->opt.pre_sweeps < 1 || H->opt.post_sweeps < 1) return 0;
  for (int l = 0; l < D; ++l)
    if (!H->lv[l].fast) return 0;
  if (H->lv[0].v32 && !H->lv[0].K.fast) return 0;
  // ---- ring geometry per level from the tile descriptors ----
  B.geom.assign(D, LevelGeomB());
  std::vector<TileDesc> td;
  for (int l = -1; l < D; ++l) {  // l = -1: the fp64 blobs of level 0 of a mixed-precision hierarchy
    if (l < 0 && !H->lv[0].K.fast) continue;
    const Level& L = H->lv[l < 0 ? 0 : l];
    const int nblk = l < 0 ? L.K.nblk : L.nblk;
    td.resize(nblk);
    if (cudaMemcpyAsync(td.data(), l < 0 ? L.K.tiles : L.tiles, sizeof(TileDesc) * nblk, cudaMemcpyDeviceToHost, st) !=
            cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess)
      return 0;
    int sb = 0, xb = 0;
    for (const TileDesc& d : td) sb = std::max(sb, tpb_stage_need(d)), xb = std::max(xb, tpb_xslot_need(d));
    sb = (sb + 127) & ~127, xb = (xb + 127) & ~127;
    LevelGeomB& G = l < 0 ? B.geomK : B.geom[l];
    G.stage_bytes = sb, G.xslot_bytes = xb;
    const int smem_cap = (l >= 0 && L.ndict > 0) ? RTB_SMEM_MAX_VD : RTB_SMEM_MAX;
    for (int S = 3; S >= 2 && !G.stages; --S) {
      const int left = smem_cap - RTB_HEADER - S * sb;
      const int XS = left / xb > RTB_MAXS ? RTB_MAXS : left / xb;
      if (XS >= 2) G.stages = S, G.xslots = XS;
    }
    if (!G.stages) return 0;
    G.smem = RTB_HEADER + G.stages * sb + G.xslots * xb;
  }
  // ---- work vectors ----
  auto alloc = [&](size_t count) { return (double*)amg_dev_alloc(H, sizeof(double) * count, st); };
  B.x.assign(D + 1, nullptr), B.x2.assign(D + 1, nullptr), B.b.assign(D + 1, nullptr);
  for (int l = 0; l <= D; ++l) {
    const size_t m = (size_t)H->lv[l].n * NB;
    if (!(B.x[l] = alloc(m))) return 0;
    if (l < D && !(B.x2[l] = alloc(m))) return 0;
    if (l > 0 && !(B.b[l] = alloc(m))) return 0;
  }
  for (auto& v : B.kv)
    if (!(v = alloc((size_t)H->lv[0].n * NB))) return 0;
  B.partials_cap = std::max(H->sm_count * 8, 4096);
  if (!(B.partials = alloc((size_t)NB * B.partials_cap))) return 0;
  B.ctl = (KrylovCtlB*)amg_dev_alloc(H, sizeof(KrylovCtlB), st);
  B.counter = (unsigned*)amg_dev_alloc(H, sizeof(unsigned), st);
  if (!B.ctl || !B.counter) return 0;
  if (cudaMemsetAsync(B.counter, 0, sizeof(unsigned), st) != cudaSuccess) return 0;
  if (cudaMallocHost((void**)&B.h_ctl, sizeof(KrylovCtlB) * 6) != cudaSuccess) return 0;
  for (auto& e : B.ev)
    if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) return 0;
  set_attr_b<OP_SPMV, 1>(), set_attr_b<OP_JACOBI, 0>(), set_attr_b<OP_JACOBI, 1>(), set_attr_b<OP_RESTRICT, 0>();
  cudaGetLastError();
  B.eligible = 1;
  return 1;
}

// S10 / NEXT-3: ncols <= NB right-hand sides (columns ld apart, natural numbering) in one batched AMG-PCG solve
amg_status amg_solve_batch_chunk(amg_handle_s* H, const double* d_B, double* d_X, int ncols, int64_t ld, double rtol,
                                 int maxit, amg_info* infos, cudaStream_t st) {
  AmgBatch& B = *H->batch;
  Level& L0 = H->lv[0];
  const int n = L0.n;
  const int64_t launches0 = gb_nlaunch;
  CtlInit ci;
  ci.rtol = rtol, ci.maxit = maxit, ci.hist = nullptr, ci.hist_cap = 0;
  launch_b(k_krylov_init_b, red_grid_b(H, n), RED_THREADS, 0, st, n, ncols, ld, d_B, (const int*)L0.inv,
           (const double*)L0.dsw[0], B.kv[1], B.kv[0], B.x2[0], B.partials, B.counter, B.ctl, ci);
  AMG_CUDA_TRY(H, cudaGetLastError());
  const bool graph = H->opt.use_graph && maxit > 0;
  if (graph) {
    if (!B.g_start) AMG_TRY(capture_b(H, true, &B.g_start, &B.nl_start));
    if (!B.g_iter) AMG_TRY(capture_b(H, false, &B.g_iter, &B.nl_iter));
    AMG_CUDA_TRY(H, cudaGraphLaunch(B.g_start, st));
    gb_nlaunch += B.nl_start;
  } else if (maxit > 0) {
    AMG_TRY(enqueue_start_b(H, st));
  }
  bool looped = false;
  if (graph && H->opt.use_while && !B.while_failed) {
    if (!B.g_while && !capture_while_b(H, &B.g_while)) B.while_failed = true, B.g_while = nullptr;
    if (B.g_while) {
      AMG_CUDA_TRY(H, cudaGraphLaunch(B.g_while, st));
      looped = true;
    }
  }
  constexpr int NSLOT = 4, LAG = 1;
  for (int it = 0; it < maxit && !looped; ++it) {
    if (graph) {
      AMG_CUDA_TRY(H, cudaGraphLaunch(B.g_iter, st));
      gb_nlaunch += B.nl_iter;
    } else
      AMG_TRY(enqueue_iteration_b(H, st));
    const int slot = it % NSLOT;
    AMG_CUDA_TRY(H, cudaMemcpyAsync(&B.h_ctl[slot], B.ctl, sizeof(KrylovCtlB), cudaMemcpyDeviceToHost, st));
    AMG_CUDA_TRY(H, cudaEventRecord(B.ev[slot], st));
    if (it >= LAG) {
      const int old = (it - LAG) % NSLOT;
      AMG_CUDA_TRY(H, cudaEventSynchronize(B.ev[old]));
      if (B.h_ctl[old].all_done) break;
    }
  }
  launch_b(k_krylov_output_b, div_up(n, 256), 256, 0, st, n, ncols, ld, (const double*)B.kv[0], (const int*)L0.inv, d_X);
  AMG_CUDA_TRY(H, cudaGetLastError());
  H->last_launches += gb_nlaunch - launches0;
  if (!infos) return AMG_OK;
  AMG_CUDA_TRY(H, cudaMemcpyAsync(&B.h_ctl[4], B.ctl, sizeof(KrylovCtlB), cudaMemcpyDeviceToHost, st));
  AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
  if (looped) {  // kernels the device-side loop launched
    int itmax = 1;
    for (int s = 0; s < NB; ++s) itmax = std::max(itmax, B.h_ctl[4].c[s].iter);
    H->last_launches += (int64_t)itmax * B.nl_iter;
  }
  for (int s = 0; s < ncols; ++s) {
    const KrylovCtl& c = B.h_ctl[4].c[s];
    infos[s].iterations = c.iter;
    infos[s].status = c.status;
    infos[s].b_norm = sqrt(c.bnorm2);
    infos[s].rel_residual = c.bnorm2 > 0.0 ? sqrt(c.rr) / sqrt(c.bnorm2) : 0.0;
    if (c.status == AMG_MAXIT && c.iter == 0) infos[s].rel_residual = c.bnorm2 > 0.0 ? 1.0 : 0.0;
  }
  return AMG_OK;
}
