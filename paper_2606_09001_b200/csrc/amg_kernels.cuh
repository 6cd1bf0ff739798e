// Solve-phase device code: the row-block streaming kernel family
// (SpMV / smoother / residual+restriction share one template), its row-vector fallback, the
// fused Krylov BLAS-1 kernels with device-side scalar updates, the dense LU solve.
#pragma once
#include "amg_internal.cuh"

// ------------------------------------------------------------------------------------------
// Programmatic dependent launch (PDL): a kernel launched with the programmatic-serialization
// attribute may become resident while its predecessor in the stream / graph is still draining.
// griddepcontrol.wait blocks until every prerequisite grid has completed and its writes are
// visible; without the attribute both instructions are no-ops.  Everything before pdl_wait()
// may only touch data no earlier kernel of the solve writes (tile descriptors, operator blobs).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_sync() {
  pdl_launch_dependents();
  pdl_wait();
}

// ------------------------------------------------------------------------------------------
// operations of the row kernels
// ------------------------------------------------------------------------------------------
enum RowOp {
  OP_SPMV = 0,            // out = A x                      dots: d0.out [, out.out]
  OP_JACOBI = 1,          // out = x + dinv o (b - A x)     dot: b.out
  OP_JACOBI0 = 2,         // two sweeps from a zero guess: x1 = dinv o b, out = x1 + dinv o (b - A x1)
  OP_RESID = 3,           // out = b - A x                  (fallback path; restriction is a second kernel)
  OP_RESTRICT = 4,        // out[I] = sum_{i in I} (b - A x)_i   (row-block path only)
  OP_JACOBI_PROLONG = 5,  // x~ = x + gamma * ec[agg];  out = x~ + dinv o (b - A x~)   dot: b.out
};

struct RowArgs {
  int n;
  const int* rowptr;
  const int* col;
  const double* val;
  const TileDesc* tiles;
  int ntiles;
  const double* x;      // gathered vector
  const double* b;
  const double* dinv;
  const double* dinv_x1; // OP_JACOBI0: diagonal of the first sweep from zero (x1 = dinv_x1 o b); = dinv unless the
                         // sweeps carry Chebyshev weights
  double* out;
  const double* dinv_c; // restriction, optional: smoother diagonal of the coarse level ...
  double* out2;         // ... then out2[I] = dinv_c[I] * out[I] (the first sweep of the coarse level from zero)
  const int* agg;       // prolongation / restriction
  const int* agg_ptr;
  const unsigned char* blob;  // tile-packed operator (row-tile kernels)
  const int* halo_idx;        // halo lists of the tiles
  const int* halo_cagg;
  const double* ec;
  double gamma;
  const double* d0;     // second operand of the fused dot (SpMV)
  double* partials;     // [ndot][gridDim.x]
  unsigned* counter;
  KrylovCtl* ctl;       // may be null (hooks)
  int fin;
  int v32;              // row-vector fallback: round every CSR value to fp32 on the fly (mixed-precision hierarchy)
  const double* vdict;  // value dictionary of the level ([256]; tiles with vb = 1 hold 8-bit codes into it), or null
};

// ------------------------------------------------------------------------------------------
// loads: the matrix stream of a level larger than L2 uses evict-first (ld.global.cs)
// ------------------------------------------------------------------------------------------
template <bool STREAM>
__device__ __forceinline__ int4 ld_i4(const int4* p) {
  return STREAM ? __ldcs(p) : __ldg(p);
}
template <bool STREAM>
__device__ __forceinline__ double2 ld_d2(const double2* p) {
  return STREAM ? __ldcs(p) : __ldg(p);
}

template <int OP>
__device__ __forceinline__ double gather_x(const RowArgs& a, int c) {
  if (OP == OP_JACOBI0) return __ldg(a.dinv_x1 + c) * __ldg(a.b + c);
  if (OP == OP_JACOBI_PROLONG) return __ldg(a.x + c) + a.gamma * __ldg(a.ec + __ldg(a.agg + c));
  return __ldg(a.x + c);
}

// row epilogue; returns the value written (for the fused dots)
template <int OP>
__device__ __forceinline__ double row_epilogue(const RowArgs& a, int i, double sum) {
  if (OP == OP_SPMV) return sum;
  if (OP == OP_RESID || OP == OP_RESTRICT) return a.b[i] - sum;
  const double di = a.dinv[i], bi = a.b[i];
  double xi;
  if (OP == OP_JACOBI0)
    xi = a.dinv_x1[i] * bi;
  else if (OP == OP_JACOBI_PROLONG)
    xi = a.x[i] + a.gamma * a.ec[a.agg[i]];
  else
    xi = a.x[i];
  return xi + di * (bi - sum);
}

// ------------------------------------------------------------------------------------------
// device-side finalisation of a reduction: Krylov scalars and loop control (S7-S9)
// ------------------------------------------------------------------------------------------
__device__ inline void krylov_finalize(KrylovCtl* c, int fin, double s0, double s1) {
  switch (fin) {
    case FIN_INIT_PCG:
    case FIN_INIT_BICG:
      c->bnorm2 = s0;
      c->rr = s0;
      c->iter = 0;
      c->first = 1;
      c->halfstep = 0;
      c->rho = 1.0;
      c->alpha = 1.0;
      c->omega = 1.0;
      c->beta = 0.0;
      c->status = AMG_MAXIT;
      c->done = 0;
      if (!isfinite(s0)) {
        c->status = AMG_NONFINITE;
        c->done = 1;
      } else if (s0 == 0.0) {
        c->status = AMG_CONVERGED;
        c->done = 1;
      } else if (c->maxit <= 0) {
        c->done = 1;
      } else if (fin == FIN_INIT_BICG) {  // rho_1 = rhat.r = ||b||^2 ; beta = (rho_1/rho)(alpha/omega)
        c->beta = s0;
        c->rho = s0;
      }
      break;
    case FIN_RZ:
      if (c->first) {
        c->beta = 0.0;
        c->first = 0;
      } else {
        c->beta = s0 / c->rho;
      }
      c->rho = s0;
      break;
    case FIN_PQ:
      c->sigma = s0;
      if (!(s0 > 0.0)) {
        c->status = isfinite(s0) ? AMG_BREAKDOWN : AMG_NONFINITE;
        c->done = 1;
      } else {
        c->alpha = c->rho / s0;
      }
      break;
    case FIN_RR: {
      c->iter += 1;
      c->rr = s0;
      double nr = sqrt(s0);
      if (c->hist != nullptr && c->iter <= c->hist_cap) c->hist[c->iter - 1] = nr / sqrt(c->bnorm2);
      if (!isfinite(nr)) {
        c->status = AMG_NONFINITE;
        c->done = 1;
      } else if (nr <= c->rtol * sqrt(c->bnorm2)) {
        c->status = AMG_CONVERGED;
        c->done = 1;
      } else if (c->iter >= c->maxit) {
        c->status = AMG_MAXIT;
        c->done = 1;
      }
    } break;
    case FIN_RV:
      c->rv = s0;
      if (s0 == 0.0 || !isfinite(s0)) {
        c->status = isfinite(s0) ? AMG_BREAKDOWN : AMG_NONFINITE;
        c->done = 1;
      } else {
        c->alpha = c->rho / s0;
      }
      break;
    case FIN_SS: {
      c->iter += 1;
      c->ss = s0;
      double ns = sqrt(s0);
      if (ns <= c->rtol * sqrt(c->bnorm2)) {  // half-step exit: x += alpha * phat in the output kernel
        if (c->hist != nullptr && c->iter <= c->hist_cap) c->hist[c->iter - 1] = ns / sqrt(c->bnorm2);
        c->rr = s0;
        c->status = AMG_CONVERGED;
        c->halfstep = 1;
        c->done = 1;
      }
    } break;
    case FIN_TS_TT:
      c->ts = s0;
      c->tt = s1;
      c->omega = s0 / s1;
      break;
    case FIN_RR_RHO: {
      c->rr = s0;
      double nr = sqrt(s0);
      if (c->hist != nullptr && c->iter <= c->hist_cap) c->hist[c->iter - 1] = nr / sqrt(c->bnorm2);
      if (!isfinite(nr)) {
        c->status = AMG_NONFINITE;
        c->done = 1;
      } else if (nr <= c->rtol * sqrt(c->bnorm2)) {
        c->status = AMG_CONVERGED;
        c->done = 1;
      } else if (c->omega == 0.0) {
        c->status = AMG_BREAKDOWN;
        c->done = 1;
      } else if (c->iter >= c->maxit) {
        c->status = AMG_MAXIT;
        c->done = 1;
      } else if (s1 == 0.0 || !isfinite(s1)) {
        c->status = isfinite(s1) ? AMG_BREAKDOWN : AMG_NONFINITE;
        c->done = 1;
      } else {
        c->beta = (s1 / c->rho) * (c->alpha / c->omega);
        c->rho = s1;
      }
    } break;
    default:
      break;
  }
}

// Block-level sum of NV values, then a grid-level sum by the last block to finish (ticket
// counter), in a fixed order: deterministic for a fixed launch configuration.  No float atomics.
template <int NV, int THREADS>
__device__ __forceinline__ void grid_reduce_finalize(double (&v)[NV], double* partials, unsigned* counter,
                                                     KrylovCtl* ctl, int fin) {
  __shared__ double sh[NV][THREADS / 32];
  __shared__ bool is_last;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    double s = v[j];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) sh[j][w] = s;
  }
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      double s = 0.0;
#pragma unroll
      for (int q = 0; q < THREADS / 32; ++q) s += sh[j][q];
      partials[(size_t)j * gridDim.x + blockIdx.x] = s;
    }
    __threadfence();
    unsigned t = atomicAdd(counter, 1u);
    is_last = (t == gridDim.x - 1);
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
  double tot[NV];
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    double s = 0.0;
    for (unsigned q = tid; q < gridDim.x; q += THREADS) s += __ldcg(partials + (size_t)j * gridDim.x + q);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) sh[j][w] = s;
  }
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int j = 0; j < NV; ++j) {
      double s = 0.0;
#pragma unroll
      for (int q = 0; q < THREADS / 32; ++q) s += sh[j][q];
      tot[j] = s;
    }
    *counter = 0;
    krylov_finalize(ctl, fin, tot[0], NV > 1 ? tot[NV - 1] : 0.0);
  }
}

// ------------------------------------------------------------------------------------------
// bulk-async copy (TMA, cp.async.bulk -> SASS UBLKCP) and mbarrier primitives
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// generic-proxy accesses to shared memory before this point are ordered before later async-proxy writes
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t addr = smem_u32(bar);
  uint32_t done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(addr), "r"(parity)
        : "memory");
  } while (!done);
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
// global -> shared, 16-byte aligned on both sides, bytes a multiple of 16; completion on `bar`
template <bool HINT>
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar, uint64_t pol) {
  if (HINT)
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
            smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol)
        : "memory");
  else
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ------------------------------------------------------------------------------------------
// Row-tile streaming kernel (S1-S4) over the sorted-ELL tile blobs (amg_tilepack.cuh).
// Persistent and warp-specialised: RT_CTAS CTAs per SM, tiles dealt round-robin to the CTAs;
// per CTA 8 consumer warps + 1 producer warp + 6 gather warps, a ring of RT_STAGES operator
// stages and a side ring of RT_XSLOTS x slots.
//
//   producer (1 thread)  waits for a stage's "empty", writes its header and issues the bulk-async
//                        copies (TMA) of the tile: its blob (one copy) and its slices of b, dinv
//                        / agg_ptr -> mbarrier "full"
//   gather warps         assemble the tile's x slot [x of its rows | x of its halo columns]: they
//                        read the tile descriptor and its halo list straight from global memory,
//                        gather once per distinct column (independent loads) and apply the per-row
//                        transform of the fused operations (x1 = dinv o b;  x~ = x + gamma
//                        ec[agg]) -> "xready".  They do not touch the operator ring, so they run
//                        up to RT_XSLOTS tiles ahead of the row walk: the gather latency is off the
//                        critical path of a stage (bulk copy -> row walk -> refill)
//   consumer warps       wait for "full" and "xready"; slices of 32 storage rows are dealt
//                        round-robin to the warps ACROSS tiles; one lane per row walks the slice's
//                        k-major slots: three shared-memory reads and one DFMA per entry, no
//                        divergence, no global gather, no row pointers; epilogue per row;
//                        -> "empty", "xempty"
//
// There is no CTA-wide barrier: HBM keeps streaming whatever the consumers are doing and warps
// drift across tiles (the round-robin deal balances them).  Only the restriction needs the tile's
// rows together (sum over an aggregate's rows): its consumers meet on one more mbarrier per tile.
// ------------------------------------------------------------------------------------------
namespace rt {
constexpr int HEADER_BYTES = 256;  // full / empty / resdone / pre [RT_STAGES], xready / xempty [RT_XSLOTS]
constexpr int SMEM_BYTES = HEADER_BYTES + RT_STAGES * RT_STAGE_BYTES + RT_XSLOTS * RT_XSLOT_BYTES;
constexpr int NCW = RT_CONSUMERS / 32;  // consumer warps
constexpr int NGW = RT_GATHERERS / 32;  // gather warps
static_assert(RT_STAGES >= 2 && (4 * RT_STAGES + 2 * RT_XSLOTS) * 8 <= HEADER_BYTES, "too many stages / slots");
static_assert(RT_STAGE_BYTES % 128 == 0 && RT_XSLOT_BYTES % 128 == 0, "stage / slot sizes must keep 128-byte alignment");
static_assert(SMEM_BYTES <= 227 * 1024, "tile ring exceeds shared memory");
static_assert((NCW & (NCW - 1)) == 0, "consumer warps must be a power of two");
static_assert(NGW % RT_GGROUPS == 0 && RT_XSLOTS >= 2 * RT_GGROUPS, "gather groups");
}  // namespace rt

struct StageDesc {  // TP_DESC_BYTES at the start of a stage, written by the producer
  int r0, nr, I0, nA;
  int nsl, nhalo, roff, aoff;    // roff = r0 - ra2 (b / dinv slices), aoff = I0 - Ia4 (agg_ptr slice)
  int o_perm, o_col, o_val, o_b;
  int o_d, o_agg, o_out, o_dc;
  int eoff, vb, pad2, pad3;      // eoff = Ia2 (coarse slice: dcs[I - eoff] = dinv_c[I]); vb = bytes per stored value
  int pad1[12];
};
static_assert(sizeof(StageDesc) == TP_DESC_BYTES, "stage header size");

// which operands of the tile are staged in the ring for which operation
template <int OP>
struct TileOps {
  static constexpr bool B = (OP != OP_SPMV);
  static constexpr bool D = (OP == OP_JACOBI || OP == OP_JACOBI0 || OP == OP_JACOBI_PROLONG);
  static constexpr bool AGGPTR = (OP == OP_RESTRICT);
  static constexpr int FLAGS = (B ? TP_B : 0) | (D ? TP_D : 0) | (AGGPTR ? TP_AGGPTR | TP_OUT : 0);
};

// mode 0: header + every copy, all on `bar`;  mode 1: header + the blob copy only, on `bar` (issued
// before the grid dependency: the blob is setup data);  mode 2: the vector slices only, on `bar`
template <int OP, int NDOT, bool STREAM>
__device__ __forceinline__ void tile_issue(const RowArgs& a, const TileDesc& d, unsigned char* stage, uint64_t* bar,
                                           uint64_t pol, int mode) {
  using T = TileOps<OP>;
  const bool d0_staged = (OP == OP_SPMV && NDOT > 0 && a.d0 != a.x);
  const bool dc = T::AGGPTR && a.dinv_c != nullptr;
  const int flags = T::FLAGS | (d0_staged ? TP_B : 0) | (dc ? TP_DC : 0);
  const BlobLayout p = tp_blob(d.nsl, d.nslots, d.vb);
  const StageLayout t = tp_stage(d, flags);
  if (mode != 2) {
    StageDesc sd;
    sd.r0 = d.r0, sd.nr = d.nr, sd.I0 = d.I0, sd.nA = d.nA;
    sd.nsl = d.nsl, sd.nhalo = d.nhalo, sd.roff = d.r0 - t.ra2, sd.aoff = d.I0 - t.Ia4;
    sd.o_perm = p.o_perm, sd.o_col = p.o_col, sd.o_val = p.o_val, sd.o_b = t.o_b;
    sd.o_d = t.o_d, sd.o_agg = t.o_agg, sd.o_out = t.o_out, sd.o_dc = t.o_dc;
    sd.eoff = t.Ia2, sd.vb = d.vb, sd.pad2 = sd.pad3 = 0;
    int4* dst = reinterpret_cast<int4*>(stage);
    const int4* src = reinterpret_cast<const int4*>(&sd);
#pragma unroll
    for (int q = 0; q < 5; ++q) dst[q] = src[q];
  }
  if (d.nr <= 0) {
    mbar_arrive(bar);
    return;
  }
  unsigned char* base = stage + TP_DESC_BYTES;
  const uint32_t nblob = (uint32_t)p.end;
  const uint32_t nrv8 = 8u * (uint32_t)t.nrv;
  const bool has_vec = T::B || d0_staged || T::D || T::AGGPTR;
  uint32_t bytes = 0;
  if (mode != 2) bytes += nblob;
  if (mode != 1) {
    if (T::B || d0_staged) bytes += nrv8;
    if (T::D) bytes += nrv8;
    if (T::AGGPTR) bytes += 4u * (uint32_t)t.nap;
    if (dc) bytes += 8u * (uint32_t)t.nec;
  }
  if (mode == 2 && !has_vec) {  // nothing but the blob is staged (SpMV without a second dot operand)
    mbar_arrive(bar);
    return;
  }
  mbar_arrive_expect_tx(bar, bytes);
  if (mode != 2) bulk_g2s<STREAM>(base, a.blob + (size_t)d.blob16 * 16u, nblob, bar, pol);
  if (mode != 1) {
    if (T::B) bulk_g2s<false>(base + t.o_b, a.b + t.ra2, nrv8, bar, pol);
    if (d0_staged) bulk_g2s<false>(base + t.o_b, a.d0 + t.ra2, nrv8, bar, pol);
    if (T::D) bulk_g2s<false>(base + t.o_d, a.dinv + t.ra2, nrv8, bar, pol);
    if (T::AGGPTR) bulk_g2s<false>(base + t.o_agg, a.agg_ptr + t.Ia4, 4u * (uint32_t)t.nap, bar, pol);
    if (dc) bulk_g2s<false>(base + t.o_dc, a.dinv_c + t.Ia2, 8u * (uint32_t)t.nec, bar, pol);
  }
}

// value of the gathered vector at index i of the level (the fused operations transform it on the fly)
template <int OP>
__device__ __forceinline__ double xvalue_local(const RowArgs& a, int i) {
  if (OP == OP_JACOBI0) return __ldg(a.dinv_x1 + i) * __ldg(a.b + i);
  if (OP == OP_JACOBI_PROLONG) return __ldg(a.x + i) + a.gamma * __ldg(a.ec + __ldg(a.agg + i));
  return __ldg(a.x + i);
}

// Tiles are dealt to the CTAs round-robin (tile = blockIdx.x + it * gridDim.x): at any moment the grid works
// on one window of consecutive tiles, so halo columns are in L2 and HBM is read as a few sequential streams
// (measured 1 % faster than one contiguous run of tiles per CTA).
#define RT_TILE(t0, it) ((t0) + (it) * (int)gridDim.x)
struct GTile {  // what the gather warps need of a tile descriptor
  int r0, nr, nhalo, hoff;
  __device__ __forceinline__ void load(const RowArgs& a, int t_begin, int my, int it) {
    r0 = nr = nhalo = hoff = 0;
    if (it < my) {
      const TileDesc* d = a.tiles + RT_TILE(t_begin, it);
      r0 = __ldg(&d->r0), nr = __ldg(&d->nr), nhalo = __ldg(&d->nhalo), hoff = __ldg(&d->halo_off);
    }
  }
};

// 256-entry value dictionary in static shared memory, only in the kernels that are instantiated for dictionary levels
template <bool ON>
struct DictStore {
  __device__ __forceinline__ static double* get() {
    __shared__ double s[256];
    return s;
  }
};
template <>
struct DictStore<false> {
  __device__ __forceinline__ static double* get() { return nullptr; }
};

template <int OP, int NDOT, bool STREAM, int GEO>
static __global__ void __launch_bounds__(RtGeo<GEO>::THREADS, RT_CTAS) k_rowtile(RowArgs a) {
  // ring geometry of this kind of level (the names shadow the fp64 geometry's constants)
  constexpr int RT_STAGES = RtGeo<GEO>::STAGES, RT_STAGE_BYTES = RtGeo<GEO>::STAGE_BYTES;
  constexpr int RT_XSLOTS = RtGeo<GEO>::XSLOTS, RT_XSLOT_BYTES = RtGeo<GEO>::XSLOT_BYTES;
  constexpr int RT_GATHER_UNROLL = RtGeo<GEO>::GATHER_UNROLL, RT_GATHER_ROWS = RtGeo<GEO>::GATHER_ROWS;
  constexpr int RT_CONSUMERS = RtGeo<GEO>::CONSUMERS, RT_GATHERERS = RtGeo<GEO>::GATHERERS, RT_THREADS = RtGeo<GEO>::THREADS;
  constexpr int NCW = RT_CONSUMERS / 32, NGW = RT_GATHERERS / 32;  // consumer / gather warps of this kind of level
  static_assert((NCW & (NCW - 1)) == 0 && NGW % RT_GGROUPS == 0, "consumer warps: a power of two; gather warps: whole groups");
  static_assert((4 * RT_STAGES + 2 * RT_XSLOTS) * 8 <= rt::HEADER_BYTES && RT_XSLOTS >= 2 * RT_GGROUPS, "ring header");
  static_assert(RT_STAGE_BYTES % 128 == 0 && RT_XSLOT_BYTES % 128 == 0, "stage / slot sizes must keep 128-byte alignment");
  extern __shared__ __align__(128) unsigned char smem[];
  uint64_t* full = reinterpret_cast<uint64_t*>(smem);
  uint64_t* empty = full + RT_STAGES;
  uint64_t* resdone = empty + RT_STAGES;
  uint64_t* pre = resdone + RT_STAGES;  // blobs of the first RT_STAGES tiles, issued before the grid dependency
  uint64_t* xready = pre + RT_STAGES;
  uint64_t* xempty = xready + RT_XSLOTS;
  unsigned char* stage0 = smem + rt::HEADER_BYTES;
  unsigned char* xslot0 = stage0 + RT_STAGES * RT_STAGE_BYTES;
  const int tid = threadIdx.x;
  const int t_begin = blockIdx.x;
  const int my = ((int)a.ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;  // this CTA's tiles
  const int npre = my < RT_STAGES ? my : RT_STAGES;
  const bool d0_staged = (OP == OP_SPMV && NDOT > 0 && a.d0 != a.x);
  // ---- before the grid dependency: nothing here reads what an earlier kernel of the solve wrote ----
  if (tid == 0) {
    for (int s = 0; s < RT_STAGES; ++s) {
      mbar_init(full + s, 1);
      mbar_init(empty + s, NCW);
      mbar_init(resdone + s, NCW);
      mbar_init(pre + s, 1);
    }
    for (int q = 0; q < RT_XSLOTS; ++q) {
      mbar_init(xready + q, NGW / RT_GGROUPS);
      mbar_init(xempty + q, NCW);
    }
    fence_mbar_init();
  }
  // value dictionary of the level (setup data; GEO 1 = levels stored as 8-bit codes: every tile has vb = 1)
  double* sdict = DictStore<GEO == 1>::get();
  if (GEO == 1 && tid < 256) sdict[tid] = __ldg(a.vdict + tid);
  __syncthreads();
  pdl_launch_dependents();
  const uint64_t pol = STREAM ? l2_policy_evict_first() : 0;
  if (tid == RT_CONSUMERS)
    for (int it = 0; it < npre; ++it)
      tile_issue<OP, NDOT, STREAM>(a, a.tiles[RT_TILE(t_begin, it)], stage0 + it * RT_STAGE_BYTES, pre + it, pol, 1);
  // gather warps: descriptors of their first two tiles and the halo indices of the first (setup data too)
  // The gather warps form RT_GGROUPS groups that take the tiles in turn: a group assembles a slot in
  // one memory round trip (HBM latency when the coarse vector is cold), and the groups overlap theirs.
  constexpr int NG = RT_GGROUPS, GU = RT_GATHER_UNROLL, GS = RT_GATHERERS / NG;
  const int g = (tid - (RT_CONSUMERS + 32)) % GS;  // lane of the group
  const int gg = (tid - (RT_CONSUMERS + 32)) / GS; // group
  constexpr int LU = RT_GATHER_ROWS;  // own rows per gather thread held in registers (more rows: fallback loop)
  GTile gc, gn;
  int idx[GU], cag[GU], la[LU];  // halo columns, their coarse indices, coarse indices of the tile's own rows
  gc.load(a, t_begin, my, tid >= RT_CONSUMERS + 32 ? gg : my);
  gn.load(a, t_begin, my, tid >= RT_CONSUMERS + 32 ? gg + NG : my);
  if (tid >= RT_CONSUMERS + 32) {
#pragma unroll
    for (int u = 0; u < GU; ++u) {
      const int h = g + u * GS;
      idx[u] = h < gc.nhalo ? __ldg(a.halo_idx + gc.hoff + h) : -1;
      if (OP == OP_JACOBI_PROLONG) cag[u] = h < gc.nhalo ? __ldg(a.halo_cagg + gc.hoff + h) : 0;
    }
    if (OP == OP_JACOBI_PROLONG) {
#pragma unroll
      for (int u = 0; u < LU; ++u) la[u] = (g + u * GS < gc.nr) ? __ldg(a.agg + gc.r0 + g + u * GS) : 0;
    }
  }
  pdl_wait();
  if (a.ctl != nullptr && a.ctl->done) {
    if (tid == RT_CONSUMERS)  // the copies in flight target this CTA's shared memory: let them land
      for (int it = 0; it < npre; ++it) mbar_wait(pre + it, 0);
    return;
  }
  double dots[NDOT > 0 ? NDOT : 1];
#pragma unroll
  for (int j = 0; j < (NDOT > 0 ? NDOT : 1); ++j) dots[j] = 0.0;

  if (tid >= RT_CONSUMERS + 32) {
    // ---------------- gather warps: x slots, up to RT_XSLOTS tiles ahead ----------------
    // software pipeline: while tile `it` is gathered, the halo indices of tile it+1 and the
    // descriptor of tile it+2 are already on their way
    for (int it = gg; it < my; it += NG) {
      const int q = it % RT_XSLOTS;
      GTile gnn;
      gnn.load(a, t_begin, my, it + 2 * NG);
      int idxn[GU], cagn[GU], lan[LU];
#pragma unroll
      for (int u = 0; u < GU; ++u) {
        const int h = g + u * GS;
        idxn[u] = h < gn.nhalo ? __ldg(a.halo_idx + gn.hoff + h) : -1;
        if (OP == OP_JACOBI_PROLONG) cagn[u] = h < gn.nhalo ? __ldg(a.halo_cagg + gn.hoff + h) : 0;
      }
      if (OP == OP_JACOBI_PROLONG) {
#pragma unroll
        for (int u = 0; u < LU; ++u) lan[u] = (g + u * GS < gn.nr) ? __ldg(a.agg + gn.r0 + g + u * GS) : 0;
      }
      // every load of the tile is issued before anything is consumed: the slot is assembled in two
      // memory round trips (one for the plain operations) however many rows and halo columns it has
      double v[GU], e[GU], lv[LU], le[LU];
#pragma unroll
      for (int u = 0; u < GU; ++u) {
        const int c = idx[u];
        v[u] = 0.0, e[u] = 0.0;
        if (c >= 0) {
          if (OP == OP_JACOBI_PROLONG) {
            v[u] = __ldg(a.x + c);
            e[u] = __ldg(a.ec + cag[u]);
          } else if (OP == OP_JACOBI0) {
            v[u] = __ldg(a.dinv_x1 + c);
            e[u] = __ldg(a.b + c);
          } else {
            v[u] = __ldg(a.x + c);
          }
        }
      }
#pragma unroll
      for (int u = 0; u < LU; ++u) {
        const int lr = g + u * GS;
        lv[u] = 0.0, le[u] = 0.0;
        if (lr < gc.nr) {
          const int i = gc.r0 + lr;
          if (OP == OP_JACOBI_PROLONG) {
            lv[u] = __ldg(a.x + i);
            le[u] = __ldg(a.ec + la[u]);
          } else if (OP == OP_JACOBI0) {
            lv[u] = __ldg(a.dinv_x1 + i);
            le[u] = __ldg(a.b + i);
          } else {
            lv[u] = __ldg(a.x + i);
          }
        }
      }
      if (it >= RT_XSLOTS) mbar_wait(xempty + q, (uint32_t)(((it / RT_XSLOTS) - 1) & 1));
      double* xc = reinterpret_cast<double*>(xslot0 + q * RT_XSLOT_BYTES);  // xc[col]: rows, then halo
      double* xh = xc + gc.nr;
#pragma unroll
      for (int u = 0; u < GU; ++u)
        if (idx[u] >= 0) {
          if (OP == OP_JACOBI_PROLONG)
            xh[g + u * GS] = v[u] + a.gamma * e[u];
          else if (OP == OP_JACOBI0)
            xh[g + u * GS] = v[u] * e[u];
          else
            xh[g + u * GS] = v[u];
        }
#pragma unroll
      for (int u = 0; u < LU; ++u) {
        const int lr = g + u * GS;
        if (lr < gc.nr) {
          if (OP == OP_JACOBI_PROLONG)
            xc[lr] = lv[u] + a.gamma * le[u];
          else if (OP == OP_JACOBI0)
            xc[lr] = lv[u] * le[u];
          else
            xc[lr] = lv[u];
        }
      }
      for (int lr = g + LU * GS; lr < gc.nr; lr += GS) xc[lr] = xvalue_local<OP>(a, gc.r0 + lr);  // more rows than registers
      for (int h = g + GU * GS; h < gc.nhalo; h += GS) {  // more halo columns than the index registers hold
        const int c = __ldg(a.halo_idx + gc.hoff + h);
        if (OP == OP_JACOBI_PROLONG)
          xh[h] = __ldg(a.x + c) + a.gamma * __ldg(a.ec + __ldg(a.halo_cagg + gc.hoff + h));
        else if (OP == OP_JACOBI0)
          xh[h] = __ldg(a.dinv_x1 + c) * __ldg(a.b + c);
        else
          xh[h] = __ldg(a.x + c);
      }
      __syncwarp();
      if ((tid & 31) == 0) mbar_arrive(xready + q);
      gc = gn, gn = gnn;
#pragma unroll
      for (int u = 0; u < GU; ++u) idx[u] = idxn[u], cag[u] = cagn[u];
      if (OP == OP_JACOBI_PROLONG) {
#pragma unroll
        for (int u = 0; u < LU; ++u) la[u] = lan[u];
      }
    }
  } else if (tid >= RT_CONSUMERS) {
    // ---------------- producer warp ----------------
    if (tid == RT_CONSUMERS && my > 0) {
      for (int it = 0; it < npre; ++it)  // their blobs are already on the way
        tile_issue<OP, NDOT, STREAM>(a, a.tiles[RT_TILE(t_begin, it)], stage0 + it * RT_STAGE_BYTES, full + it, pol, 2);
      for (int it = npre; it < my; ++it) {
        const int s = it % RT_STAGES;
        const TileDesc d = a.tiles[RT_TILE(t_begin, it)];
        mbar_wait(empty + s, (uint32_t)(((it / RT_STAGES) - 1) & 1));
        tile_issue<OP, NDOT, STREAM>(a, d, stage0 + s * RT_STAGE_BYTES, full + s, pol, 0);
      }
    }
  } else {
    // ---------------- consumers ----------------
    const int lane = tid & 31, w = tid >> 5;
    int sbase = 0;  // slices of the tiles so far: the round-robin deal continues across tiles
    for (int it = 0; it < my; ++it) {
      const int s = it % RT_STAGES, q = it % RT_XSLOTS;
      const uint32_t par = (uint32_t)((it / RT_STAGES) & 1);
      unsigned char* stage = stage0 + s * RT_STAGE_BYTES;
      if (it < RT_STAGES) mbar_wait(pre + s, 0);
      mbar_wait(full + s, par);                                      // the bulk copies have landed ...
      mbar_wait(xready + q, (uint32_t)((it / RT_XSLOTS) & 1));       // ... and the tile's x slot is assembled
      const StageDesc* sd = reinterpret_cast<const StageDesc*>(stage);
      const int nr = sd->nr, nsl = sd->nsl, r0 = sd->r0;
      if (nr > 0) {
        unsigned char* base = stage + TP_DESC_BYTES;
        const int2* slices = reinterpret_cast<const int2*>(base);
        const unsigned short* perm = reinterpret_cast<const unsigned short*>(base + sd->o_perm);
        const unsigned short* scol = reinterpret_cast<const unsigned short*>(base + sd->o_col) + lane;
        const double* sval = reinterpret_cast<const double*>(base + sd->o_val) + lane;
        const float* sval32 = reinterpret_cast<const float*>(base + sd->o_val) + lane;  // mixed-precision hierarchy
        const uint32_t* scw = reinterpret_cast<const uint32_t*>(base + sd->o_col) + lane;  // value dictionary: column | code << 16
        const bool v32 = sd->vb == 4;
        constexpr bool v8 = (GEO == 1);
        const double* xc = reinterpret_cast<const double*>(xslot0 + q * RT_XSLOT_BYTES);
        const double* bs = reinterpret_cast<const double*>(base + sd->o_b) + sd->roff;
        const double* ds = reinterpret_cast<const double*>(base + sd->o_d) + sd->roff;
        double* outs = reinterpret_cast<double*>(base + sd->o_out);
        for (int j = (w - sbase) & (NCW - 1); j < nsl; j += NCW) {
          const int2 sl = slices[j];
          const unsigned short* cp = scol + sl.x;
          double sum = 0.0;
          if (v8) {  // 8-bit codes into the level's table of distinct fp64 values: the same values, bit for bit
            const uint32_t* wp = scw + sl.x;
#pragma unroll 4
            for (int k = 0; k < sl.y; ++k) {
              const uint32_t w = wp[k * 32];
              sum += sdict[w >> 16] * xc[w & 0xFFFFu];
            }
          } else if (v32) {  // values stored in fp32 (exactly representable), arithmetic in fp64
            const float* vp = sval32 + sl.x;
#pragma unroll 4
            for (int k = 0; k < sl.y; ++k) sum += (double)vp[k * 32] * xc[cp[k * 32]];
          } else {
            const double* vp = sval + sl.x;
#pragma unroll 4
            for (int k = 0; k < sl.y; ++k) sum += vp[k * 32] * xc[cp[k * 32]];
          }
          const int lr = perm[j * 32 + lane];
          if (lr != 0xFFFF) {
            if (OP == OP_RESTRICT) {
              outs[lr] = bs[lr] - sum;
            } else {
              double o;
              if (OP == OP_SPMV)
                o = sum;
              else
                o = xc[lr] + ds[lr] * (bs[lr] - sum);
              a.out[r0 + lr] = o;
              if (NDOT >= 1) dots[0] += (OP == OP_SPMV ? (d0_staged ? bs[lr] : xc[lr]) : bs[lr]) * o;
              if (NDOT >= 2) dots[1] += o * o;
            }
          }
        }
        if (OP == OP_RESTRICT) {
          // the rows of an aggregate are consecutive tile rows: all residuals of the tile first
          __syncwarp();
          if (lane == 0) mbar_arrive(resdone + s);
          mbar_wait(resdone + s, par);
          const int nA = sd->nA, I0 = sd->I0;
          const int* aps = reinterpret_cast<const int*>(base + sd->o_agg) + sd->aoff;  // aps[al] = agg_ptr[I0 + al]
          const double* dcs = reinterpret_cast<const double*>(base + sd->o_dc) - sd->eoff;  // dcs[I] = dinv_c[I]
          for (int al = tid; al < nA; al += RT_CONSUMERS) {
            double sum = 0.0;
            for (int lr = aps[al] - r0, le = aps[al + 1] - r0; lr < le; ++lr) sum += outs[lr];
            a.out[I0 + al] = sum;
            if (a.out2 != nullptr) a.out2[I0 + al] = dcs[I0 + al] * sum;
          }
        }
      }
      sbase = (sbase + nsl) & (NCW - 1);
      // ---- this warp is done with the stage and the x slot ----
      if (OP == OP_RESTRICT) fence_proxy_async();  // residuals were written into a region the next bulk copy overwrites
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(empty + s);
        mbar_arrive(xempty + q);
      }
    }
  }
  if (NDOT > 0) grid_reduce_finalize<(NDOT > 0 ? NDOT : 1), RT_THREADS>(dots, a.partials, a.counter, a.ctl, a.fin);
}

// ------------------------------------------------------------------------------------------
// Row-vector fallback: LPR lanes per row (any row length, any aggregate size).
// ------------------------------------------------------------------------------------------
template <int OP, int NDOT, int LPR>
static __global__ void __launch_bounds__(RB_THREADS) k_rowvec(RowArgs a) {
  pdl_sync();
  if (a.ctl != nullptr && a.ctl->done) return;
  const int tid = threadIdx.x;
  const int sub = tid & (LPR - 1);
  const int64_t row0 = ((int64_t)blockIdx.x * RB_THREADS + tid) / LPR;
  const int64_t rstride = (int64_t)gridDim.x * RB_THREADS / LPR;
  double dots[NDOT > 0 ? NDOT : 1];
#pragma unroll
  for (int j = 0; j < (NDOT > 0 ? NDOT : 1); ++j) dots[j] = 0.0;
  // every lane of a warp runs the same number of trips (shuffles need full participation)
  const int64_t nloop = (a.n + rstride - 1) / rstride;
  for (int64_t it = 0; it < nloop; ++it) {
    const int64_t i = row0 + it * rstride;
    double s = 0.0;
    if (i < a.n)
      for (int k = a.rowptr[i] + sub, e = a.rowptr[i + 1]; k < e; k += LPR)
        s += (a.v32 ? (double)(float)a.val[k] : a.val[k]) * gather_x<OP>(a, a.col[k]);
#pragma unroll
    for (int o = LPR / 2; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (i < a.n && sub == 0) {
      const double o = row_epilogue<OP>(a, (int)i, s);
      a.out[i] = o;
      if (NDOT >= 1) dots[0] += (OP == OP_SPMV ? a.d0[i] : a.b[i]) * o;
      if (NDOT >= 2) dots[1] += o * o;
    }
  }
  if (NDOT > 0) grid_reduce_finalize<(NDOT > 0 ? NDOT : 1), RB_THREADS>(dots, a.partials, a.counter, a.ctl, a.fin);
}

// restriction of a stored residual (fallback path): rc[I] = sum of r over the contiguous rows of I
static __global__ void k_restrict_rows(int nc, const int* __restrict__ agg_ptr, const double* __restrict__ r,
                                double* __restrict__ rc, const KrylovCtl* ctl) {
  pdl_sync();
  if (ctl != nullptr && ctl->done) return;
  int I = blockIdx.x * blockDim.x + threadIdx.x;
  if (I >= nc) return;
  double s = 0.0;
  for (int t = agg_ptr[I]; t < agg_ptr[I + 1]; ++t) s += r[t];
  rc[I] = s;
}

// S4 standalone: x_i += gamma * ec[agg_i]
static __global__ void k_prolong_add(int n, const int* __restrict__ agg, const double* __restrict__ ec, double gamma,
                              const double* xin, double* xout /* may be xin */, const KrylovCtl* ctl) {
  pdl_sync();
  if (ctl != nullptr && ctl->done) return;
  // two rows per thread and trip: 128-bit accesses of x, 64-bit of agg (all arrays are 16-byte aligned)
  const int n2 = n >> 1;
  const int2* agg2 = reinterpret_cast<const int2*>(agg);
  const double2* xi2 = reinterpret_cast<const double2*>(xin);
  double2* xo2 = reinterpret_cast<double2*>(xout);
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += gridDim.x * blockDim.x) {
    const int2 a = agg2[i];
    double2 v = xi2[i];
    v.x += gamma * ec[a.x];
    v.y += gamma * ec[a.y];
    xo2[i] = v;
  }
  if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) xout[n - 1] = xin[n - 1] + gamma * ec[agg[n - 1]];
}

static __global__ void k_scale_dinv(int n, const double* __restrict__ dinv, const double* __restrict__ b,
                             double* __restrict__ x, const KrylovCtl* ctl) {
  pdl_sync();
  if (ctl != nullptr && ctl->done) return;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) x[i] = dinv[i] * b[i];
}

static __global__ void k_zero(int n, double* __restrict__ x, const KrylovCtl* ctl) {
  pdl_sync();
  if (ctl != nullptr && ctl->done) return;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) x[i] = 0.0;
}

// ------------------------------------------------------------------------------------------
// S5: coarsest solve with the dense LU factors (one CTA; y in shared memory)
// ------------------------------------------------------------------------------------------
static __global__ void k_lu_solve(int n, const double* __restrict__ lu, const int* __restrict__ piv,
                           const double* __restrict__ b, double* __restrict__ x, const KrylovCtl* ctl) {
  pdl_sync();
  if (ctl != nullptr && ctl->done) return;
  extern __shared__ double y[];
  const int tid = threadIdx.x, T = blockDim.x;
  for (int i = tid; i < n; i += T) y[i] = b[i];
  __syncthreads();
  if (tid == 0)
    for (int k = 0; k < n; ++k) {
      int p = piv[k];
      if (p != k) {
        double t = y[k];
        y[k] = y[p];
        y[p] = t;
      }
    }
  __syncthreads();
  for (int k = 0; k < n - 1; ++k) {  // forward substitution, unit lower triangle
    const double yk = y[k];
    for (int i = k + 1 + tid; i < n; i += T) y[i] -= lu[(size_t)i * n + k] * yk;
    __syncthreads();
  }
  for (int i = n - 1; i >= 0; --i) {  // backward substitution
    if (tid == 0) y[i] = y[i] / lu[(size_t)i * n + i];
    __syncthreads();
    const double yi = y[i];
    for (int j = tid; j < i; j += T) y[j] -= lu[(size_t)j * n + i] * yi;
    __syncthreads();
  }
  for (int i = tid; i < n; i += T) x[i] = y[i];
}

// n <= LU_SMALL_MAX: the factors (row pitch n+1: conflict-free column reads) and y sit in shared
// memory and ONE warp runs both substitutions, lane i owning rows i, i+32, ...: no block-wide
// barrier inside the 2n dependent steps.  `sm` holds n*(n+1) + n doubles.
constexpr int LU_SMALL_MAX = 72;  // 72*73*8 + 72*8 bytes < 48 KB
template <bool CG>  // CG: b was written by other CTAs of this kernel (read through L2)
__device__ __forceinline__ void lu_solve_small_cta(int n, const double* __restrict__ lu, const int* __restrict__ piv,
                                                   const double* b, double* x, double* sm) {
  const int tid = threadIdx.x, T = blockDim.x, P = n + 1;
  double* y = sm + (size_t)n * P;
  for (int t = tid; t < n * n; t += T) sm[(t / n) * P + (t % n)] = __ldg(lu + t);
  for (int i = tid; i < n; i += T) y[i] = CG ? __ldcg(b + i) : b[i];
  __syncthreads();
  if (tid < 32) {
    const int lane = tid;
    if (lane == 0)
      for (int k = 0; k < n; ++k) {
        const int p = __ldg(piv + k);
        if (p != k) {
          const double t = y[k];
          y[k] = y[p];
          y[p] = t;
        }
      }
    __syncwarp();
    for (int k = 0; k < n - 1; ++k) {  // forward substitution, unit lower triangle
      const double yk = y[k];
      for (int i = lane; i < n; i += 32)
        if (i > k) y[i] -= sm[i * P + k] * yk;
      __syncwarp();
    }
    for (int i = n - 1; i >= 0; --i) {  // backward substitution
      const double yi = y[i] / sm[i * P + i];
      __syncwarp();
      if (lane == 0) y[i] = yi;
      for (int j = lane; j < i; j += 32) y[j] -= sm[j * P + i] * yi;
      __syncwarp();
    }
  }
  __syncthreads();
  for (int i = tid; i < n; i += T) x[i] = y[i];
}

static __global__ void __launch_bounds__(256) k_lu_solve_small(int n, const double* __restrict__ lu,
                                                        const int* __restrict__ piv, const double* __restrict__ b,
                                                        double* __restrict__ x, const KrylovCtl* ctl) {
  pdl_sync();
  if (ctl != nullptr && ctl->done) return;
  extern __shared__ double lu_sm[];
  lu_solve_small_cta<true>(n, lu, piv, b, x, lu_sm);
}

// rtol / maxit / residual-history buffer of one solve, handed to the init kernel by value
struct CtlInit {
  double rtol;
  double* hist;
  int maxit, hist_cap;
  __device__ __forceinline__ void apply(KrylovCtl* c) const {
    c->rtol = rtol, c->maxit = maxit, c->hist = hist, c->hist_cap = hist_cap;
    c->done = 0, c->status = AMG_MAXIT, c->iter = 0, c->halfstep = 0;
  }
};

// ------------------------------------------------------------------------------------------
// S7/S8: fused Krylov vector kernels (grid-stride, one pass each, scalars read from KrylovCtl)
// ------------------------------------------------------------------------------------------
// r = b (permuted in), x = 0, optional extra vectors zeroed / copied; ||b||^2
static __global__ void __launch_bounds__(RED_THREADS) k_krylov_init(int n, const double* __restrict__ b_nat,
                                                             const int* __restrict__ inv, double* __restrict__ r,
                                                             double* __restrict__ x, double* __restrict__ z0,
                                                             double* __restrict__ z1, double* __restrict__ rhat,
                                                             const double* __restrict__ dinv, double* __restrict__ x1,
                                                             double* partials, unsigned* counter, KrylovCtl* ctl,
                                                             int fin, CtlInit ci) {
  // loop control of this solve: written here (no host-to-device copy that a following call could race with);
  // ordered before the last block's finalisation by this block's fence + ticket in grid_reduce_finalize
  if (blockIdx.x == 0 && threadIdx.x == 0) ci.apply(ctl);
  double acc[1] = {0.0};
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * RED_THREADS) {
    const double v = b_nat[inv[i]];
    r[i] = v;
    if (x1) x1[i] = dinv[i] * v;  // first sweep from zero of the V-cycle this solve starts with (PCG: on r)
    x[i] = 0.0;
    if (z0) z0[i] = 0.0;
    if (z1) z1[i] = 0.0;
    if (rhat) rhat[i] = v;
    acc[0] += v * v;
  }
  grid_reduce_finalize<1, RED_THREADS>(acc, partials, counter, ctl, fin);
}

// p = z + beta p.  The last kernel of a PCG iteration: inside a conditional WHILE graph node it also sets the
// loop condition (continue while the solve is not done; `loop` = 0 outside such a graph)
static __global__ void __launch_bounds__(RED_THREADS) k_pcg_p(int n, const double* __restrict__ z, double* __restrict__ p,
                                                       const KrylovCtl* ctl, cudaGraphConditionalHandle loop) {
  pdl_sync();
  if (loop != 0 && blockIdx.x == 0 && threadIdx.x == 0) cudaGraphSetConditional(loop, ctl->done ? 0u : 1u);
  if (ctl->done) return;
  const double beta = ctl->beta;
  const int64_t n2 = n / 2, stride = (int64_t)gridDim.x * RED_THREADS;
  const double2* z2 = reinterpret_cast<const double2*>(z);
  double2* p2 = reinterpret_cast<double2*>(p);
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n2; i += stride) {
    const double2 a = z2[i];
    double2 b = p2[i];
    b.x = a.x + beta * b.x;
    b.y = a.y + beta * b.y;
    p2[i] = b;
  }
  if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) p[n - 1] = z[n - 1] + beta * p[n - 1];
}

// x += alpha p ; r -= alpha q ; ||r||^2
static __global__ void __launch_bounds__(RED_THREADS) k_pcg_xr(int n, const double* __restrict__ p,
                                                        const double* __restrict__ q, double* __restrict__ x,
                                                        double* __restrict__ r, const double* __restrict__ dinv,
                                                        double* __restrict__ x1, double* partials, unsigned* counter,
                                                        KrylovCtl* ctl) {
  pdl_sync();
  if (ctl->done) return;
  const double alpha = ctl->alpha;
  double acc[1] = {0.0};
  // x1 = dinv o r (optional): the first sweep from zero of the V-cycle that follows, so that its level-0 pair of
  // sweeps is a plain sweep on x1 (one gather per halo column instead of two)
  const double2* d2 = reinterpret_cast<const double2*>(dinv);
  double2* y2 = reinterpret_cast<double2*>(x1);
  // 128-bit accesses, two independent pairs per thread and trip (the work vectors are 16-byte aligned)
  const int64_t n2 = n / 2, stride = (int64_t)gridDim.x * RED_THREADS;
  const double2* p2 = reinterpret_cast<const double2*>(p);
  const double2* q2 = reinterpret_cast<const double2*>(q);
  double2* x2 = reinterpret_cast<double2*>(x);
  double2* r2 = reinterpret_cast<double2*>(r);
  int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x;
  for (; i + stride < n2; i += 2 * stride) {
    const double2 pa = p2[i], pb = p2[i + stride], qa = q2[i], qb = q2[i + stride];
    double2 xa = x2[i], xb = x2[i + stride], ra = r2[i], rb = r2[i + stride];
    xa.x += alpha * pa.x, xa.y += alpha * pa.y, xb.x += alpha * pb.x, xb.y += alpha * pb.y;
    ra.x -= alpha * qa.x, ra.y -= alpha * qa.y, rb.x -= alpha * qb.x, rb.y -= alpha * qb.y;
    x2[i] = xa, x2[i + stride] = xb, r2[i] = ra, r2[i + stride] = rb;
    if (x1) {
      const double2 da = d2[i], db = d2[i + stride];
      y2[i] = make_double2(da.x * ra.x, da.y * ra.y), y2[i + stride] = make_double2(db.x * rb.x, db.y * rb.y);
    }
    acc[0] += (ra.x * ra.x + ra.y * ra.y) + (rb.x * rb.x + rb.y * rb.y);
  }
  for (; i < n2; i += stride) {
    const double2 pa = p2[i], qa = q2[i];
    double2 xa = x2[i], ra = r2[i];
    xa.x += alpha * pa.x, xa.y += alpha * pa.y;
    ra.x -= alpha * qa.x, ra.y -= alpha * qa.y;
    x2[i] = xa, r2[i] = ra;
    if (x1) {
      const double2 da = d2[i];
      y2[i] = make_double2(da.x * ra.x, da.y * ra.y);
    }
    acc[0] += ra.x * ra.x + ra.y * ra.y;
  }
  if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
    x[n - 1] += alpha * p[n - 1];
    const double ri = r[n - 1] - alpha * q[n - 1];
    r[n - 1] = ri;
    if (x1) x1[n - 1] = dinv[n - 1] * ri;
    acc[0] += ri * ri;
  }
  grid_reduce_finalize<1, RED_THREADS>(acc, partials, counter, ctl, FIN_RR);
}

// sum a.b  (used when no smoother sweep can carry the r.z product)
static __global__ void __launch_bounds__(RED_THREADS) k_dot(int n, const double* __restrict__ a, const double* __restrict__ b,
                                                     double* partials, unsigned* counter, KrylovCtl* ctl, int fin) {
  pdl_sync();
  if (ctl->done) return;
  double acc[1] = {0.0};
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * RED_THREADS)
    acc[0] += a[i] * b[i];
  grid_reduce_finalize<1, RED_THREADS>(acc, partials, counter, ctl, fin);
}

// p = r + beta (p - omega v) ; optional x1 = dinv o p (first sweep from zero of the V-cycle on p)
static __global__ void __launch_bounds__(RED_THREADS) k_bicg_p(int n, const double* __restrict__ r,
                                                        const double* __restrict__ v, double* __restrict__ p,
                                                        const double* __restrict__ dinv, double* __restrict__ x1,
                                                        const KrylovCtl* ctl) {
  pdl_sync();
  if (ctl->done) return;
  const double beta = ctl->beta, omega = ctl->omega;
  const int64_t n2 = n / 2, stride = (int64_t)gridDim.x * RED_THREADS;  // 128-bit accesses
  const double2* r2 = reinterpret_cast<const double2*>(r);
  const double2* v2 = reinterpret_cast<const double2*>(v);
  const double2* d2 = reinterpret_cast<const double2*>(dinv);
  double2* p2 = reinterpret_cast<double2*>(p);
  double2* y2 = reinterpret_cast<double2*>(x1);
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n2; i += stride) {
    const double2 rv = r2[i], vv = v2[i];
    double2 pv = p2[i];
    pv.x = rv.x + beta * (pv.x - omega * vv.x), pv.y = rv.y + beta * (pv.y - omega * vv.y);
    p2[i] = pv;
    if (x1) {
      const double2 dv = d2[i];
      y2[i] = make_double2(dv.x * pv.x, dv.y * pv.y);
    }
  }
  if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
    const double pi = r[n - 1] + beta * (p[n - 1] - omega * v[n - 1]);
    p[n - 1] = pi;
    if (x1) x1[n - 1] = dinv[n - 1] * pi;
  }
}

// s = r - alpha v ; ||s||^2 ; optional x1 = dinv o s
static __global__ void __launch_bounds__(RED_THREADS) k_bicg_s(int n, const double* __restrict__ r,
                                                        const double* __restrict__ v, double* __restrict__ s,
                                                        const double* __restrict__ dinv, double* __restrict__ x1,
                                                        double* partials, unsigned* counter, KrylovCtl* ctl) {
  pdl_sync();
  if (ctl->done) return;
  const double alpha = ctl->alpha;
  double acc[1] = {0.0};
  const int64_t n2 = n / 2, stride = (int64_t)gridDim.x * RED_THREADS;
  const double2* r2 = reinterpret_cast<const double2*>(r);
  const double2* v2 = reinterpret_cast<const double2*>(v);
  const double2* d2 = reinterpret_cast<const double2*>(dinv);
  double2* s2 = reinterpret_cast<double2*>(s);
  double2* y2 = reinterpret_cast<double2*>(x1);
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n2; i += stride) {
    const double2 rv = r2[i], vv = v2[i];
    const double2 sv = make_double2(rv.x - alpha * vv.x, rv.y - alpha * vv.y);
    s2[i] = sv;
    if (x1) {
      const double2 dv = d2[i];
      y2[i] = make_double2(dv.x * sv.x, dv.y * sv.y);
    }
    acc[0] += sv.x * sv.x + sv.y * sv.y;
  }
  if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
    const double si = r[n - 1] - alpha * v[n - 1];
    s[n - 1] = si;
    if (x1) x1[n - 1] = dinv[n - 1] * si;
    acc[0] += si * si;
  }
  grid_reduce_finalize<1, RED_THREADS>(acc, partials, counter, ctl, FIN_SS);
}

// x += alpha phat + omega shat ; r = s - omega t ; ||r||^2 , rhat.r
static __global__ void __launch_bounds__(RED_THREADS) k_bicg_xr(int n, const double* __restrict__ ph,
                                                         const double* __restrict__ sh, const double* __restrict__ s,
                                                         const double* __restrict__ t, const double* __restrict__ rhat,
                                                         double* __restrict__ x, double* __restrict__ r,
                                                         double* partials, unsigned* counter, KrylovCtl* ctl) {
  pdl_sync();
  if (ctl->done) return;
  const double alpha = ctl->alpha, omega = ctl->omega;
  double acc[2] = {0.0, 0.0};
  const int64_t n2 = n / 2, stride = (int64_t)gridDim.x * RED_THREADS;
  const double2* ph2 = reinterpret_cast<const double2*>(ph);
  const double2* sh2 = reinterpret_cast<const double2*>(sh);
  const double2* s2 = reinterpret_cast<const double2*>(s);
  const double2* t2 = reinterpret_cast<const double2*>(t);
  const double2* rh2 = reinterpret_cast<const double2*>(rhat);
  double2* x2 = reinterpret_cast<double2*>(x);
  double2* r2 = reinterpret_cast<double2*>(r);
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n2; i += stride) {
    const double2 pv = ph2[i], hv = sh2[i], sv = s2[i], tv = t2[i], qv = rh2[i];
    double2 xv = x2[i];
    xv.x += alpha * pv.x + omega * hv.x, xv.y += alpha * pv.y + omega * hv.y;
    const double2 rv = make_double2(sv.x - omega * tv.x, sv.y - omega * tv.y);
    x2[i] = xv, r2[i] = rv;
    acc[0] += rv.x * rv.x + rv.y * rv.y;
    acc[1] += qv.x * rv.x + qv.y * rv.y;
  }
  if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {
    x[n - 1] += alpha * ph[n - 1] + omega * sh[n - 1];
    const double ri = s[n - 1] - omega * t[n - 1];
    r[n - 1] = ri;
    acc[0] += ri * ri;
    acc[1] += rhat[n - 1] * ri;
  }
  grid_reduce_finalize<2, RED_THREADS>(acc, partials, counter, ctl, FIN_RR_RHO);
}

// loop condition of a conditional WHILE graph node whose body is one Krylov iteration (BiCGSTAB: its last kernel
// finalises the convergence test itself, so the condition is set by this one-thread kernel after it)
static __global__ void k_while_ctl(const KrylovCtl* ctl, cudaGraphConditionalHandle loop) {
  pdl_sync();
  cudaGraphSetConditional(loop, ctl->done ? 0u : 1u);
}

// x_out (natural numbering) = x [+ alpha * phat after a BiCGSTAB half-step exit]
static __global__ void k_krylov_output(int n, const double* __restrict__ x, const double* __restrict__ ph,
                                const int* __restrict__ inv, double* __restrict__ x_nat, const KrylovCtl* ctl) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double v = x[i];
  if (ph != nullptr && ctl->halfstep) v += ctl->alpha * ph[i];
  x_nat[inv[i]] = v;
}

static __global__ void k_permute_in(int n, const double* __restrict__ nat, const int* __restrict__ inv,
                             double* __restrict__ out) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = nat[inv[i]];
}
static __global__ void k_permute_out(int n, const double* __restrict__ in, const int* __restrict__ inv,
                              double* __restrict__ nat) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) nat[inv[i]] = in[i];
}

// ------------------------------------------------------------------------------------------
// G2: gA[k] (+)= - sum_s lambda_s[i] x_s[col[k]]  on the natural pattern; LPR lanes per row
// ------------------------------------------------------------------------------------------
template <int LPR>
static __global__ void __launch_bounds__(256) k_grad_values(int n, const int* __restrict__ rowptr,
                                                     const int* __restrict__ col, const double* __restrict__ lam,
                                                     const double* __restrict__ x, int nrhs, int64_t ld,
                                                     double* __restrict__ gA, int accumulate) {
  const int64_t gt = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t i = gt / LPR;
  const int sub = (int)(gt % LPR);
  if (i >= n) return;
  for (int k = rowptr[i] + sub, e = rowptr[i + 1]; k < e; k += LPR) {
    const int j = col[k];
    double s = 0.0;
    for (int b = 0; b < nrhs; ++b) s += __ldg(lam + (size_t)b * ld + i) * __ldg(x + (size_t)b * ld + j);
    gA[k] = accumulate ? gA[k] - s : -s;
  }
}

// Single right-hand side, short rows: ONE thread per row, the row's entries in chunks of 8 whose loads are
// all issued before any is used (the lanes-per-row kernel above keeps one dependent chain rowptr -> col -> x ->
// store per thread and is bound by that latency: 1.7 TB/s; here a thread has up to 8 gathers in flight).
static __global__ void __launch_bounds__(256) k_grad_values_rows(int n, const int* __restrict__ rowptr,
                                                                 const int* __restrict__ col,
                                                                 const double* __restrict__ lam,
                                                                 const double* __restrict__ x, double* __restrict__ gA,
                                                                 int accumulate) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int k0 = __ldg(rowptr + i), k1 = __ldg(rowptr + i + 1);
  const double li = __ldg(lam + i);
  for (int k = k0; k < k1; k += 8) {
    int j[8];
    double xv[8], old[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) j[u] = k + u < k1 ? __ldg(col + k + u) : -1;
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      xv[u] = j[u] >= 0 ? __ldg(x + j[u]) : 0.0;
      old[u] = (accumulate && j[u] >= 0) ? gA[k + u] : 0.0;
    }
#pragma unroll
    for (int u = 0; u < 8; ++u)
      if (j[u] >= 0) gA[k + u] = old[u] - li * xv[u];
  }
}

// Single right-hand side, any row length: ONE lane per stored ENTRY.  A warp owns 32 consecutive rows, i.e. one
// contiguous run of entries; lane l keeps rowptr[i0 + l] and lambda[i0 + l], the row of an entry is found by a
// 5-step binary search over the lanes' row pointers (shuffles), its lambda by one more shuffle: col and gA are read
// and written fully coalesced, the only gather is x[col[k]], with 4 independent entries per lane in flight.
static __global__ void __launch_bounds__(256) k_grad_values_entries(int n, const int* __restrict__ rowptr,
                                                                    const int* __restrict__ col,
                                                                    const double* __restrict__ lam,
                                                                    const double* __restrict__ x,
                                                                    double* __restrict__ gA, int accumulate) {
  const int lane = threadIdx.x & 31;
  const int i0 = (blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 32;
  if (i0 >= n) return;  // whole warp
  const int il = min(i0 + lane, n - 1);
  const int rp = __ldg(rowptr + il);  // non-decreasing over the lanes (rows past n repeat the last row: never found)
  const double li = __ldg(lam + il);
  const int kb = __shfl_sync(0xffffffffu, rp, 0), ke = __ldg(rowptr + min(i0 + 32, n));
  constexpr int U = 4;
  for (int k = kb; k < ke; k += 32 * U) {
    int c[U], r[U];
    double xv[U], old[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int e = k + u * 32 + lane;
      c[u] = e < ke ? __ldg(col + e) : -1;
      int lo = 0;  // largest lane with rp <= e
#pragma unroll
      for (int st = 16; st > 0; st >>= 1) {
        const int v = __shfl_sync(0xffffffffu, rp, (lo + st) & 31);
        if (lo + st < 32 && v <= e) lo += st;
      }
      r[u] = lo;
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      xv[u] = c[u] >= 0 ? __ldg(x + c[u]) : 0.0;
      old[u] = (accumulate && c[u] >= 0) ? gA[k + u * 32 + lane] : 0.0;
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const double l = __shfl_sync(0xffffffffu, li, r[u]);
      if (c[u] >= 0) gA[k + u * 32 + lane] = old[u] - l * xv[u];
    }
  }
}

// Batched G2 (nrhs > 1).  With the right-hand sides stored one after the other, the gather
// x_s[col[k]] touches a different 32-byte sector for every s: 16 sectors per stored entry on the
// permuted systems (cfg 5: 14 ms, 170 GB/s).  X is therefore first interleaved to XT[j][s] (one
// coalesced pass), so that all nrhs values of a column are ONE contiguous gather; lambda_s[i] is
// unit-stride along the rows as it stands.
constexpr int GT_ROWS = 64;  // rows per CTA of the interleave kernel
static __global__ void __launch_bounds__(256) k_interleave_rhs(int n, int nrhs, int64_t ld, const double* __restrict__ X,
                                                        double* __restrict__ XT) {
  extern __shared__ double tile[];  // [nrhs][GT_ROWS + 1]
  const int i0 = blockIdx.x * GT_ROWS;
  for (int t = threadIdx.x; t < nrhs * GT_ROWS; t += blockDim.x) {
    const int s = t / GT_ROWS, r = t % GT_ROWS;
    if (i0 + r < n) tile[s * (GT_ROWS + 1) + r] = X[(size_t)s * ld + i0 + r];
  }
  __syncthreads();
  for (int t = threadIdx.x; t < nrhs * GT_ROWS; t += blockDim.x) {
    const int r = t / nrhs, s = t % nrhs;
    if (i0 + r < n) XT[(size_t)(i0 + r) * nrhs + s] = tile[s * (GT_ROWS + 1) + r];
  }
}

template <int LPR, int NR>  // NR > 0: nrhs known at compile time (registers for lambda); 0: generic
static __global__ void __launch_bounds__(256) k_grad_values_batched(int n, const int* __restrict__ rowptr,
                                                             const int* __restrict__ col,
                                                             const double* __restrict__ lam, int64_t ld,
                                                             const double* __restrict__ XT, int nrhs_rt,
                                                             double* __restrict__ gA, int accumulate) {
  const int64_t gt = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t i = gt / LPR;
  const int sub = (int)(gt % LPR);
  if (i >= n) return;
  const int nrhs = NR > 0 ? NR : nrhs_rt;
  double l[NR > 0 ? NR : 1];
  if (NR > 0) {
#pragma unroll
    for (int s = 0; s < NR; ++s) l[s] = __ldg(lam + (size_t)s * ld + i);
  }
  for (int k = rowptr[i] + sub, e = rowptr[i + 1]; k < e; k += LPR) {
    const double* xj = XT + (size_t)col[k] * nrhs;
    double acc = 0.0;
    if (NR > 0 && (NR % 2) == 0) {
      const double2* x2 = reinterpret_cast<const double2*>(xj);  // rows of XT are 16-byte aligned for even nrhs
#pragma unroll
      for (int s = 0; s < NR / 2; ++s) {
        const double2 v = __ldg(x2 + s);
        acc += l[2 * s] * v.x;
        acc += l[2 * s + 1] * v.y;
      }
    } else if (NR > 0) {
#pragma unroll
      for (int s = 0; s < NR; ++s) acc += l[s] * __ldg(xj + s);
    } else {
      for (int s = 0; s < nrhs; ++s) acc += __ldg(lam + (size_t)s * ld + i) * __ldg(xj + s);
    }
    gA[k] = accumulate ? gA[k] - acc : -acc;
  }
}

// Batched G2, NR = 8 or 16 right-hand sides, cooperative gather: G = NR / 2 lanes share one stored entry, lane j
// holds lambda of the right-hand sides 2j, 2j + 1 of its row and reads the 16 bytes [2j, 2j + 1] of XT[col[k]]:
// one entry is ONE coalesced 64- / 128-byte request (the lane-per-entry kernel above issues NR / 2 separate
// 16-byte loads of that line per lane: 8 x the tag lookups, which is what bounds it on randomly permuted
// systems); the products are summed over the G lanes by shuffles.  All loads of up to 8 entries of a row are
// issued before any is used.
template <int NR>
static __global__ void __launch_bounds__(256, 4) k_grad_values_coop(int n, const int* __restrict__ rowptr,
                                                                 const int* __restrict__ col,
                                                                 const double* __restrict__ lam, int64_t ld,
                                                                 const double* __restrict__ XT,
                                                                 double* __restrict__ gA, int accumulate) {
  constexpr int G = NR / 2;
  const int64_t gt = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t iw = gt / G;
  const int j = (int)(gt % G);
  const bool live = iw < n;
  const int i = live ? (int)iw : n - 1;
  const double l0 = __ldg(lam + (size_t)(2 * j) * ld + i), l1 = __ldg(lam + (size_t)(2 * j + 1) * ld + i);
  const int k0 = __ldg(rowptr + i), k1 = live ? __ldg(rowptr + i + 1) : k0;
  const double2* X2 = reinterpret_cast<const double2*>(XT);
  // the trip count is made uniform over the warp (the shuffles need every lane)
  int len = k1 - k0;
#pragma unroll
  for (int o = 16; o >= G; o >>= 1) len = max(len, __shfl_xor_sync(0xffffffffu, len, o));
  constexpr int U = 8;
  for (int kk = 0; kk < len; kk += U) {
    int c[U];
    double2 v[U];
    double old[U];
#pragma unroll
    for (int u = 0; u < U; ++u) c[u] = k0 + kk + u < k1 ? __ldg(col + k0 + kk + u) : -1;
#pragma unroll
    for (int u = 0; u < U; ++u) {
      v[u] = c[u] >= 0 ? __ldg(X2 + (size_t)c[u] * G + j) : make_double2(0.0, 0.0);
      old[u] = (accumulate && j == 0 && c[u] >= 0) ? gA[k0 + kk + u] : 0.0;
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      double acc = l0 * v[u].x;
      acc += l1 * v[u].y;
#pragma unroll
      for (int o = G / 2; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
      if (j == 0 && c[u] >= 0) gA[k0 + kk + u] = old[u] - acc;
    }
  }
}
