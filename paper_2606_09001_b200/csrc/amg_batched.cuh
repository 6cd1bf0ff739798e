// Batched multi-right-hand-side solve (NEXT-3; "the matrix is shared
// across the batch"): ONE pass over a level operator serves NB = 8 right-hand sides.  ~75 % of the
// bytes of a single-RHS iteration are the operator stream (4 M_l of 4 M_l + 13 V_l); with 8 vectors
// riding on one stream the per-RHS traffic drops to M/8 + vectors.
//
// Vectors are interleaved [row][NB] (64 contiguous bytes per row), so that the gather of a halo column
// fetches all 8 right-hand sides as two full 32-byte sectors, and a tile's rows of any vector are ONE
// contiguous range.  The row-tile kernel is the single-RHS one (amg_kernels.cuh) with
//   - the same tile blobs (one bulk-async copy per tile), nothing else of the operator;
//   - the tile's rows of b and x brought into the stage, and its rows of the result taken out of it, by
//     bulk-async copies / one bulk-async store; x slots [halo column][NB] for the halo only;
//   - 8 accumulators per row in registers, NB/2 LDS.128 per stored entry;
//   - one CTA per SM, 12 consumer warps, 8 gather warps in two groups;
//   - per-column Krylov scalars and convergence flags (KrylovCtlB): a converged column keeps riding
//     with alpha = beta = 0 (its x, r stay as they are) until every column is done.
// The operations with two gathers per column are split: the first sweep from zero (x1 = dinv o r) is
// emitted by the kernel that produces r (level 0) or by the restriction above (other levels), as in the
// single-RHS path, and the coarse correction is its own pass (k_prolong_add_b).
#pragma once
#include "amg_kernels.cuh"

constexpr int NB = 8;        // right-hand sides per batch
constexpr int NB2 = NB / 2;  // double2 per row
constexpr int RTB_CONSUMERS = 384;  // 12 warps walk the slices (672 threads per CTA leave 96 registers per thread: no spills;
                                    // measured on cfg 3 / cfg 4, 8 right-hand sides: 8 warps 33.8 / 155.6 ms, 12: 32.7 / 150.4, 16: 35.3 / 161.1)
constexpr int RTB_GATHERERS = 256;  // 8 warps in RTB_GGROUPS groups: they fetch the halo columns only
constexpr int RTB_GGROUPS = 2;
constexpr int RTB_THREADS = RTB_CONSUMERS + 32 + RTB_GATHERERS;
constexpr int RTB_GU = 12;          // columns per gather thread whose indices are held in registers
constexpr int RTB_MAXS = 4;         // most ring stages / x slots
constexpr int RTB_HEADER = 256;
constexpr int RTB_SMEM_MAX = 224 * 1024;  // dynamic part: the reductions keep ~2.5 KB of static shared memory ...
constexpr int RTB_SMEM_MAX_VD = 222 * 1024;  // ... and the value dictionary of a level stored as 8-bit codes 2 KB more

struct KrylovCtlB {
  KrylovCtl c[NB];
  int all_done, pad0, pad1, pad2;
};

struct RowArgsB {
  int n;
  const TileDesc* tiles;
  int ntiles;
  const unsigned char* blob;
  const int* halo_idx;
  const double* x;       // gathered vector, [n][NB]
  const double* b;
  const double* dinv;    // [n]
  double* out;
  const double* dinv_c;  // restriction, optional: smoother diagonal of the coarse level ...
  double* out2;          // ... then out2[I][s] = dinv_c[I] * out[I][s]
  const int* agg_ptr;
  const double* vdict;   // value dictionary of the level ([256]; tiles with vb = 1 hold 8-bit codes), or null
  double* partials;      // [NB][gridDim.x]
  unsigned* counter;
  KrylovCtlB* ctl;       // may be null (hooks)
  int fin;
  int stages, xslots, stage_bytes, xslot_bytes;  // shared-memory ring geometry (host: fits RTB_SMEM_MAX)
};

// ---- placement of a tile inside its ring stage (after the TP_DESC_BYTES header); blob at 0 ----
// Every operation keeps a ROW BUFFER [nr][NB] in the stage (64 bytes per row, the layout the vectors
// have in global memory): the tile's rows of b arrive in it by one bulk-async copy, the result of a
// row overwrites its b in place, and the finished tile leaves by one bulk-async store.
struct StageLayoutB {
  int ra2, nrv;  // dinv slice (even start / count)
  int Ia4, nap;  // agg_ptr slice
  int Ia2, nec;  // dinv_c slice
  int o_d, o_agg, o_dc, o_row, o_xown, end;
};
enum { TPB_D = 1, TPB_RESTRICT = 2 };
__host__ __device__ inline StageLayoutB tpb_stage(const TileDesc& d, int flags) {
  StageLayoutB t;
  const BlobLayout p = tp_blob(d.nsl, d.nslots, d.vb);
  const int r1 = d.r0 + d.nr;
  t.ra2 = d.r0 & ~1;
  t.nrv = tp_up(r1 - t.ra2, 2);
  t.Ia4 = d.I0 & ~3;
  t.nap = tp_up(d.I0 + d.nA + 1 - t.Ia4, 4);
  t.Ia2 = d.I0 & ~1;
  t.nec = tp_up(d.I0 + d.nA - t.Ia2, 2);
  int o = p.end;
  t.o_d = o;
  if (flags & TPB_D) o += 8 * t.nrv;
  t.o_agg = o;
  if (flags & TPB_RESTRICT) o += 4 * t.nap;
  t.o_dc = o;
  if (flags & TPB_RESTRICT) o += 8 * t.nec;
  // both 128-byte aligned (stages and x slots are): the class of a column the packer orders a row's entries by
  // (amg_setup.cu, k_pack_tiles) is then the half of the 128-byte bank line its 64 bytes occupy
  o = tp_up(o, 128);
  t.o_row = o;
  o += tp_up(8 * NB * d.nr, 128);
  t.o_xown = o;  // the tile's own rows of x, [nr][NB]
  o += 8 * NB * d.nr;
  t.end = o;
  return t;
}
__host__ __device__ inline int tpb_stage_need(const TileDesc& d) {
  const int a = tpb_stage(d, TPB_D).end, b = tpb_stage(d, TPB_RESTRICT).end;
  return TP_DESC_BYTES + (a > b ? a : b);
}
// x slot: the tile's halo columns, [nhalo][NB], 64 bytes per column (the own rows travel with the stage)
__host__ __device__ inline int tpb_xslot_need(const TileDesc& d) { return 8 * NB * (d.nhalo > 0 ? d.nhalo : 1); }

// ---- per-column finalisation of a reduction; a finished column is frozen ----
__device__ inline void krylov_finalize_b(KrylovCtlB* cb, int fin, const double* s0) {
  int all = 1;
#pragma unroll 1
  for (int s = 0; s < NB; ++s) {
    KrylovCtl& c = cb->c[s];
    if (!c.done) krylov_finalize(&c, fin, s0[s], 0.0);
    if (c.done) {  // no further update of x, r; p = z
      c.alpha = 0.0;
      c.beta = 0.0;
    }
    all &= c.done;
  }
  cb->all_done = all;
}

template <int THREADS>
__device__ __forceinline__ void grid_reduce_finalize_b(double (&v)[NB], double* partials, unsigned* counter,
                                                       KrylovCtlB* ctl, int fin) {
  __shared__ double sh[NB][THREADS / 32];
  __shared__ bool is_last;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
#pragma unroll
  for (int j = 0; j < NB; ++j) {
    double s = v[j];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) sh[j][w] = s;
  }
  __syncthreads();
  if (tid < NB) {
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < THREADS / 32; ++q) s += sh[tid][q];
    partials[(size_t)tid * gridDim.x + blockIdx.x] = s;
  }
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    unsigned t = atomicAdd(counter, 1u);
    is_last = (t == gridDim.x - 1);
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
#pragma unroll
  for (int j = 0; j < NB; ++j) {
    double s = 0.0;
    for (unsigned q = tid; q < gridDim.x; q += THREADS) s += __ldcg(partials + (size_t)j * gridDim.x + q);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) sh[j][w] = s;
  }
  __syncthreads();
  if (tid == 0) {
    double tot[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      double s = 0.0;
#pragma unroll
      for (int q = 0; q < THREADS / 32; ++q) s += sh[j][q];
      tot[j] = s;
    }
    *counter = 0;
    krylov_finalize_b(ctl, fin, tot);
  }
}

// The same reduction for a kernel in which only NW warps hold values (the consumer warps of the row-tile kernel):
// they leave their warp totals in `sh` inside their own branch (cta_partial_b), so that the NB accumulators are
// live in that branch only; every thread of the CTA then calls grid_finalize_b.
template <int NW>
__device__ __forceinline__ void cta_partial_b(const double (&v)[NB], double (*sh)[NW], int w, int lane) {
#pragma unroll
  for (int j = 0; j < NB; ++j) {
    double s = v[j];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) sh[j][w] = s;
  }
}
template <int THREADS, int NW>
__device__ __forceinline__ void grid_finalize_b(double (*shw)[NW], double* partials, unsigned* counter, KrylovCtlB* ctl,
                                                int fin) {
  __shared__ double sh[NB][THREADS / 32];
  __shared__ bool is_last;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  __syncthreads();
  if (tid < NB) {
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < NW; ++q) s += shw[tid][q];
    partials[(size_t)tid * gridDim.x + blockIdx.x] = s;
  }
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    unsigned t = atomicAdd(counter, 1u);
    is_last = (t == gridDim.x - 1);
  }
  __syncthreads();
  if (!is_last) return;
  __threadfence();
#pragma unroll 1
  for (int j = 0; j < NB; ++j) {
    double s = 0.0;
    for (unsigned q = tid; q < gridDim.x; q += THREADS) s += __ldcg(partials + (size_t)j * gridDim.x + q);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) sh[j][w] = s;
  }
  __syncthreads();
  if (tid == 0) {
    double tot[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      double s = 0.0;
#pragma unroll
      for (int q = 0; q < THREADS / 32; ++q) s += sh[j][q];
      tot[j] = s;
    }
    *counter = 0;
    krylov_finalize_b(ctl, fin, tot);
  }
}

// ------------------------------------------------------------------------------------------
// Batched row-tile kernel.  OP: OP_SPMV (dot: x.out per column), OP_JACOBI (dot: b.out), OP_RESTRICT.
// (The coarse correction x += gamma P e_c is its own pass, k_prolong_add_b: a prolongation-fused sweep needs
// two gathers per column and keeps the own rows off the bulk copies; measured slower on every level.)
//
// Everything contiguous moves by bulk-async copies (TMA), not through the load/store pipe, which
// is what bounds this kernel: the tile's blob, dinv / agg_ptr / dinv_c slices (setup data, issued
// before the grid dependency), its rows of b (into the stage's row buffer), its OWN rows of x (into
// the stage as well; the gather warps fetch the halo columns only, into the x slot) and its rows of
// the result (row buffer -> global, one bulk store per tile issued by the producer thread once every
// consumer warp has released the stage).
//
// Shared-memory layout of the vectors is the global one, [row or column][NB] = 64 bytes each.  A
// consumer lane reads the NB2 16-byte chunks of a column in the order h ^ rot, rot = (lane / 2) & 3:
// its accumulator pair h belongs to right-hand sides 2 (h ^ rot), 2 (h ^ rot) + 1.  The row buffers
// and x slots start on 128-byte lines, so a column's 64 bytes are the lower or the upper half of a
// line; the packer (amg_setup.cu, k_pack_tiles) stores a row's entries so that lane l reads a
// lower-half column at step k when (l ^ k) is even and an upper-half one when it is odd.  With the
// rotation every 16-byte bank group is then read by exactly 2 of the 16 lanes of a half-warp -- the
// minimum for a 128-bit access.
// ------------------------------------------------------------------------------------------
struct StageDescB {  // TP_DESC_BYTES at the start of a stage, written by the producer
  int r0, nr, I0, nA;
  int nsl, nhalo, roff, aoff;  // roff = r0 - ra2 (dinv slice), aoff = I0 - Ia4 (agg_ptr slice)
  int o_perm, o_col, o_val, o_d;
  int o_agg, o_row, o_dc, eoff;  // eoff = Ia2 (dcs[I - eoff] = dinv_c[I])
  int vb;                        // bytes per stored value (8, or 4 with the mixed-precision hierarchy)
  int o_xown;
  int pad[14];
};
static_assert(sizeof(StageDescB) == TP_DESC_BYTES, "stage header size");

// shared -> global bulk-async store; completion is tracked by the issuing thread's bulk async-group
__device__ __forceinline__ void bulk_s2g(void* dst, const void* src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read_all() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

// mode 0: header + every copy, all on `bar`;  mode 1: header + the setup data (blob, dinv, agg_ptr,
// dinv_c), on `bar` (issued before the grid dependency);  mode 2: the tile's rows of b and x only, on `bar`
template <int OP, bool STREAM>
__device__ __forceinline__ void tile_issue_b(const RowArgsB& a, const TileDesc& d, unsigned char* stage, uint64_t* bar,
                                             uint64_t pol, int mode) {
  constexpr bool SWEEP = (OP == OP_JACOBI);
  constexpr bool RES = (OP == OP_RESTRICT);
  constexpr bool HASB = (OP != OP_SPMV);
  const bool dc = RES && a.dinv_c != nullptr;
  const BlobLayout p = tp_blob(d.nsl, d.nslots, d.vb);
  const StageLayoutB t = tpb_stage(d, (SWEEP ? TPB_D : 0) | (RES ? TPB_RESTRICT : 0));
  if (mode != 2) {
    StageDescB sd;
    sd.r0 = d.r0, sd.nr = d.nr, sd.I0 = d.I0, sd.nA = d.nA;
    sd.nsl = d.nsl, sd.nhalo = d.nhalo, sd.roff = d.r0 - t.ra2, sd.aoff = d.I0 - t.Ia4;
    sd.o_perm = p.o_perm, sd.o_col = p.o_col, sd.o_val = p.o_val, sd.o_d = t.o_d;
    sd.o_agg = t.o_agg, sd.o_row = t.o_row, sd.o_dc = t.o_dc, sd.eoff = t.Ia2;
    sd.vb = d.vb, sd.o_xown = t.o_xown;
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
  const uint32_t rowbytes = 8u * NB * (uint32_t)d.nr;
  uint32_t bytes = 0;
  if (mode != 2) {
    bytes += (uint32_t)p.end;
    if (SWEEP) bytes += 8u * (uint32_t)t.nrv;
    if (RES) bytes += 4u * (uint32_t)t.nap;
    if (dc) bytes += 8u * (uint32_t)t.nec;
  }
  if (mode != 1) bytes += (HASB ? 2u : 1u) * rowbytes;
  mbar_arrive_expect_tx(bar, bytes);
  if (mode != 2) {
    bulk_g2s<STREAM>(base, a.blob + (size_t)d.blob16 * 16u, (uint32_t)p.end, bar, pol);
    if (SWEEP) bulk_g2s<false>(base + t.o_d, a.dinv + t.ra2, 8u * (uint32_t)t.nrv, bar, pol);
    if (RES) bulk_g2s<false>(base + t.o_agg, a.agg_ptr + t.Ia4, 4u * (uint32_t)t.nap, bar, pol);
    if (dc) bulk_g2s<false>(base + t.o_dc, a.dinv_c + t.Ia2, 8u * (uint32_t)t.nec, bar, pol);
  }
  if (mode != 1) {
    if (HASB) bulk_g2s<false>(base + t.o_row, a.b + (size_t)d.r0 * NB, rowbytes, bar, pol);
    bulk_g2s<false>(base + t.o_xown, a.x + (size_t)d.r0 * NB, rowbytes, bar, pol);
  }
}

// the finished rows of the tile in `stage` leave by one bulk store (producer thread)
__device__ __forceinline__ void tile_store_b(const RowArgsB& a, unsigned char* stage) {
  const StageDescB* sd = reinterpret_cast<const StageDescB*>(stage);
  if (sd->nr > 0)
    bulk_s2g(a.out + (size_t)sd->r0 * NB, stage + TP_DESC_BYTES + sd->o_row, 8u * NB * (uint32_t)sd->nr);
}

struct GTileB {
  int r0, nr, nhalo, hoff;
  __device__ __forceinline__ void load(const RowArgsB& a, int t_begin, int my, int it) {
    r0 = nr = nhalo = hoff = 0;
    if (it < my) {
      const TileDesc* d = a.tiles + RT_TILE(t_begin, it);
      r0 = __ldg(&d->r0), nr = __ldg(&d->nr), nhalo = __ldg(&d->nhalo), hoff = __ldg(&d->halo_off);
    }
  }
};

template <int OP, int NDOT, bool STREAM, bool VD>  // VD: the level is stored as 8-bit codes (every tile has vb = 1)
static __global__ void __launch_bounds__(RTB_THREADS, 1) k_rowtile_b(RowArgsB a) {
  extern __shared__ __align__(128) unsigned char smem[];
  uint64_t* full = reinterpret_cast<uint64_t*>(smem);
  uint64_t* empty = full + RTB_MAXS;
  uint64_t* resdone = empty + RTB_MAXS;
  uint64_t* pre = resdone + RTB_MAXS;  // setup data of the first ring stages, issued before the grid dependency
  uint64_t* xready = pre + RTB_MAXS;
  uint64_t* xempty = xready + RTB_MAXS;
  static_assert(6 * RTB_MAXS * 8 <= RTB_HEADER, "barrier header");
  static_assert(OP == OP_SPMV || OP == OP_JACOBI || OP == OP_RESTRICT, "operations of the batched kernel");
  constexpr bool STORE = (OP != OP_RESTRICT);          // the tile's rows of the result leave by a bulk store
  const int S = a.stages, XS = a.xslots;
  unsigned char* stage0 = smem + RTB_HEADER;
  unsigned char* xslot0 = stage0 + (size_t)S * a.stage_bytes;
  constexpr int NCW = RTB_CONSUMERS / 32, NGW = RTB_GATHERERS / 32, NG = RTB_GGROUPS;
  const int tid = threadIdx.x;
  const int t_begin = blockIdx.x;
  const int my = ((int)a.ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;  // this CTA's tiles
  const int npre = my < S ? my : S;
  // ---- before the grid dependency: nothing here reads what an earlier kernel of the solve wrote ----
  if (tid == 0) {
    for (int s = 0; s < S; ++s) {
      mbar_init(full + s, 1);
      mbar_init(empty + s, NCW);
      mbar_init(resdone + s, NCW);
      mbar_init(pre + s, 1);
    }
    for (int q = 0; q < XS; ++q) {
      mbar_init(xready + q, NGW / NG);
      mbar_init(xempty + q, NCW);
    }
    fence_mbar_init();
  }
  double* sdict = DictStore<VD>::get();  // value dictionary of the level (setup data)
  if (VD && tid < 256) sdict[tid] = __ldg(a.vdict + tid);
  __syncthreads();
  pdl_launch_dependents();
  const uint64_t pol = STREAM ? l2_policy_evict_first() : 0;
  if (tid == RTB_CONSUMERS)  // the first ring stages: operator blobs and setup vectors only
    for (int it = 0; it < npre; ++it)
      tile_issue_b<OP, STREAM>(a, a.tiles[RT_TILE(t_begin, it)], stage0 + (size_t)it * a.stage_bytes, pre + it, pol, 1);
  // gather warps: descriptor and halo column indices of their first tile
  constexpr int GS = RTB_GATHERERS / NG;  // threads of a group
  constexpr int CL = GS / NB2;            // column lanes of a group
  constexpr int GU = RTB_GU;
  const int gt = tid - (RTB_CONSUMERS + 32);
  const int g = gt % GS, gg = gt / GS;
  const int sub = g & (NB2 - 1), cl = g / NB2;
  const bool is_gather = tid >= RTB_CONSUMERS + 32;
  GTileB gc, gn;
  int src[GU];  // level index of this thread's halo columns
  gc.load(a, t_begin, my, is_gather ? gg : my);
  gn.load(a, t_begin, my, is_gather ? gg + NG : my);
  auto load_indices = [&](const GTileB& t, int (&si)[GU]) {
#pragma unroll
    for (int u = 0; u < GU; ++u) {
      const int c = cl + u * CL;
      si[u] = c < t.nhalo ? __ldg(a.halo_idx + t.hoff + c) : -1;
    }
  };
  if (is_gather) load_indices(gc, src);
  pdl_wait();
  if (a.ctl != nullptr && a.ctl->all_done) {
    if (tid == RTB_CONSUMERS)  // the copies in flight target this CTA's shared memory: let them land
      for (int it = 0; it < npre; ++it) mbar_wait(pre + it, 0);
    return;
  }
  __shared__ double shdot[NB][RTB_CONSUMERS / 32];  // warp totals of the fused dot products (consumer warps)
  const double2* x2g = reinterpret_cast<const double2*>(a.x);

  if (is_gather) {
    // ---------------- gather warps: x slots [halo column][NB], up to XS tiles ahead ----------------
    // every load of a tile is issued before the slot is waited for: a slot is busy for a store burst only
    int q = gg % XS, xk = gg / XS;  // slot and use count of the slot for tile `it` (no division in the loop)
    for (int it = gg; it < my; it += NG) {
      GTileB gnn;
      gnn.load(a, t_begin, my, it + 2 * NG);
      int srcn[GU];
      load_indices(gn, srcn);  // the next tile's indices travel while this tile is gathered
      double2 v[GU];
#pragma unroll
      for (int u = 0; u < GU; ++u) {
        v[u] = make_double2(0.0, 0.0);
        if (src[u] >= 0) v[u] = __ldg(x2g + (size_t)src[u] * NB2 + sub);
      }
      if (xk > 0) mbar_wait(xempty + q, (uint32_t)((xk - 1) & 1));
      double2* xc = reinterpret_cast<double2*>(xslot0 + (size_t)q * a.xslot_bytes) + sub;
#pragma unroll
      for (int u = 0; u < GU; ++u)
        if (src[u] >= 0) xc[(size_t)(cl + u * CL) * NB2] = v[u];
      for (int c = cl + GU * CL; c < gc.nhalo; c += CL)  // more halo columns than the index registers hold
        xc[(size_t)c * NB2] = __ldg(x2g + (size_t)__ldg(a.halo_idx + gc.hoff + c) * NB2 + sub);
      __syncwarp();
      if ((tid & 31) == 0) mbar_arrive(xready + q);
      gc = gn, gn = gnn;
#pragma unroll
      for (int u = 0; u < GU; ++u) src[u] = srcn[u];
      q += NG;
      while (q >= XS) q -= XS, ++xk;
    }
  } else if (tid >= RTB_CONSUMERS) {
    // ---------------- producer warp ----------------
    if (tid == RTB_CONSUMERS && my > 0) {
      for (int it = 0; it < npre; ++it)  // their setup data is already on the way: the rows of b
        tile_issue_b<OP, STREAM>(a, a.tiles[RT_TILE(t_begin, it)], stage0 + (size_t)it * a.stage_bytes, full + it, pol, 2);
      int s = 0, sk = 1;  // stage and use count of the stage for tile `it` (it = npre = S here if the loop runs)
      for (int it = npre; it < my; ++it) {
        const TileDesc d = a.tiles[RT_TILE(t_begin, it)];
        unsigned char* stage = stage0 + (size_t)s * a.stage_bytes;
        mbar_wait(empty + s, (uint32_t)((sk - 1) & 1));  // every consumer warp is done with tile it - S
        if (STORE) {
          tile_store_b(a, stage);
          bulk_commit();
          bulk_wait_read_all();  // the store has read the row buffer: the stage may be overwritten
        }
        tile_issue_b<OP, STREAM>(a, d, stage, full + s, pol, 0);
        if (++s == S) s = 0, ++sk;
      }
      if (STORE) {
        // the tiles still in the ring: tile `it` is use number it / S of stage it % S
        int it = my > S ? my - S : 0;
        int s2 = it % S, k2 = it / S;
        for (; it < my; ++it) {
          mbar_wait(empty + s2, (uint32_t)(k2 & 1));
          tile_store_b(a, stage0 + (size_t)s2 * a.stage_bytes);
          bulk_commit();
          if (++s2 == S) s2 = 0, ++k2;
        }
        bulk_wait_all();
      }
    }
  } else {
    // ---------------- consumers ----------------
    const int lane = tid & 31, w = tid >> 5;
    const int rot = (lane >> 1) & (NB2 - 1);  // chunk rotation of this lane
    int o4[NB2];
#pragma unroll
    for (int h = 0; h < NB2; ++h) o4[h] = h ^ rot;
    constexpr int ND = NDOT > 0 ? NB : 1;
    double dots[ND];
#pragma unroll
    for (int j = 0; j < ND; ++j) dots[j] = 0.0;
    int sbase = 0;  // slices of the tiles so far: the round-robin deal continues across tiles
    int s = 0, q = 0;
    uint32_t par = 0, xpar = 0;  // phase parities of the stage / the x slot of tile `it`
    for (int it = 0; it < my; ++it) {
      unsigned char* stage = stage0 + (size_t)s * a.stage_bytes;
      if (it < S) mbar_wait(pre + s, 0);
      mbar_wait(full + s, par);           // the bulk copies have landed ...
      mbar_wait(xready + q, xpar);        // ... and the tile's x slot is assembled
      const StageDescB* sd = reinterpret_cast<const StageDescB*>(stage);
      const int nr = sd->nr, nsl = sd->nsl, r0 = sd->r0;
      if (nr > 0) {
        unsigned char* base = stage + TP_DESC_BYTES;
        const int2* slices = reinterpret_cast<const int2*>(base);
        const unsigned short* perm = reinterpret_cast<const unsigned short*>(base + sd->o_perm);
        const unsigned short* scol = reinterpret_cast<const unsigned short*>(base + sd->o_col) + lane;
        const double* sval = reinterpret_cast<const double*>(base + sd->o_val) + lane;
        const float* sval32 = reinterpret_cast<const float*>(base + sd->o_val) + lane;
        const uint32_t* scw = reinterpret_cast<const uint32_t*>(base + sd->o_col) + lane;  // column | code << 16
        const bool v32 = sd->vb == 4;
        constexpr bool v8 = VD;
        // tile-local column c: c < nr -> own row c (stage), else halo column c - nr (x slot); both [..][NB2]
        const double2* xown = reinterpret_cast<const double2*>(base + sd->o_xown);
        const double2* xhal = reinterpret_cast<const double2*>(xslot0 + (size_t)q * a.xslot_bytes) - (size_t)nr * NB2;
        const double* ds = reinterpret_cast<const double*>(base + sd->o_d) + sd->roff;
        double2* rowb = reinterpret_cast<double2*>(base + sd->o_row);  // [row][NB2]: b in, result out
        for (int j = (w >= sbase ? w - sbase : w - sbase + NCW); j < nsl; j += NCW) {
          const int2 sl = slices[j];
          const int lr = perm[j * 32 + lane];
          const bool valid = lr != 0xFFFF;
          const unsigned short* cp = scol + sl.x;
          const double* vp = sval + sl.x;
          const float* vp32 = sval32 + sl.x;
          const uint32_t* wp = scw + sl.x;
          double acc[NB];
#pragma unroll
          for (int t = 0; t < NB; ++t) acc[t] = 0.0;
#pragma unroll 2
          for (int k = 0; k < sl.y; ++k) {
            int c;
            double av;
            if (v8) {
              const uint32_t w = wp[k * 32];
              av = sdict[w >> 16], c = (int)(w & 0xFFFFu);
            } else {
              av = v32 ? (double)vp32[k * 32] : vp[k * 32], c = cp[k * 32];
            }
            const double2* xp = (c < nr ? xown : xhal) + (size_t)c * NB2;
#pragma unroll
            for (int h = 0; h < NB2; ++h) {
              const double2 xv = xp[o4[h]];
              acc[2 * h] += av * xv.x;
              acc[2 * h + 1] += av * xv.y;
            }
          }
          if (valid) {
            double2* rb = rowb + (size_t)lr * NB2;
            const double2* xo = xown + (size_t)lr * NB2;  // the row's own x
            if (OP == OP_RESTRICT) {
#pragma unroll
              for (int h = 0; h < NB2; ++h) {
                const double2 bv = rb[o4[h]];
                rb[o4[h]] = make_double2(bv.x - acc[2 * h], bv.y - acc[2 * h + 1]);
              }
            } else {
              const double di = (OP == OP_SPMV) ? 0.0 : ds[lr];
#pragma unroll
              for (int h = 0; h < NB2; ++h) {
                double2 o;
                const double2 xv = xo[o4[h]];
                if (OP == OP_SPMV) {
                  o = make_double2(acc[2 * h], acc[2 * h + 1]);
                  if (NDOT) dots[(2 * h) % ND] += xv.x * o.x, dots[(2 * h + 1) % ND] += xv.y * o.y;
                } else {
                  const double2 bv = rb[o4[h]];
                  o.x = xv.x + di * (bv.x - acc[2 * h]);
                  o.y = xv.y + di * (bv.y - acc[2 * h + 1]);
                  if (NDOT) dots[(2 * h) % ND] += bv.x * o.x, dots[(2 * h + 1) % ND] += bv.y * o.y;
                }
                rb[o4[h]] = o;
              }
            }
          }
        }
        if (OP == OP_RESTRICT) {
          // the rows of an aggregate are consecutive tile rows: all residuals of the tile first
          __syncwarp();
          if (lane == 0) mbar_arrive(resdone + s);
          mbar_wait(resdone + s, par);
          const int nA = sd->nA, I0 = sd->I0;
          const int* aps = reinterpret_cast<const int*>(base + sd->o_agg) + sd->aoff;      // aps[al] = agg_ptr[I0 + al]
          const double* dcs = reinterpret_cast<const double*>(base + sd->o_dc) - sd->eoff;  // dcs[I] = dinv_c[I]
          double2* o2g = reinterpret_cast<double2*>(a.out);
          double2* o22g = reinterpret_cast<double2*>(a.out2);
          for (int t = tid; t < nA * NB2; t += RTB_CONSUMERS) {
            const int al = t / NB2, h = t % NB2;
            double2 sum = make_double2(0.0, 0.0);
            for (int lr = aps[al] - r0, le = aps[al + 1] - r0; lr < le; ++lr) {
              const double2 rv = rowb[lr * NB2 + h];
              sum.x += rv.x, sum.y += rv.y;
            }
            o2g[(size_t)(I0 + al) * NB2 + h] = sum;
            if (a.out2 != nullptr) {
              const double dcv = dcs[I0 + al];
              o22g[(size_t)(I0 + al) * NB2 + h] = make_double2(dcv * sum.x, dcv * sum.y);
            }
          }
        }
      }
      sbase = (sbase + nsl) % NCW;
      // ---- this warp is done with the stage and the x slot: its writes to the row buffer become visible to
      // the async proxy (the bulk store reads them, the next bulk copy overwrites them) ----
      fence_proxy_async();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(empty + s);
        mbar_arrive(xempty + q);
      }
      if (++s == S) s = 0, par ^= 1u;
      if (++q == XS) q = 0, xpar ^= 1u;
    }
    if (NDOT > 0) {
      // this lane's accumulator pair h holds the right-hand sides 2 (h ^ rot), 2 (h ^ rot) + 1
      double dt[NB];
#pragma unroll
      for (int hh = 0; hh < NB2; ++hh) {
        dt[2 * hh] = dt[2 * hh + 1] = 0.0;
#pragma unroll
        for (int h = 0; h < NB2; ++h)
          if ((h ^ rot) == hh) dt[2 * hh] = dots[(2 * h) % ND], dt[2 * hh + 1] = dots[(2 * h + 1) % ND];
      }
      cta_partial_b<RTB_CONSUMERS / 32>(dt, shdot, w, lane);
    }
  }
  if (NDOT > 0) grid_finalize_b<RTB_THREADS, RTB_CONSUMERS / 32>(shdot, a.partials, a.counter, a.ctl, a.fin);
}

// ------------------------------------------------------------------------------------------
// Batched Krylov vector kernels (interleaved [row][NB] vectors, per-column scalars)
// ------------------------------------------------------------------------------------------
// r[i][s] = b_s[inv[i]] (columns >= ncols: 0), x = 0, x1 = dinv o r (first sweep of level 0 from zero);
// ||b_s||^2 per column
static __global__ void __launch_bounds__(RED_THREADS) k_krylov_init_b(int n, int ncols, int64_t ld,
                                                               const double* __restrict__ b_nat,
                                                               const int* __restrict__ inv,
                                                               const double* __restrict__ dinv, double* __restrict__ r,
                                                               double* __restrict__ x, double* __restrict__ x1,
                                                               double* partials, unsigned* counter, KrylovCtlB* ctl,
                                                               CtlInit ci) {
  if (blockIdx.x == 0 && threadIdx.x == 0) {  // loop control of every column (see k_krylov_init)
    for (int s = 0; s < NB; ++s) ci.apply(&ctl->c[s]);
    ctl->all_done = 0;
  }
  double acc[NB];
#pragma unroll
  for (int s = 0; s < NB; ++s) acc[s] = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * RED_THREADS) {
    const int src = inv[i];
    const double di = x1 ? dinv[i] : 0.0;
    double v[NB];
#pragma unroll
    for (int s = 0; s < NB; ++s) v[s] = s < ncols ? __ldg(b_nat + (size_t)s * ld + src) : 0.0;
    double2* r2 = reinterpret_cast<double2*>(r) + i * NB2;
    double2* x2 = reinterpret_cast<double2*>(x) + i * NB2;
#pragma unroll
    for (int h = 0; h < NB2; ++h) {
      r2[h] = make_double2(v[2 * h], v[2 * h + 1]);
      x2[h] = make_double2(0.0, 0.0);
      if (x1) reinterpret_cast<double2*>(x1)[i * NB2 + h] = make_double2(di * v[2 * h], di * v[2 * h + 1]);
      acc[2 * h] += v[2 * h] * v[2 * h];
      acc[2 * h + 1] += v[2 * h + 1] * v[2 * h + 1];
    }
  }
  grid_reduce_finalize_b<RED_THREADS>(acc, partials, counter, ctl, FIN_INIT_PCG);
}

// x += alpha_s p ; r -= alpha_s q ; ||r_s||^2 ; x1 = dinv o r (first sweep of the next V-cycle on level 0)
static __global__ void __launch_bounds__(RED_THREADS) k_pcg_xr_b(int n, const double* __restrict__ p,
                                                          const double* __restrict__ q, double* __restrict__ x,
                                                          double* __restrict__ r, const double* __restrict__ dinv,
                                                          double* __restrict__ x1, double* partials, unsigned* counter,
                                                          KrylovCtlB* ctl) {
  pdl_sync();
  if (ctl->all_done) return;
  // gridDim.x * RED_THREADS is a multiple of NB2: a thread keeps its pair of columns over the loop
  const int h = threadIdx.x & (NB2 - 1);
  const double a0 = ctl->c[2 * h].done ? 0.0 : ctl->c[2 * h].alpha;
  const double a1 = ctl->c[2 * h + 1].done ? 0.0 : ctl->c[2 * h + 1].alpha;
  double s0 = 0.0, s1 = 0.0;
  const int64_t m = (int64_t)n * NB2, stride = (int64_t)gridDim.x * RED_THREADS;
  const double2* p2 = reinterpret_cast<const double2*>(p);
  const double2* q2 = reinterpret_cast<const double2*>(q);
  double2* x2 = reinterpret_cast<double2*>(x);
  double2* r2 = reinterpret_cast<double2*>(r);
  double2* y2 = reinterpret_cast<double2*>(x1);
  for (int64_t t = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; t < m; t += stride) {
    const double2 pv = p2[t], qv = q2[t];
    double2 xv = x2[t], rv = r2[t];
    xv.x += a0 * pv.x, xv.y += a1 * pv.y;
    rv.x -= a0 * qv.x, rv.y -= a1 * qv.y;
    x2[t] = xv, r2[t] = rv;
    if (x1) {
      const double di = __ldg(dinv + t / NB2);
      y2[t] = make_double2(di * rv.x, di * rv.y);
    }
    s0 += rv.x * rv.x, s1 += rv.y * rv.y;
  }
  double acc[NB];
#pragma unroll
  for (int s = 0; s < NB; ++s) acc[s] = (s == 2 * h) ? s0 : ((s == 2 * h + 1) ? s1 : 0.0);
  grid_reduce_finalize_b<RED_THREADS>(acc, partials, counter, ctl, FIN_RR);
}

// p = z + beta_s p
static __global__ void __launch_bounds__(RED_THREADS) k_pcg_p_b(int n, const double* __restrict__ z, double* __restrict__ p,
                                                         const KrylovCtlB* ctl, cudaGraphConditionalHandle loop) {
  pdl_sync();
  // the last kernel of an iteration: inside a conditional WHILE node it sets the loop condition (0 = outside)
  if (loop != 0 && blockIdx.x == 0 && threadIdx.x == 0) cudaGraphSetConditional(loop, ctl->all_done ? 0u : 1u);
  if (ctl->all_done) return;
  const int h = threadIdx.x & (NB2 - 1);
  const double b0 = ctl->c[2 * h].beta, b1 = ctl->c[2 * h + 1].beta;
  const int64_t m = (int64_t)n * NB2, stride = (int64_t)gridDim.x * RED_THREADS;
  const double2* z2 = reinterpret_cast<const double2*>(z);
  double2* p2 = reinterpret_cast<double2*>(p);
  for (int64_t t = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; t < m; t += stride) {
    const double2 zv = z2[t];
    double2 pv = p2[t];
    // beta = 0 (first iteration, frozen column): p = z exactly, whatever the buffer held (it is not initialised)
    pv.x = b0 != 0.0 ? zv.x + b0 * pv.x : zv.x;
    pv.y = b1 != 0.0 ? zv.y + b1 * pv.y : zv.y;
    p2[t] = pv;
  }
}

// x[i][s] += gamma ec[agg[i]][s]: the coarse correction as its own unit-stride pass (large levels: the
// prolongation-fused sweep needs two gathers per column and assembles the own rows in the gather warps)
static __global__ void __launch_bounds__(RED_THREADS) k_prolong_add_b(int n, const int* __restrict__ agg,
                                                               const double* __restrict__ ec, double gamma,
                                                               double* __restrict__ x, const KrylovCtlB* ctl) {
  pdl_sync();
  if (ctl != nullptr && ctl->all_done) return;
  const int64_t m = (int64_t)n * NB2, stride = (int64_t)gridDim.x * RED_THREADS;
  const double2* e2 = reinterpret_cast<const double2*>(ec);
  double2* x2 = reinterpret_cast<double2*>(x);
  for (int64_t t = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; t < m; t += stride) {
    const int i = (int)(t / NB2), h = (int)(t % NB2);
    const double2 e = __ldg(e2 + (size_t)__ldg(agg + i) * NB2 + h);
    double2 v = x2[t];
    v.x += gamma * e.x, v.y += gamma * e.y;
    x2[t] = v;
  }
}

// x_nat column s (s < ncols), natural numbering
static __global__ void k_krylov_output_b(int n, int ncols, int64_t ld, const double* __restrict__ x,
                                  const int* __restrict__ inv, double* __restrict__ x_nat) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int dst = inv[i];
  const double2* x2 = reinterpret_cast<const double2*>(x) + i * NB2;
#pragma unroll
  for (int h = 0; h < NB2; ++h) {
    const double2 v = x2[h];
    if (2 * h < ncols) x_nat[(size_t)(2 * h) * ld + dst] = v.x;
    if (2 * h + 1 < ncols) x_nat[(size_t)(2 * h + 1) * ld + dst] = v.y;
  }
}

// interleave / de-interleave of a level vector batch for the hooks: nat[s * ld + inv[i]] <-> v[i][s]
static __global__ void k_permute_in_b(int n, int ncols, int64_t ld, const double* __restrict__ nat,
                               const int* __restrict__ inv, double* __restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int src = inv[i];
#pragma unroll
  for (int s = 0; s < NB; ++s) out[i * NB + s] = s < ncols ? nat[(size_t)s * ld + src] : 0.0;
}

// z[i][s] = sum_j B[i][j] b[j][s]: the dense collapsed tail for NB right-hand sides; one warp per row
struct TailArgsB {
  int n;
  const double* dense_B;
  const double* b;
  double* z;
  double* partials;
  unsigned* counter;
  KrylovCtlB* ctl;
  int fin;
};
constexpr int TAILB_T = 1024;
static __global__ void __launch_bounds__(TAILB_T, 1) k_dense_tail_b(TailArgsB a) {
  pdl_launch_dependents();
  const int G = gridDim.x, cta = blockIdx.x;
  const int i0 = (int)((int64_t)cta * a.n / G), i1 = (int)((int64_t)(cta + 1) * a.n / G);
  {
    const char* p0 = reinterpret_cast<const char*>(a.dense_B + (size_t)i0 * a.n);
    const size_t bytes = (size_t)(i1 - i0) * a.n * sizeof(double);
    for (size_t o = (size_t)threadIdx.x * 128; o < bytes; o += (size_t)TAILB_T * 128)
      asm volatile("prefetch.global.L2 [%0];" ::"l"(p0 + o));
  }
  pdl_wait();
  if (a.ctl != nullptr && a.ctl->all_done) return;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const double2* b2 = reinterpret_cast<const double2*>(a.b);
  double dots[NB];
#pragma unroll
  for (int s = 0; s < NB; ++s) dots[s] = 0.0;
  for (int i = i0 + w; i < i1; i += TAILB_T / 32) {
    const double* row = a.dense_B + (size_t)i * a.n;
    double acc[NB];
#pragma unroll
    for (int s = 0; s < NB; ++s) acc[s] = 0.0;
    for (int j = lane; j < a.n; j += 32) {
      const double v = __ldg(row + j);
#pragma unroll
      for (int h = 0; h < NB2; ++h) {
        const double2 bv = b2[(size_t)j * NB2 + h];
        acc[2 * h] += v * bv.x, acc[2 * h + 1] += v * bv.y;
      }
    }
#pragma unroll
    for (int s = 0; s < NB; ++s)
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) acc[s] += __shfl_xor_sync(0xffffffffu, acc[s], o);
    if (lane == 0) {
#pragma unroll
      for (int s = 0; s < NB; ++s) {
        a.z[(size_t)i * NB + s] = acc[s];
        if (a.fin != FIN_NONE) dots[s] += a.b[(size_t)i * NB + s] * acc[s];
      }
    }
  }
  if (a.fin != FIN_NONE) grid_reduce_finalize_b<TAILB_T>(dots, a.partials, a.counter, a.ctl, a.fin);
}
