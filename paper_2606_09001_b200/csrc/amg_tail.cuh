// Coarse tail of the V-cycle (S2-S6 on the small levels): ONE persistent kernel runs every level
// from `first` down to the coarsest solve and back up.  The levels below ~64 k rows hold < 3 % of
// the V-cycle's bytes but three quarters of its kernel launches, and every pass over them is a
// chain of dependent memory round trips, not a bandwidth problem.  Three measures:
//
//  * the CTAs stay resident (one per SM) and the dependency between two passes is a grid-wide
//    barrier (one atomic arrival per CTA, one polled release flag) instead of a kernel boundary
//    (measured: such a phase costs MORE than a row-tile launch in the PDL-chained graph, so by
//    default only the third measure is active: tail_max_rows = tail_dense_rows);
//  * every CTA owns a FIXED contiguous chunk of each level's rows (cut on aggregate starts,
//    balanced by nonzeros) and copies its slice of that level's operator (rowptr / col / val /
//    dinv) into shared memory once, at kernel start, with bulk-async copies (TMA): the four passes
//    over a level then read the operator at shared-memory latency, and only the x gathers (values
//    written by other CTAs in the previous pass) go to L2;
//  * the levels with at most `tail_dense_rows` rows are not visited at all: the V-cycle from level
//    D down is a fixed linear operator z = B_D r, assembled once at setup as a dense matrix (by
//    running that V-cycle on the unit vectors) and applied as one dense matrix-vector product
//    spread over all CTAs -- 1 pass instead of 4 passes x 5 levels + the LU solve.
//
// Vectors written inside the kernel are read with ld.global.cg (L2): L1 is not coherent across
// CTAs.  No floating-point atomics: every sum has a fixed order for a fixed grid.
#pragma once
#include "amg_kernels.cuh"

constexpr int TAIL_THREADS = 1024;
constexpr int TAIL_MAX_LEVELS = 32;
#ifndef TAIL_POLL_NS
#define TAIL_POLL_NS 100
#endif
constexpr int TAIL_STAGE_BUDGET = 176 * 1024;  // shared memory for the staged operator chunks

struct TailLevel {
  int n, nc, nnz, lpr;
  const int* rowptr;
  const int* col;
  const double* val;
  const double* dinv;
  const int* agg;
  const int* agg_ptr;
  double* b;   // right-hand side buffer of this level (unused for the level the call starts at)
  double* x;
  double* x2;
  // staging of this level's chunks (same offsets in every CTA; -1: not staged, read through L1)
  int s_rp, s_col, s_val, s_dinv;
};

struct TailChunk {  // rows [R0, R1), nonzeros [K0, K1), aggregates [A0, A1) of one CTA on one level
  int R0, R1, K0, K1, A0, A1, pad0, pad1;
};

struct TailArgs {
  const TailLevel* lv;     // device array indexed by level
  const TailChunk* chunk;  // [level][gridDim.x]
  int first, last;         // first level of the call, coarsest level
  const double* b_first;   // right-hand side of level `first`
  int nu1, nu2;
  double gamma;
  int nL;
  const double* lu;
  const int* piv;
  int dense_level;         // -1: none; else levels >= dense_level are applied as dense_B
  const double* dense_B;   // [nD x nD] row-major
  unsigned long long* bar;  // [0] arrival counter, [16] release word, [32 + cta] generation flags (variant 0)
  double* partials;
  KrylovCtl* ctl;           // may be null (hooks)
  int fin;                  // FIN_RZ: b_first . result is reduced and finalised (first == 0 only)
  int lu_smem;              // bytes reserved at the start of dynamic shared memory for the LU solve
  unsigned long long* prof; // -DAMG_TAIL_PROFILE: CTA 0 stamps %globaltimer after every phase
};
#ifdef AMG_TAIL_PROFILE
#define TAIL_STAMP(a, slot)                                                         \
  do {                                                                              \
    if ((a).prof != nullptr && blockIdx.x == 0 && threadIdx.x == 0) {               \
      unsigned long long _t;                                                        \
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(_t));                        \
      (a).prof[(slot)] = _t;                                                        \
    }                                                                               \
  } while (0)
#else
#define TAIL_STAMP(a, slot) do { } while (0)
#endif

__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_u64(unsigned long long* p, unsigned long long v) {
  asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
// Grid barrier.  All CTAs of the grid are co-resident (grid <= number of SMs, one CTA each).
// Three variants were measured on B200 (cfg 3, 21 barriers per V-cycle at the time):
//   1 (default) one arrival counter + one polled release word, thread 0 of every CTA:   136 us per tail
//   2           the same with the lightest fences that still form a release / acquire pair: 135 us
//   0           per-CTA generation flags, warp 0 of every CTA polls all of them (no atomics): 172 us
// A barrier costs 3-5 us whichever way: 1.5-4 us of it is the arrival skew between the CTAs.
// SASS on sm_100a: st.release.gpu = MEMBAR.ALL.GPU + STG.STRONG; ld.relaxed.gpu = LDG.STRONG alone;
// fence.acq_rel.gpu = MEMBAR.ALL.GPU + CCTL.IVALL; __threadfence() = MEMBAR.SC.GPU + CCTL.IVALL;
// ld.acquire.gpu = LDG.STRONG + CCTL.IVALL (an L1 invalidation per poll).
#ifndef TAIL_BAR_VARIANT
#define TAIL_BAR_VARIANT 1
#endif
__device__ __forceinline__ void tail_grid_barrier(unsigned long long* flags, unsigned long long& gen) {
  __syncthreads();
#if TAIL_BAR_VARIANT == 0
  // per-CTA generation flags, warp 0 polls all of them
  if (threadIdx.x < 32) {
    gen += 1ULL;
    if (threadIdx.x == 0) st_release_u64(flags + 32 + blockIdx.x, gen);
    const unsigned G = gridDim.x;
    for (;;) {
      bool ok = true;
      for (unsigned q = threadIdx.x; q < G; q += 32) ok &= (ld_relaxed_u64(flags + 32 + q) >= gen);
      if (__all_sync(0xffffffffu, ok)) break;
    }
    asm volatile("fence.acq_rel.gpu;" ::: "memory");
  }
#elif TAIL_BAR_VARIANT == 1
  // one arrival counter (only grows: every launch performs whole barriers, so it stays a multiple
  // of gridDim.x) and one release word; thread 0 of every CTA arrives and polls
  if (threadIdx.x == 0) {
    const unsigned long long G = gridDim.x;
    __threadfence();
    const unsigned long long t = atomicAdd(flags, 1ULL);
    const unsigned long long g = t / G + 1ULL;
    if (t % G == G - 1ULL) {
      st_release_u64(flags + 16, g);
    } else {
      while (ld_acquire_u64(flags + 16) < g) {
      }
    }
    __threadfence();
  }
#else
  // as 1 with the lightest fences that are still a release / acquire pair
  if (threadIdx.x == 0) {
    const unsigned long long G = gridDim.x;
    unsigned long long t;
    asm volatile("atom.add.release.gpu.global.u64 %0, [%1], 1;" : "=l"(t) : "l"(flags) : "memory");
    const unsigned long long g = t / G + 1ULL;
    if (t % G == G - 1ULL) {
      asm volatile("fence.acq_rel.gpu;" ::: "memory");
      asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(flags + 16), "l"(g) : "memory");
    } else {
      while (ld_relaxed_u64(flags + 16) < g) {
      }
      asm volatile("fence.acq_rel.gpu;" ::: "memory");
    }
  }
#endif
  __syncthreads();
}

enum TailOp { T_JAC0 = 0, T_JAC = 1, T_JACP = 2, T_SCALE = 3, T_ZERO = 4, T_PROLONG = 5 };

// vector loads: CG = written by other CTAs during this kernel (L2); else plain (shared memory /
// CTA-private data)
template <bool CG>
__device__ __forceinline__ double tl_ld(const double* p) {
  return CG ? __ldcg(p) : *p;
}

// Operator of one level as seen by one group of threads: generic pointers, indexed by the
// level's own row / nonzero numbers (shared-memory copies are biased accordingly).  rp / col /
// val / dinv may point into shared memory (the group's own rows only); dinv_g / agg are the
// level's global arrays (read-only during the kernel: L1), used for the column gathers.
struct TailOpView {
  const int* rp;
  const int* col;
  const double* val;
  const double* dinv;
  const double* dinv_g;
  const int* agg;
  const int* agg_ptr;
  int lpr;
};

// one smoother-type pass over rows [R0, R1) by the T threads of a group (this thread is t);
// returns this thread's share of b . out
template <int OP, bool CG>
__device__ __forceinline__ double tl_row_pass(const TailOpView& A, int R0, int R1, int t, int T, const double* b,
                                              const double* x, const double* ec, double gamma, double* out,
                                              bool want_dot) {
  const int lpr = A.lpr;
  const int g = t / lpr, sub = t & (lpr - 1), ng = T / lpr;
  double dot = 0.0;
  const int trips = (R1 - R0 + ng - 1) / ng;  // every lane of a warp runs the same number of trips
  for (int q = 0; q < trips; ++q) {
    const int i = R0 + g + q * ng;
    const bool act = i < R1;
    double s = 0.0, di = 0.0, bi = 0.0, xi = 0.0;
    if (act) {
      const int k0 = A.rp[i], k1 = A.rp[i + 1];
      if (sub == 0) {  // own-row operands: issued before the gathers, consumed after the reduction
        di = A.dinv[i];
        bi = tl_ld<CG>(b + i);
        if (OP == T_JAC0)
          xi = di * bi;
        else if (OP == T_JACP)
          xi = tl_ld<CG>(x + i) + gamma * tl_ld<CG>(ec + __ldg(A.agg + i));
        else
          xi = tl_ld<CG>(x + i);
      }
      for (int k = k0 + sub; k < k1; k += lpr) {
        const int c = A.col[k];
        double xc;
        if (OP == T_JAC0)
          xc = __ldg(A.dinv_g + c) * tl_ld<CG>(b + c);
        else if (OP == T_JACP)
          xc = tl_ld<CG>(x + c) + gamma * tl_ld<CG>(ec + __ldg(A.agg + c));
        else
          xc = tl_ld<CG>(x + c);
        s += A.val[k] * xc;
      }
    }
    for (int o = lpr >> 1; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (act && sub == 0) {
      const double o = xi + di * (bi - s);
      out[i] = o;
      if (want_dot) dot += bi * o;
    }
  }
  return dot;
}

// vector-only passes (nu1 < 2 or nu2 == 0) over rows [R0, R1)
template <int OP, bool CG>
__device__ __forceinline__ double tl_vec_pass(const TailOpView& A, int R0, int R1, int t, int T, const double* b,
                                              const double* x, const double* ec, double gamma, double* out,
                                              bool want_dot) {
  double dot = 0.0;
  for (int i = R0 + t; i < R1; i += T) {
    double o;
    if (OP == T_SCALE)
      o = A.dinv[i] * tl_ld<CG>(b + i);
    else if (OP == T_ZERO)
      o = 0.0;
    else
      o = tl_ld<CG>(x + i) + gamma * tl_ld<CG>(ec + __ldg(A.agg + i));
    out[i] = o;
    if (want_dot) dot += tl_ld<CG>(b + i) * o;
  }
  return dot;
}

// rc[I] = sum_{i in I} (b_i - sum_j a_ij x_j) for aggregates [A0, A1): the rows of I are
// consecutive, so the sum over the nonzeros of all its rows is one contiguous range
template <bool CG>
__device__ __forceinline__ void tl_restrict_pass(const TailOpView& A, int A0, int A1, int t, int T, const double* b,
                                                 const double* x, double* rc) {
  const int lpr = A.lpr;
  const int g = t / lpr, sub = t & (lpr - 1), ng = T / lpr;
  const int trips = (A1 - A0 + ng - 1) / ng;
  for (int q = 0; q < trips; ++q) {
    const int I = A0 + g + q * ng;
    const bool act = I < A1;
    double s = 0.0;
    if (act) {
      const int ra = __ldg(A.agg_ptr + I), rb = __ldg(A.agg_ptr + I + 1);
      for (int k = A.rp[ra] + sub, e = A.rp[rb]; k < e; k += lpr) s -= A.val[k] * tl_ld<CG>(x + A.col[k]);
      for (int i = ra + sub; i < rb; i += lpr) s += tl_ld<CG>(b + i);
    }
    for (int o = lpr >> 1; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (act && sub == 0) rc[I] = s;
  }
}

// coarsest solve by one CTA for n > LU_SMALL_MAX: factors stay in global memory (L2), y in shared
template <bool CG>
__device__ __forceinline__ void lu_solve_big_cta(int n, const double* __restrict__ lu, const int* __restrict__ piv,
                                                 const double* b, double* x, double* y) {
  const int tid = threadIdx.x, T = blockDim.x;
  for (int i = tid; i < n; i += T) y[i] = tl_ld<CG>(b + i);
  __syncthreads();
  if (tid == 0)
    for (int k = 0; k < n; ++k) {
      const int p = __ldg(piv + k);
      if (p != k) {
        const double t = y[k];
        y[k] = y[p];
        y[p] = t;
      }
    }
  __syncthreads();
  for (int k = 0; k < n - 1; ++k) {
    const double yk = y[k];
    for (int i = k + 1 + tid; i < n; i += T) y[i] -= __ldg(lu + (size_t)i * n + k) * yk;
    __syncthreads();
  }
  for (int i = n - 1; i >= 0; --i) {
    if (tid == 0) y[i] = y[i] / __ldg(lu + (size_t)i * n + i);
    __syncthreads();
    const double yi = y[i];
    for (int j = tid; j < i; j += T) y[j] -= __ldg(lu + (size_t)j * n + i) * yi;
    __syncthreads();
  }
  for (int i = tid; i < n; i += T) x[i] = y[i];
}

inline size_t tail_smem_bytes(int nL) {
  return nL <= LU_SMALL_MAX ? sizeof(double) * ((size_t)nL * (nL + 1) + nL) : sizeof(double) * (size_t)nL;
}

// result buffer of level l after the down sweep / after the whole cycle (same rule on the host)
__host__ __device__ inline bool tail_down_in_x2(int nu1) { return nu1 > 2 && ((nu1 - 2) & 1); }
__host__ __device__ inline bool tail_result_in_x2(int nu1, int nu2) {
  const int swaps = (nu1 > 2 ? nu1 - 2 : 0) + (nu2 >= 1 ? nu2 : 1);
  return swaps & 1;
}

// aligned slices of a chunk (bulk copies need 16-byte aligned sources and sizes)
struct TailSlices {
  int ra4, nrp, ka4, nk4, ka2, nk2, ra2, nr2;
};
__host__ __device__ inline TailSlices tail_slices(const TailChunk& c) {
  TailSlices s;
  s.ra4 = c.R0 & ~3;
  s.nrp = (c.R1 + 1 - s.ra4 + 3) & ~3;
  s.ka4 = c.K0 & ~3;
  s.nk4 = (c.K1 - s.ka4 + 3) & ~3;
  s.ka2 = c.K0 & ~1;
  s.nk2 = (c.K1 - s.ka2 + 1) & ~1;
  s.ra2 = c.R0 & ~1;
  s.nr2 = (c.R1 - s.ra2 + 1) & ~1;
  return s;
}

__device__ __forceinline__ TailOpView tail_view(const TailLevel& L, const TailChunk& ch, unsigned char* stage) {
  TailOpView A;
  if (L.s_rp >= 0) {
    const TailSlices s = tail_slices(ch);
    A.rp = reinterpret_cast<const int*>(stage + L.s_rp) - s.ra4;
    A.col = reinterpret_cast<const int*>(stage + L.s_col) - s.ka4;
    A.val = reinterpret_cast<const double*>(stage + L.s_val) - s.ka2;
    A.dinv = reinterpret_cast<const double*>(stage + L.s_dinv) - s.ra2;
  } else {
    A.rp = L.rowptr, A.col = L.col, A.val = L.val, A.dinv = L.dinv;
  }
  A.dinv_g = L.dinv, A.agg = L.agg, A.agg_ptr = L.agg_ptr, A.lpr = L.lpr;
  return A;
}

// z = B b over rows [i0, i1) of the dense operator (row-major, n x n); `tpr` threads per row
template <bool CG>
__device__ __forceinline__ double tail_dense_rows(int n, const double* __restrict__ B, const double* b, double* z,
                                                  int i0, int i1, bool want_dot, double* red /*[TAIL_THREADS/32]*/) {
  const int tid = threadIdx.x, T = blockDim.x;
  const int nrows = i1 - i0;
  int RB = 1;  // rows per batch: the smallest power of two >= nrows, at least one warp per row
  while (RB < nrows && RB < T / 32) RB <<= 1;
  const int tpr = T / RB;
  const int wpr = tpr >> 5;  // warps per row
  double dot = 0.0;
  for (int rb = i0; rb < i1; rb += RB) {
    const int r = rb + tid / tpr, t = tid & (tpr - 1);
    double s = 0.0;
    if (r < i1) {
      const double* row = B + (size_t)r * n;
      for (int j = t; j < n; j += tpr) s += __ldg(row + j) * tl_ld<CG>(b + j);
    }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((tid & 31) == 0) red[tid >> 5] = s;
    __syncthreads();
    if (tid < RB && rb + tid < i1) {
      double v = 0.0;
      for (int q = 0; q < wpr; ++q) v += red[tid * wpr + q];
      z[rb + tid] = v;
      if (want_dot) dot += tl_ld<CG>(b + rb + tid) * v;
    }
    __syncthreads();
  }
  return dot;
}

__global__ void __launch_bounds__(TAIL_THREADS, 1) k_vcycle_tail(TailArgs a) {
  pdl_launch_dependents();
  {  // before the grid dependency: pull this CTA's rows of the dense operator (setup data) into L2
    const bool dense0 = a.dense_level >= 0 && a.first <= a.dense_level;
    if (dense0) {
      const int nD = a.lv[a.dense_level].n;
      const int i0 = (int)((int64_t)blockIdx.x * nD / gridDim.x), i1 = (int)((int64_t)(blockIdx.x + 1) * nD / gridDim.x);
      const char* p0 = reinterpret_cast<const char*>(a.dense_B + (size_t)i0 * nD);
      const size_t bytes = (size_t)(i1 - i0) * nD * sizeof(double);
      for (size_t o = (size_t)threadIdx.x * 128; o < bytes; o += (size_t)TAIL_THREADS * 128)
        asm volatile("prefetch.global.L2 [%0];" ::"l"(p0 + o));
    }
  }
  pdl_wait();
  if (a.ctl != nullptr && a.ctl->done) return;
  extern __shared__ __align__(128) unsigned char tail_sm[];
  __shared__ uint64_t lvbar[TAIL_MAX_LEVELS];
  __shared__ double red[TAIL_THREADS / 32];
  const int tid = threadIdx.x, G = gridDim.x, cta = blockIdx.x;
  const bool use_dense = a.dense_level >= 0 && a.first <= a.dense_level;
  const int E = use_dense ? a.dense_level : a.last;  // sparse levels [first, E), then the bottom solve on E
  unsigned char* stage = tail_sm + a.lu_smem;
  double dot = 0.0;
  unsigned long long gen = ld_acquire_u64(a.bar + 32 + blockIdx.x);  // flag variant: warp 0 keeps it current
  int pslot = 0;
  TAIL_STAMP(a, pslot++);

  // ---- stage this CTA's operator chunks of every sparse level ----
  if (tid == 0) {
    for (int l = a.first; l < E; ++l) mbar_init(&lvbar[l], 1);
    fence_mbar_init();
    for (int l = a.first; l < E; ++l) {
      const TailLevel& L = a.lv[l];
      if (L.s_rp < 0) continue;
      const TailChunk ch = a.chunk[l * G + cta];
      if (ch.R1 <= ch.R0) {
        mbar_arrive(&lvbar[l]);
        continue;
      }
      const TailSlices s = tail_slices(ch);
      mbar_arrive_expect_tx(&lvbar[l], 4u * s.nrp + 4u * s.nk4 + 8u * s.nk2 + 8u * s.nr2);
      bulk_g2s<false>(stage + L.s_rp, L.rowptr + s.ra4, 4u * s.nrp, &lvbar[l], 0);
      bulk_g2s<false>(stage + L.s_col, L.col + s.ka4, 4u * s.nk4, &lvbar[l], 0);
      bulk_g2s<false>(stage + L.s_val, L.val + s.ka2, 8u * s.nk2, &lvbar[l], 0);
      bulk_g2s<false>(stage + L.s_dinv, L.dinv + s.ra2, 8u * s.nr2, &lvbar[l], 0);
    }
  }
  __syncthreads();

  // ---- down ----
  for (int l = a.first; l < E; ++l) {
    const TailLevel L = a.lv[l];
    const TailChunk ch = a.chunk[l * G + cta];
    if (L.s_rp >= 0) mbar_wait(&lvbar[l], 0);
    TAIL_STAMP(a, pslot++);
    const TailOpView A = tail_view(L, ch, stage);
    const double* b = (l == a.first) ? a.b_first : L.b;
    double* cur = L.x;
    double* oth = L.x2;
    int done;
    if (a.nu1 >= 2) {
      tl_row_pass<T_JAC0, true>(A, ch.R0, ch.R1, tid, TAIL_THREADS, b, nullptr, nullptr, 0.0, cur, false);
      done = 2;
    } else if (a.nu1 == 1) {
      tl_vec_pass<T_SCALE, true>(A, ch.R0, ch.R1, tid, TAIL_THREADS, b, nullptr, nullptr, 0.0, cur, false);
      done = 1;
    } else {
      tl_vec_pass<T_ZERO, true>(A, ch.R0, ch.R1, tid, TAIL_THREADS, b, nullptr, nullptr, 0.0, cur, false);
      done = 0;
    }
    TAIL_STAMP(a, pslot++);
    tail_grid_barrier(a.bar, gen);
    TAIL_STAMP(a, pslot++);
    for (int s = done; s < a.nu1; ++s) {
      tl_row_pass<T_JAC, true>(A, ch.R0, ch.R1, tid, TAIL_THREADS, b, cur, nullptr, 0.0, oth, false);
      double* t = cur;
      cur = oth;
      oth = t;
      tail_grid_barrier(a.bar, gen);
    }
    tl_restrict_pass<true>(A, ch.A0, ch.A1, tid, TAIL_THREADS, b, cur, a.lv[l + 1].b);
    TAIL_STAMP(a, pslot++);
    tail_grid_barrier(a.bar, gen);
    TAIL_STAMP(a, pslot++);
  }

  // ---- bottom: the dense collapsed operator of levels >= E, or the LU solve of the coarsest level ----
  {
    const TailLevel L = a.lv[E];
    const double* b = (E == a.first) ? a.b_first : L.b;
    const bool want = (E == a.first) && a.fin != FIN_NONE;
    if (use_dense) {
      const int i0 = (int)((int64_t)cta * L.n / G), i1 = (int)((int64_t)(cta + 1) * L.n / G);
      dot += tail_dense_rows<true>(L.n, a.dense_B, b, L.x, i0, i1, want, red);
    } else if (cta == 0) {
      if (a.nL <= LU_SMALL_MAX)
        lu_solve_small_cta<true>(a.nL, a.lu, a.piv, b, L.x, reinterpret_cast<double*>(tail_sm));
      else
        lu_solve_big_cta<true>(a.nL, a.lu, a.piv, b, L.x, reinterpret_cast<double*>(tail_sm));
      if (want)
        for (int i = tid; i < L.n; i += TAIL_THREADS) dot += __ldcg(b + i) * L.x[i];
    }
    TAIL_STAMP(a, pslot++);
    if (a.first < E) tail_grid_barrier(a.bar, gen);
    TAIL_STAMP(a, pslot++);
  }

  // ---- up ----
  for (int l = E - 1; l >= a.first; --l) {
    const TailLevel L = a.lv[l];
    const TailChunk ch = a.chunk[l * G + cta];
    const TailOpView A = tail_view(L, ch, stage);
    const double* b = (l == a.first) ? a.b_first : L.b;
    const bool top = (l == a.first) && a.fin != FIN_NONE;
    double* cur = tail_down_in_x2(a.nu1) ? L.x2 : L.x;
    double* oth = tail_down_in_x2(a.nu1) ? L.x : L.x2;
    const TailLevel& C = a.lv[l + 1];
    const double* ec = (l + 1 == E) ? C.x : (tail_result_in_x2(a.nu1, a.nu2) ? C.x2 : C.x);
    if (a.nu2 >= 1) {
      dot += tl_row_pass<T_JACP, true>(A, ch.R0, ch.R1, tid, TAIL_THREADS, b, cur, ec, a.gamma, oth, top && a.nu2 == 1);
      double* t = cur;
      cur = oth;
      oth = t;
      for (int s = 1; s < a.nu2; ++s) {
        TAIL_STAMP(a, pslot++);
        tail_grid_barrier(a.bar, gen);
        TAIL_STAMP(a, pslot++);
        dot += tl_row_pass<T_JAC, true>(A, ch.R0, ch.R1, tid, TAIL_THREADS, b, cur, nullptr, 0.0, oth,
                                        top && s == a.nu2 - 1);
        t = cur;
        cur = oth;
        oth = t;
      }
    } else {
      dot += tl_vec_pass<T_PROLONG, true>(A, ch.R0, ch.R1, tid, TAIL_THREADS, b, cur, ec, a.gamma, oth, top);
    }
    TAIL_STAMP(a, pslot++);
    if (l > a.first) tail_grid_barrier(a.bar, gen);
    TAIL_STAMP(a, pslot++);
  }

  // ---- fused r.z of a cycle that starts at level 0 (small systems: the whole cycle is this kernel) ----
  if (a.fin != FIN_NONE) {
    for (int o = 16; o > 0; o >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, o);
    __syncthreads();
    if ((tid & 31) == 0) red[tid >> 5] = dot;
    __syncthreads();
    if (tid == 0) {
      double s = 0.0;
      for (int q = 0; q < TAIL_THREADS / 32; ++q) s += red[q];
      a.partials[blockIdx.x] = s;
    }
    tail_grid_barrier(a.bar, gen);
    if (blockIdx.x == 0 && tid < 32) {
      double s = 0.0;
      for (unsigned q = tid; q < gridDim.x; q += 32) s += __ldcg(a.partials + q);
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      if (tid == 0) krylov_finalize(a.ctl, a.fin, s, 0.0);
    }
  }
}

// ------------------------------------------------------------------------------------------
// Setup of the dense collapsed operator: CTA j runs the V-cycle of levels D..last on the unit
// vector e_j with every vector in shared memory (operators through L1/L2) and writes column j.
// B[i][j] = (Vcycle_D e_j)_i, stored row-major, so that z = B r is exactly the V-cycle applied
// to r up to the rounding of a different summation order.
// ------------------------------------------------------------------------------------------
constexpr int TAILB_THREADS = 256;
struct TailBuildArgs {
  const TailLevel* lv;
  int D, last, nu1, nu2;
  double gamma;
  int nL;
  const double* lu;
  const int* piv;
  double* B;
  int lu_smem;
};

__global__ void __launch_bounds__(TAILB_THREADS) k_tail_dense_build(TailBuildArgs a) {
  extern __shared__ __align__(16) unsigned char tb_sm[];
  double* vec = reinterpret_cast<double*>(tb_sm + a.lu_smem);
  const int tid = threadIdx.x, j = blockIdx.x;
  auto vb = [&](int l) {  // b_l, then x_l, x2_l
    int off = 0;
    for (int q = a.D; q < l; ++q) off += 3 * a.lv[q].n;
    return vec + off;
  };
  const int nD = a.lv[a.D].n;
  {
    double* b = vb(a.D);
    for (int i = tid; i < nD; i += TAILB_THREADS) b[i] = (i == j) ? 1.0 : 0.0;
  }
  __syncthreads();
  for (int l = a.D; l < a.last; ++l) {
    const TailLevel L = a.lv[l];
    TailOpView A;
    A.rp = L.rowptr, A.col = L.col, A.val = L.val, A.dinv = L.dinv;
    A.dinv_g = L.dinv, A.agg = L.agg, A.agg_ptr = L.agg_ptr, A.lpr = L.lpr;
    double* b = vb(l);
    double* cur = b + L.n;
    double* oth = cur + L.n;
    int done;
    if (a.nu1 >= 2) {
      tl_row_pass<T_JAC0, false>(A, 0, L.n, tid, TAILB_THREADS, b, nullptr, nullptr, 0.0, cur, false);
      done = 2;
    } else if (a.nu1 == 1) {
      tl_vec_pass<T_SCALE, false>(A, 0, L.n, tid, TAILB_THREADS, b, nullptr, nullptr, 0.0, cur, false);
      done = 1;
    } else {
      tl_vec_pass<T_ZERO, false>(A, 0, L.n, tid, TAILB_THREADS, b, nullptr, nullptr, 0.0, cur, false);
      done = 0;
    }
    __syncthreads();
    for (int s = done; s < a.nu1; ++s) {
      tl_row_pass<T_JAC, false>(A, 0, L.n, tid, TAILB_THREADS, b, cur, nullptr, 0.0, oth, false);
      double* t = cur;
      cur = oth;
      oth = t;
      __syncthreads();
    }
    tl_restrict_pass<false>(A, 0, L.nc, tid, TAILB_THREADS, b, cur, vb(l + 1));
    __syncthreads();
  }
  {
    double* b = vb(a.last);
    double* x = b + a.lv[a.last].n;
    if (a.nL <= LU_SMALL_MAX)
      lu_solve_small_cta<false>(a.nL, a.lu, a.piv, b, x, reinterpret_cast<double*>(tb_sm));
    else
      lu_solve_big_cta<false>(a.nL, a.lu, a.piv, b, x, reinterpret_cast<double*>(tb_sm));
    __syncthreads();
  }
  for (int l = a.last - 1; l >= a.D; --l) {
    const TailLevel L = a.lv[l];
    TailOpView A;
    A.rp = L.rowptr, A.col = L.col, A.val = L.val, A.dinv = L.dinv;
    A.dinv_g = L.dinv, A.agg = L.agg, A.agg_ptr = L.agg_ptr, A.lpr = L.lpr;
    double* b = vb(l);
    double* x = b + L.n;
    double* x2 = x + L.n;
    double* cur = tail_down_in_x2(a.nu1) ? x2 : x;
    double* oth = tail_down_in_x2(a.nu1) ? x : x2;
    double* cb = vb(l + 1);
    const int ncn = a.lv[l + 1].n;
    const double* ec = (l + 1 == a.last) ? cb + ncn : (tail_result_in_x2(a.nu1, a.nu2) ? cb + 2 * ncn : cb + ncn);
    if (a.nu2 >= 1) {
      tl_row_pass<T_JACP, false>(A, 0, L.n, tid, TAILB_THREADS, b, cur, ec, a.gamma, oth, false);
      double* t = cur;
      cur = oth;
      oth = t;
      for (int s = 1; s < a.nu2; ++s) {
        __syncthreads();
        tl_row_pass<T_JAC, false>(A, 0, L.n, tid, TAILB_THREADS, b, cur, nullptr, 0.0, oth, false);
        t = cur;
        cur = oth;
        oth = t;
      }
    } else {
      tl_vec_pass<T_PROLONG, false>(A, 0, L.n, tid, TAILB_THREADS, b, cur, ec, a.gamma, oth, false);
    }
    __syncthreads();
  }
  {
    const double* b = vb(a.D);
    const double* z;
    if (a.D == a.last)
      z = b + nD;
    else
      z = tail_result_in_x2(a.nu1, a.nu2) ? b + 2 * nD : b + nD;
    for (int i = tid; i < nD; i += TAILB_THREADS) a.B[(size_t)i * nD + j] = z[i];
  }
}
