// Coarse tail of the V-cycle (S2-S6 on the small levels): ONE persistent kernel runs every level
// from `first` down to the coarsest solve and back up.  The levels below ~64 k rows hold < 3 % of
// the V-cycle's bytes but three quarters of its kernel launches; each of those launches costs
// 8-11 us (launch + pipeline fill + reduction tail) for < 1 us of memory time.  Here the CTAs
// stay resident (one per SM), the operators are read from L2, and the dependency between two
// passes is a grid-wide barrier (~1 us: one atomic arrival per CTA, one polled release flag)
// instead of a kernel boundary.
//
// Work split: LPR lanes per row (per aggregate for the restriction: its rows are contiguous, so
// its nonzeros are ONE contiguous range); rows are dealt round-robin to the sub-warps of the grid.
// Vectors written inside the kernel are read with ld.global.cg (L2) -- L1 is not coherent across
// CTAs; the operator arrays are read-only for the whole kernel and go through L1.
#pragma once
#include "amg_kernels.cuh"

constexpr int TAIL_THREADS = 512;
constexpr int TAIL_MAX_LEVELS = 32;

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
};

struct TailArgs {
  const TailLevel* lv;   // device array indexed by level
  int first, last;       // first level of the call, coarsest level
  const double* b_first; // right-hand side of level `first`
  int nu1, nu2;
  double gamma;
  int nL;
  const double* lu;
  const int* piv;
  unsigned long long* bar;  // [0] arrival counter, [16] release generation
  double* partials;
  KrylovCtl* ctl;           // may be null (hooks)
  int fin;                  // FIN_RZ: b_first . result is reduced and finalised (first == 0 only)
};

__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_u64(unsigned long long* p, unsigned long long v) {
  asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// All CTAs of the grid are co-resident (grid <= number of SMs, one CTA each).  The arrival
// counter only grows: every launch performs whole barriers, so it stays a multiple of gridDim.x.
__device__ __forceinline__ void tail_grid_barrier(unsigned long long* bar) {
  __syncthreads();
  if (threadIdx.x == 0) {
    const unsigned long long G = gridDim.x;
    __threadfence();
    const unsigned long long t = atomicAdd(bar, 1ULL);
    const unsigned long long gen = t / G + 1ULL;
    if (t % G == G - 1ULL) {
      st_release_u64(bar + 16, gen);
    } else {
      while (ld_acquire_u64(bar + 16) < gen) {
      }
    }
    __threadfence();
  }
  __syncthreads();
}

enum TailOp { T_JAC0 = 0, T_JAC = 1, T_JACP = 2, T_SCALE = 3, T_ZERO = 4, T_PROLONG = 5 };

// one smoother-type pass over the rows of a level; returns this thread's share of b . out
template <int OP>
__device__ __forceinline__ double tail_row_pass(const TailLevel& L, const double* b, const double* x,
                                                const double* ec, double gamma, double* out, bool want_dot) {
  const int lpr = L.lpr;
  const int gsub = (blockIdx.x * TAIL_THREADS + threadIdx.x) / lpr;
  const int sub = threadIdx.x & (lpr - 1);
  const int nsub = gridDim.x * TAIL_THREADS / lpr;
  const int n = L.n;
  double dot = 0.0;
  const int trips = (n + nsub - 1) / nsub;  // every lane of a warp runs the same number of trips
  for (int t = 0; t < trips; ++t) {
    const int i = gsub + t * nsub;
    double s = 0.0;
    if (i < n) {
      for (int k = __ldg(L.rowptr + i) + sub, e = __ldg(L.rowptr + i + 1); k < e; k += lpr) {
        const int c = __ldg(L.col + k);
        double xc;
        if (OP == T_JAC0)
          xc = __ldg(L.dinv + c) * __ldcg(b + c);
        else if (OP == T_JACP)
          xc = __ldcg(x + c) + gamma * __ldcg(ec + __ldg(L.agg + c));
        else
          xc = __ldcg(x + c);
        s += __ldg(L.val + k) * xc;
      }
    }
    for (int o = lpr >> 1; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (i < n && sub == 0) {
      const double di = __ldg(L.dinv + i), bi = __ldcg(b + i);
      double xi;
      if (OP == T_JAC0)
        xi = di * bi;
      else if (OP == T_JACP)
        xi = __ldcg(x + i) + gamma * __ldcg(ec + __ldg(L.agg + i));
      else
        xi = __ldcg(x + i);
      const double o = xi + di * (bi - s);
      out[i] = o;
      if (want_dot) dot += bi * o;
    }
  }
  return dot;
}

// vector-only passes (nu1 < 2 or nu2 == 0)
template <int OP>
__device__ __forceinline__ double tail_vec_pass(const TailLevel& L, const double* b, const double* x,
                                                const double* ec, double gamma, double* out, bool want_dot) {
  double dot = 0.0;
  for (int i = blockIdx.x * TAIL_THREADS + threadIdx.x; i < L.n; i += gridDim.x * TAIL_THREADS) {
    double o;
    if (OP == T_SCALE)
      o = __ldg(L.dinv + i) * __ldcg(b + i);
    else if (OP == T_ZERO)
      o = 0.0;
    else
      o = __ldcg(x + i) + gamma * __ldcg(ec + __ldg(L.agg + i));
    out[i] = o;
    if (want_dot) dot += __ldcg(b + i) * o;
  }
  return dot;
}

// rc[I] = sum_{i in I} (b_i - sum_j a_ij x_j): the rows of I are consecutive, so the sum over the
// nonzeros of all its rows is one contiguous range
__device__ __forceinline__ void tail_restrict_pass(const TailLevel& L, const double* b, const double* x, double* rc) {
  const int lpr = L.lpr;
  const int gsub = (blockIdx.x * TAIL_THREADS + threadIdx.x) / lpr;
  const int sub = threadIdx.x & (lpr - 1);
  const int nsub = gridDim.x * TAIL_THREADS / lpr;
  const int nc = L.nc;
  const int trips = (nc + nsub - 1) / nsub;
  for (int t = 0; t < trips; ++t) {
    const int I = gsub + t * nsub;
    double s = 0.0;
    if (I < nc) {
      const int ra = __ldg(L.agg_ptr + I), rb = __ldg(L.agg_ptr + I + 1);
      for (int k = __ldg(L.rowptr + ra) + sub, e = __ldg(L.rowptr + rb); k < e; k += lpr)
        s -= __ldg(L.val + k) * __ldcg(x + __ldg(L.col + k));
      for (int i = ra + sub; i < rb; i += lpr) s += __ldcg(b + i);
    }
    for (int o = lpr >> 1; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (I < nc && sub == 0) rc[I] = s;
  }
}

// coarsest solve by one CTA for n > LU_SMALL_MAX: factors stay in global memory (L2), y in shared
__device__ __forceinline__ void lu_solve_big_cta(int n, const double* __restrict__ lu, const int* __restrict__ piv,
                                                 const double* b, double* x, double* y) {
  const int tid = threadIdx.x, T = blockDim.x;
  for (int i = tid; i < n; i += T) y[i] = __ldcg(b + i);
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

__global__ void __launch_bounds__(TAIL_THREADS, 1) k_vcycle_tail(TailArgs a) {
  if (a.ctl != nullptr && a.ctl->done) return;
  extern __shared__ double tail_sm[];
  __shared__ double red[TAIL_THREADS / 32];
  const int tid = threadIdx.x;
  double dot = 0.0;

  // ---- down ----
  for (int l = a.first; l < a.last; ++l) {
    const TailLevel L = a.lv[l];
    const double* b = (l == a.first) ? a.b_first : L.b;
    double* cur = L.x;
    double* oth = L.x2;
    int done;
    if (a.nu1 >= 2) {
      tail_row_pass<T_JAC0>(L, b, nullptr, nullptr, 0.0, cur, false);
      done = 2;
    } else if (a.nu1 == 1) {
      tail_vec_pass<T_SCALE>(L, b, nullptr, nullptr, 0.0, cur, false);
      done = 1;
    } else {
      tail_vec_pass<T_ZERO>(L, b, nullptr, nullptr, 0.0, cur, false);
      done = 0;
    }
    tail_grid_barrier(a.bar);
    for (int s = done; s < a.nu1; ++s) {
      tail_row_pass<T_JAC>(L, b, cur, nullptr, 0.0, oth, false);
      double* t = cur;
      cur = oth;
      oth = t;
      tail_grid_barrier(a.bar);
    }
    tail_restrict_pass(L, b, cur, a.lv[l + 1].b);
    tail_grid_barrier(a.bar);
  }

  // ---- coarsest ----
  {
    const TailLevel L = a.lv[a.last];
    const double* b = (a.last == a.first) ? a.b_first : L.b;
    if (blockIdx.x == 0) {
      if (a.nL <= LU_SMALL_MAX)
        lu_solve_small_cta(a.nL, a.lu, a.piv, b, L.x, tail_sm);
      else
        lu_solve_big_cta(a.nL, a.lu, a.piv, b, L.x, tail_sm);
      if (a.first == a.last && a.fin != FIN_NONE)
        for (int i = tid; i < L.n; i += TAIL_THREADS) dot += __ldcg(b + i) * L.x[i];
    }
    if (a.first < a.last) tail_grid_barrier(a.bar);
  }

  // ---- up ----
  for (int l = a.last - 1; l >= a.first; --l) {
    const TailLevel L = a.lv[l];
    const double* b = (l == a.first) ? a.b_first : L.b;
    const bool top = (l == a.first) && a.fin != FIN_NONE;
    double* cur = tail_down_in_x2(a.nu1) ? L.x2 : L.x;
    double* oth = tail_down_in_x2(a.nu1) ? L.x : L.x2;
    const TailLevel& C = a.lv[l + 1];
    const double* ec = (l + 1 == a.last) ? C.x : (tail_result_in_x2(a.nu1, a.nu2) ? C.x2 : C.x);
    if (a.nu2 >= 1) {
      dot += tail_row_pass<T_JACP>(L, b, cur, ec, a.gamma, oth, top && a.nu2 == 1);
      double* t = cur;
      cur = oth;
      oth = t;
      for (int s = 1; s < a.nu2; ++s) {
        tail_grid_barrier(a.bar);
        dot += tail_row_pass<T_JAC>(L, b, cur, nullptr, 0.0, oth, top && s == a.nu2 - 1);
        t = cur;
        cur = oth;
        oth = t;
      }
    } else {
      dot += tail_vec_pass<T_PROLONG>(L, b, cur, ec, a.gamma, oth, top);
    }
    if (l > a.first) tail_grid_barrier(a.bar);
  }

  // ---- fused r.z of a cycle that starts at level 0 (small systems: the whole cycle is this kernel) ----
  if (a.fin != FIN_NONE) {
    for (int o = 16; o > 0; o >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, o);
    if ((tid & 31) == 0) red[tid >> 5] = dot;
    __syncthreads();
    if (tid == 0) {
      double s = 0.0;
      for (int q = 0; q < TAIL_THREADS / 32; ++q) s += red[q];
      a.partials[blockIdx.x] = s;
    }
    tail_grid_barrier(a.bar);
    if (blockIdx.x == 0 && tid < 32) {
      double s = 0.0;
      for (unsigned q = tid; q < gridDim.x; q += 32) s += __ldcg(a.partials + q);
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      if (tid == 0) krylov_finalize(a.ctl, a.fin, s, 0.0);
    }
  }
}
