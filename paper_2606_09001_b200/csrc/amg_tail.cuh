// Coarse tail of the V-cycle (S2-S6 on the small levels).  The levels below a few thousand rows hold
// < 2 % of the V-cycle's bytes but a third of its kernel launches, and every pass over them is a
// chain of dependent memory round trips, not a bandwidth problem.  They are therefore not visited at
// all: the V-cycle from the first level D with at most `tail_dense_rows` rows down to the coarsest
// solve and back is a FIXED linear operator z = B_D r.  It is assembled once at setup as a dense
// matrix (k_tail_dense_build runs that V-cycle on the unit vectors, all vectors in shared memory) and
// applied as one dense matrix-vector product spread over all SMs (k_dense_tail): 1 pass instead of
// 4 passes x 5 levels + the LU solve.  The same map up to summation order (parity <= 1e-12).
//
// (Round 1 also carried sparse levels inside one persistent kernel with grid barriers between the
// passes; on B200 such a phase measured dearer than a row-tile launch in the PDL-chained graph on
// every level -- 3-5 us of barrier, mostly arrival skew -- and a spinning grid barrier needs all
// CTAs co-resident, which a plain launch next to other work does not guarantee.  It was removed.)
//
// No floating-point atomics: every sum has a fixed order for a fixed grid.
#pragma once
#include "amg_kernels.cuh"

constexpr int TAIL_THREADS = 1024;
constexpr int TAIL_MAX_LEVELS = 32;

struct TailLevel {
  int n, nc, nnz, lpr;
  int v32, pad;  // v32: the level's values are rounded to fp32 on the fly (mixed-precision hierarchy)
  const int* rowptr;
  const int* col;
  const double* val;
  const double* dinv;
  const double* dsw[AMG_MAX_SWEEPS];  // diagonal of every sweep of a cycle (Level::dsw)
  const int* agg;
  const int* agg_ptr;
};

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
  int v32;
  __device__ __forceinline__ double a(int k) const { return v32 ? (double)(float)val[k] : val[k]; }
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
          xi = __ldg(A.dinv_g + i) * bi;  // x1 with the diagonal of the first sweep, the epilogue with the second's
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
        s += A.a(k) * xc;
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
      for (int k = A.rp[ra] + sub, e = A.rp[rb]; k < e; k += lpr) s -= A.a(k) * tl_ld<CG>(x + A.col[k]);
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

struct TailArgs {
  int n;                   // rows of level D (the level the dense operator starts at)
  const double* dense_B;   // [n x n] row-major: z = B_D b
  const double* b;         // right-hand side of level D
  double* z;               // result
  double* partials;
  unsigned* counter;
  KrylovCtl* ctl;          // may be null (hooks)
  int fin;                 // FIN_RZ: b . z is reduced and finalised (cycles that start at level D = 0)
};

static __global__ void __launch_bounds__(TAIL_THREADS, 1) k_dense_tail(TailArgs a) {
  pdl_launch_dependents();
  const int G = gridDim.x, cta = blockIdx.x;
  const int i0 = (int)((int64_t)cta * a.n / G), i1 = (int)((int64_t)(cta + 1) * a.n / G);
  {  // before the grid dependency: pull this CTA's rows of the dense operator (setup data) into L2
    const char* p0 = reinterpret_cast<const char*>(a.dense_B + (size_t)i0 * a.n);
    const size_t bytes = (size_t)(i1 - i0) * a.n * sizeof(double);
    for (size_t o = (size_t)threadIdx.x * 128; o < bytes; o += (size_t)TAIL_THREADS * 128)
      asm volatile("prefetch.global.L2 [%0];" ::"l"(p0 + o));
  }
  pdl_wait();
  if (a.ctl != nullptr && a.ctl->done) return;
  __shared__ double red[TAIL_THREADS / 32];
  const bool want = a.fin != FIN_NONE;
  double dot[1];
  dot[0] = tail_dense_rows<false>(a.n, a.dense_B, a.b, a.z, i0, i1, want, red);
  // fused r.z of a cycle that starts at level 0 (small systems: the whole cycle is this kernel)
  if (want) grid_reduce_finalize<1, TAIL_THREADS>(dot, a.partials, a.counter, a.ctl, a.fin);
}

// ------------------------------------------------------------------------------------------
// Setup of the dense collapsed operator: CTA j runs the V-cycle of levels D..last on the unit
// vector e_j with every vector in shared memory (operators through L1/L2) and writes column j.
// B[i][j] = (Vcycle_D e_j)_i, stored row-major, so that z = B r is exactly the V-cycle applied
// to r up to the rounding of a different summation order.
// ------------------------------------------------------------------------------------------
constexpr int TAILB_THREADS = 1024;
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

static __global__ void __launch_bounds__(TAILB_THREADS) k_tail_dense_build(TailBuildArgs a) {
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
    A.dinv_g = L.dinv, A.agg = L.agg, A.agg_ptr = L.agg_ptr, A.lpr = L.lpr, A.v32 = L.v32;
    double* b = vb(l);
    double* cur = b + L.n;
    double* oth = cur + L.n;
    int done;
    if (a.nu1 >= 2) {
      A.dinv_g = L.dsw[0], A.dinv = L.dsw[1];
      tl_row_pass<T_JAC0, false>(A, 0, L.n, tid, TAILB_THREADS, b, nullptr, nullptr, 0.0, cur, false);
      done = 2;
    } else if (a.nu1 == 1) {
      A.dinv = L.dsw[0];
      tl_vec_pass<T_SCALE, false>(A, 0, L.n, tid, TAILB_THREADS, b, nullptr, nullptr, 0.0, cur, false);
      done = 1;
    } else {
      tl_vec_pass<T_ZERO, false>(A, 0, L.n, tid, TAILB_THREADS, b, nullptr, nullptr, 0.0, cur, false);
      done = 0;
    }
    __syncthreads();
    for (int s = done; s < a.nu1; ++s) {
      A.dinv = L.dsw[s];
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
    A.dinv_g = L.dinv, A.agg = L.agg, A.agg_ptr = L.agg_ptr, A.lpr = L.lpr, A.v32 = L.v32;
    double* b = vb(l);
    double* x = b + L.n;
    double* x2 = x + L.n;
    double* cur = tail_down_in_x2(a.nu1) ? x2 : x;
    double* oth = tail_down_in_x2(a.nu1) ? x : x2;
    double* cb = vb(l + 1);
    const int ncn = a.lv[l + 1].n;
    const double* ec = (l + 1 == a.last) ? cb + ncn : (tail_result_in_x2(a.nu1, a.nu2) ? cb + 2 * ncn : cb + ncn);
    if (a.nu2 >= 1) {
      A.dinv = L.dsw[a.nu1];
      tl_row_pass<T_JACP, false>(A, 0, L.n, tid, TAILB_THREADS, b, cur, ec, a.gamma, oth, false);
      double* t = cur;
      cur = oth;
      oth = t;
      for (int s = 1; s < a.nu2; ++s) {
        __syncthreads();
        A.dinv = L.dsw[a.nu1 + s];
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
