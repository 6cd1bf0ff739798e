// Solve-phase device code: the row-block streaming kernel family
// (SpMV / smoother / residual+restriction share one template), its row-vector fallback, the
// fused Krylov BLAS-1 kernels with device-side scalar updates, the dense LU solve.
#pragma once
#include "amg_internal.cuh"

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
  const int* blk_ptr;
  const double* x;      // gathered vector
  const double* b;
  const double* dinv;
  double* out;
  const int* agg;       // prolongation / restriction
  const int* agg_ptr;
  const double* ec;
  double gamma;
  const double* d0;     // second operand of the fused dot (SpMV)
  double* partials;     // [ndot][gridDim.x]
  unsigned* counter;
  KrylovCtl* ctl;       // may be null (hooks)
  int fin;
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
  if (OP == OP_JACOBI0) return __ldg(a.dinv + c) * __ldg(a.b + c);
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
    xi = di * bi;
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
// Row-block streaming kernel.  One CTA owns the rows [blk_ptr[b], blk_ptr[b+1]) (boundaries on
// aggregate starts, <= RB_CAP nonzeros, <= RB_MAXROWS rows):
//   phase 1  the CTA streams its contiguous slice of val/col with 128-bit coalesced loads,
//            gathers x[col] through L1/L2 and stages the products in shared memory;
//   phase 2  one thread per row adds its segment of products (fixed order) and applies the
//            row epilogue (SpMV / Jacobi / fused two-sweep Jacobi / prolongation-fused Jacobi);
//   phase 3  (OP_RESTRICT) one thread per aggregate adds the residuals of its contiguous rows.
// ------------------------------------------------------------------------------------------
template <int OP, int NDOT, bool STREAM>
__global__ void __launch_bounds__(RB_THREADS) k_rowblock(RowArgs a) {
  if (a.ctl != nullptr && a.ctl->done) return;
  __shared__ __align__(16) double prod[RB_CAP];
  __shared__ int srp[RB_MAXROWS + 1];
  const int tid = threadIdx.x;
  const int r0 = a.blk_ptr[blockIdx.x], r1 = a.blk_ptr[blockIdx.x + 1];
  const int nrows = r1 - r0;
  double dots[NDOT > 0 ? NDOT : 1];
#pragma unroll
  for (int j = 0; j < (NDOT > 0 ? NDOT : 1); ++j) dots[j] = 0.0;

  if (nrows > 0) {
    for (int i = tid; i <= nrows; i += RB_THREADS) srp[i] = a.rowptr[r0 + i];
    __syncthreads();
    const int k0 = srp[0], k1 = srp[nrows];
    const int ka = k0 & ~3;
    const int nq = (k1 - ka + 3) >> 2;
    const int4* col4 = reinterpret_cast<const int4*>(a.col + ka);
    const double2* val2 = reinterpret_cast<const double2*>(a.val + ka);
    for (int q = tid; q < nq; q += RB_THREADS) {
      const int4 c = ld_i4<STREAM>(col4 + q);
      const double2 v01 = ld_d2<STREAM>(val2 + 2 * q);
      const double2 v23 = ld_d2<STREAM>(val2 + 2 * q + 1);
      const double x0 = gather_x<OP>(a, c.x), x1 = gather_x<OP>(a, c.y);
      const double x2 = gather_x<OP>(a, c.z), x3 = gather_x<OP>(a, c.w);
      double2* dst = reinterpret_cast<double2*>(prod + 4 * q);
      dst[0] = make_double2(v01.x * x0, v01.y * x1);
      dst[1] = make_double2(v23.x * x2, v23.y * x3);
    }
    __syncthreads();
    if (OP == OP_RESTRICT) {
      double res[RB_MAXROWS / RB_THREADS];
#pragma unroll
      for (int t = 0; t < RB_MAXROWS / RB_THREADS; ++t) {
        const int lr = tid + t * RB_THREADS;
        if (lr < nrows) {
          double s = 0.0;
          for (int k = srp[lr] - ka, e = srp[lr + 1] - ka; k < e; ++k) s += prod[k];
          res[t] = row_epilogue<OP>(a, r0 + lr, s);
        }
      }
      __syncthreads();  // all segments consumed: reuse prod[] for the row residuals
#pragma unroll
      for (int t = 0; t < RB_MAXROWS / RB_THREADS; ++t) {
        const int lr = tid + t * RB_THREADS;
        if (lr < nrows) prod[lr] = res[t];
      }
      __syncthreads();
      const int I0 = a.agg[r0], I1 = a.agg[r1 - 1];
      for (int I = I0 + tid; I <= I1; I += RB_THREADS) {
        double s = 0.0;
        for (int r = a.agg_ptr[I] - r0, e = a.agg_ptr[I + 1] - r0; r < e; ++r) s += prod[r];
        a.out[I] = s;
      }
    } else {
      for (int lr = tid; lr < nrows; lr += RB_THREADS) {
        double s = 0.0;
        for (int k = srp[lr] - ka, e = srp[lr + 1] - ka; k < e; ++k) s += prod[k];
        const int i = r0 + lr;
        const double o = row_epilogue<OP>(a, i, s);
        a.out[i] = o;
        if (NDOT >= 1) dots[0] += (OP == OP_SPMV ? a.d0[i] : a.b[i]) * o;
        if (NDOT >= 2) dots[1] += o * o;
      }
    }
  }
  if (NDOT > 0) grid_reduce_finalize<(NDOT > 0 ? NDOT : 1), RB_THREADS>(dots, a.partials, a.counter, a.ctl, a.fin);
}

// ------------------------------------------------------------------------------------------
// Row-vector fallback: LPR lanes per row (any row length, any aggregate size).
// ------------------------------------------------------------------------------------------
template <int OP, int NDOT, int LPR>
__global__ void __launch_bounds__(RB_THREADS) k_rowvec(RowArgs a) {
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
      for (int k = a.rowptr[i] + sub, e = a.rowptr[i + 1]; k < e; k += LPR) s += a.val[k] * gather_x<OP>(a, a.col[k]);
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
__global__ void k_restrict_rows(int nc, const int* __restrict__ agg_ptr, const double* __restrict__ r,
                                double* __restrict__ rc, const KrylovCtl* ctl) {
  if (ctl != nullptr && ctl->done) return;
  int I = blockIdx.x * blockDim.x + threadIdx.x;
  if (I >= nc) return;
  double s = 0.0;
  for (int t = agg_ptr[I]; t < agg_ptr[I + 1]; ++t) s += r[t];
  rc[I] = s;
}

// S4 standalone: x_i += gamma * ec[agg_i]
__global__ void k_prolong_add(int n, const int* __restrict__ agg, const double* __restrict__ ec, double gamma,
                              const double* __restrict__ xin, double* __restrict__ xout, const KrylovCtl* ctl) {
  if (ctl != nullptr && ctl->done) return;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) xout[i] = xin[i] + gamma * ec[agg[i]];
}

__global__ void k_scale_dinv(int n, const double* __restrict__ dinv, const double* __restrict__ b,
                             double* __restrict__ x, const KrylovCtl* ctl) {
  if (ctl != nullptr && ctl->done) return;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) x[i] = dinv[i] * b[i];
}

__global__ void k_zero(int n, double* __restrict__ x, const KrylovCtl* ctl) {
  if (ctl != nullptr && ctl->done) return;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) x[i] = 0.0;
}

// ------------------------------------------------------------------------------------------
// S5: coarsest solve with the dense LU factors (one CTA; y in shared memory)
// ------------------------------------------------------------------------------------------
__global__ void k_lu_solve(int n, const double* __restrict__ lu, const int* __restrict__ piv,
                           const double* __restrict__ b, double* __restrict__ x, const KrylovCtl* ctl) {
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

// ------------------------------------------------------------------------------------------
// S7/S8: fused Krylov vector kernels (grid-stride, one pass each, scalars read from KrylovCtl)
// ------------------------------------------------------------------------------------------
// r = b (permuted in), x = 0, optional extra vectors zeroed / copied; ||b||^2
__global__ void __launch_bounds__(RED_THREADS) k_krylov_init(int n, const double* __restrict__ b_nat,
                                                             const int* __restrict__ inv, double* __restrict__ r,
                                                             double* __restrict__ x, double* __restrict__ z0,
                                                             double* __restrict__ z1, double* __restrict__ rhat,
                                                             double* partials, unsigned* counter, KrylovCtl* ctl,
                                                             int fin) {
  double acc[1] = {0.0};
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * RED_THREADS) {
    const double v = b_nat[inv[i]];
    r[i] = v;
    x[i] = 0.0;
    if (z0) z0[i] = 0.0;
    if (z1) z1[i] = 0.0;
    if (rhat) rhat[i] = v;
    acc[0] += v * v;
  }
  grid_reduce_finalize<1, RED_THREADS>(acc, partials, counter, ctl, fin);
}

// p = z + beta p
__global__ void __launch_bounds__(RED_THREADS) k_pcg_p(int n, const double* __restrict__ z, double* __restrict__ p,
                                                       const KrylovCtl* ctl) {
  if (ctl->done) return;
  const double beta = ctl->beta;
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * RED_THREADS)
    p[i] = z[i] + beta * p[i];
}

// x += alpha p ; r -= alpha q ; ||r||^2
__global__ void __launch_bounds__(RED_THREADS) k_pcg_xr(int n, const double* __restrict__ p,
                                                        const double* __restrict__ q, double* __restrict__ x,
                                                        double* __restrict__ r, double* partials, unsigned* counter,
                                                        KrylovCtl* ctl) {
  if (ctl->done) return;
  const double alpha = ctl->alpha;
  double acc[1] = {0.0};
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * RED_THREADS) {
    x[i] += alpha * p[i];
    const double ri = r[i] - alpha * q[i];
    r[i] = ri;
    acc[0] += ri * ri;
  }
  grid_reduce_finalize<1, RED_THREADS>(acc, partials, counter, ctl, FIN_RR);
}

// sum a.b  (used when no smoother sweep can carry the r.z product)
__global__ void __launch_bounds__(RED_THREADS) k_dot(int n, const double* __restrict__ a, const double* __restrict__ b,
                                                     double* partials, unsigned* counter, KrylovCtl* ctl, int fin) {
  if (ctl->done) return;
  double acc[1] = {0.0};
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * RED_THREADS)
    acc[0] += a[i] * b[i];
  grid_reduce_finalize<1, RED_THREADS>(acc, partials, counter, ctl, fin);
}

// p = r + beta (p - omega v)
__global__ void __launch_bounds__(RED_THREADS) k_bicg_p(int n, const double* __restrict__ r,
                                                        const double* __restrict__ v, double* __restrict__ p,
                                                        const KrylovCtl* ctl) {
  if (ctl->done) return;
  const double beta = ctl->beta, omega = ctl->omega;
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * RED_THREADS)
    p[i] = r[i] + beta * (p[i] - omega * v[i]);
}

// s = r - alpha v ; ||s||^2
__global__ void __launch_bounds__(RED_THREADS) k_bicg_s(int n, const double* __restrict__ r,
                                                        const double* __restrict__ v, double* __restrict__ s,
                                                        double* partials, unsigned* counter, KrylovCtl* ctl) {
  if (ctl->done) return;
  const double alpha = ctl->alpha;
  double acc[1] = {0.0};
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * RED_THREADS) {
    const double si = r[i] - alpha * v[i];
    s[i] = si;
    acc[0] += si * si;
  }
  grid_reduce_finalize<1, RED_THREADS>(acc, partials, counter, ctl, FIN_SS);
}

// x += alpha phat + omega shat ; r = s - omega t ; ||r||^2 , rhat.r
__global__ void __launch_bounds__(RED_THREADS) k_bicg_xr(int n, const double* __restrict__ ph,
                                                         const double* __restrict__ sh, const double* __restrict__ s,
                                                         const double* __restrict__ t, const double* __restrict__ rhat,
                                                         double* __restrict__ x, double* __restrict__ r,
                                                         double* partials, unsigned* counter, KrylovCtl* ctl) {
  if (ctl->done) return;
  const double alpha = ctl->alpha, omega = ctl->omega;
  double acc[2] = {0.0, 0.0};
  for (int64_t i = (int64_t)blockIdx.x * RED_THREADS + threadIdx.x; i < n; i += (int64_t)gridDim.x * RED_THREADS) {
    x[i] += alpha * ph[i] + omega * sh[i];
    const double ri = s[i] - omega * t[i];
    r[i] = ri;
    acc[0] += ri * ri;
    acc[1] += rhat[i] * ri;
  }
  grid_reduce_finalize<2, RED_THREADS>(acc, partials, counter, ctl, FIN_RR_RHO);
}

// x_out (natural numbering) = x [+ alpha * phat after a BiCGSTAB half-step exit]
__global__ void k_krylov_output(int n, const double* __restrict__ x, const double* __restrict__ ph,
                                const int* __restrict__ inv, double* __restrict__ x_nat, const KrylovCtl* ctl) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double v = x[i];
  if (ph != nullptr && ctl->halfstep) v += ctl->alpha * ph[i];
  x_nat[inv[i]] = v;
}

__global__ void k_permute_in(int n, const double* __restrict__ nat, const int* __restrict__ inv,
                             double* __restrict__ out) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = nat[inv[i]];
}
__global__ void k_permute_out(int n, const double* __restrict__ in, const int* __restrict__ inv,
                              double* __restrict__ nat) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) nat[inv[i]] = in[i];
}

// ------------------------------------------------------------------------------------------
// G2: gA[k] (+)= - sum_s lambda_s[i] x_s[col[k]]  on the natural pattern; LPR lanes per row
// ------------------------------------------------------------------------------------------
template <int LPR>
__global__ void __launch_bounds__(256) k_grad_values(int n, const int* __restrict__ rowptr,
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
