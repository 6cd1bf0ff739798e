// Setup phase on the device: strength / row maxima, handshake matching,
// singleton merge + numbering, Galerkin product, smoother diagonal, dense LU of the coarsest
// operator, and the aggregate-contiguous renumbering of the whole hierarchy.
//
// The matching is the deterministic definition of DESIGN.md §readings (O-2): the result is a
// pure function of the matrix and the salt, independent of the thread schedule, so a sequential
// program following the same definition produces the same integers.
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>

#include "amg_internal.cuh"

namespace {

constexpr int TPB = 256;

inline double now_ms() {
  using namespace std::chrono;
  return duration<double, std::milli>(steady_clock::now().time_since_epoch()).count();
}

// ------------------------------------------------------------------------------------------
// exclusive scan of int32 (n inputs -> n+1 outputs, out[n] = total)
// ------------------------------------------------------------------------------------------
constexpr int SCAN_T = 512;
constexpr int SCAN_ITEMS = 4;
constexpr int SCAN_BLOCK = SCAN_T * SCAN_ITEMS;

__global__ void __launch_bounds__(SCAN_T) k_scan_block(const int* __restrict__ in, int* __restrict__ out,
                                                       int n, int* __restrict__ bsum) {
  __shared__ int wsum[32];
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const int64_t base = (int64_t)blockIdx.x * SCAN_BLOCK + tid * SCAN_ITEMS;
  int v[SCAN_ITEMS];
  int tsum = 0;
#pragma unroll
  for (int j = 0; j < SCAN_ITEMS; ++j) {
    int64_t idx = base + j;
    v[j] = idx < n ? in[idx] : 0;
    tsum += v[j];
  }
  int inc = tsum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) wsum[w] = inc;
  __syncthreads();
  if (w == 0) {
    int s = lane < SCAN_T / 32 ? wsum[lane] : 0;
    int inc2 = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int t = __shfl_up_sync(0xffffffffu, inc2, o);
      if (lane >= o) inc2 += t;
    }
    wsum[lane] = inc2 - s;
  }
  __syncthreads();
  int excl = wsum[w] + inc - tsum;
#pragma unroll
  for (int j = 0; j < SCAN_ITEMS; ++j) {
    int64_t idx = base + j;
    if (idx <= n) out[idx] = excl;
    excl += v[j];
  }
  if (tid == SCAN_T - 1 && bsum) bsum[blockIdx.x] = excl;
}

__global__ void k_scan_add(int* __restrict__ out, int n1, const int* __restrict__ boff) {
  int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx < n1) out[idx] += boff[idx / SCAN_BLOCK];
}

}  // namespace

amg_status amg_exclusive_scan(amg_handle_s* H, const int* d_in, int* d_out, int n, cudaStream_t st) {
  const int n1 = n + 1;
  const int nb = div_up(n1, SCAN_BLOCK);
  if (nb == 1) {
    k_scan_block<<<1, SCAN_T, 0, st>>>(d_in, d_out, n, nullptr);
    AMG_CUDA_TRY(H, cudaGetLastError());
    return AMG_OK;
  }
  int* bsum;
  AMG_ALLOC(H, bsum, int, nb + 1, st);
  k_scan_block<<<nb, SCAN_T, 0, st>>>(d_in, d_out, n, bsum);
  AMG_CUDA_TRY(H, cudaGetLastError());
  AMG_TRY(amg_exclusive_scan(H, bsum, bsum, nb, st));  // in place: every block reads before it writes
  k_scan_add<<<div_up(n1, TPB), TPB, 0, st>>>(d_out, n1, bsum);
  AMG_CUDA_TRY(H, cudaGetLastError());
  amg_dev_free(H, bsum);  // (frees are stream-ordered: no synchronisation)
  return AMG_OK;
}

namespace {

// ------------------------------------------------------------------------------------------
// validation
// ------------------------------------------------------------------------------------------
__global__ void k_validate_csr(int n, int nnz, const int* __restrict__ rowptr, const int* __restrict__ col,
                               const double* __restrict__ val, int* __restrict__ bad) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int s = rowptr[i], e = rowptr[i + 1];
  if (s < 0 || e < s || e > nnz) {
    *bad = 1;
    return;
  }
  bool diag = false;
  int prev = -1;
  for (int k = s; k < e; ++k) {
    int c = col[k];
    if (c < 0 || c >= n || c <= prev) {
      *bad = 1;
      return;
    }
    prev = c;
    if (c == i) diag = val[k] > 0.0;
  }
  if (!diag) *bad = 1;
}

// bitwise symmetry check: a_ij == a_ji for every stored entry (options.symmetric = -1)
__global__ void k_check_symmetric(int n, const int* __restrict__ rowptr, const int* __restrict__ col,
                                  const double* __restrict__ val, int* __restrict__ nonsym) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) {
    int j = col[k];
    int lo = rowptr[j], hi = rowptr[j + 1] - 1;
    bool found = false;
    while (lo <= hi) {
      int mid = (lo + hi) >> 1;
      int c = col[mid];
      if (c == i) {
        found = (val[mid] == val[k]);
        break;
      }
      if (c < i)
        lo = mid + 1;
      else
        hi = mid - 1;
    }
    if (!found) {
      *nonsym = 1;
      return;
    }
  }
}

// ------------------------------------------------------------------------------------------
// U1-U3: strength, handshake matching, singleton merge, numbering
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint64_t mix64(uint64_t z) {
  z ^= z >> 30;
  z *= 0xBF58476D1CE4E5B9ULL;
  z ^= z >> 27;
  z *= 0x94D049BB133111EBULL;
  z ^= z >> 31;
  return z;
}

struct EdgeKey {  // (-q, h, -lo, -hi): larger is better
  int q;
  uint64_t h;
  int lo, hi;
};

__device__ __forceinline__ bool key_better(const EdgeKey& a, const EdgeKey& b) {
  if (a.q != b.q) return a.q < b.q;
  if (a.h != b.h) return a.h > b.h;
  if (a.lo != b.lo) return a.lo < b.lo;
  return a.hi < b.hi;
}

// candidate test and key of the entry (i, j, a_ij); m = row maxima of w = -a
__device__ __forceinline__ bool edge_candidate(int i, int j, double aij, const double* __restrict__ m,
                                               double mi, double beta, uint64_t salt, EdgeKey& key) {
  if (j == i) return false;
  double w = -aij;
  if (!(w > 0.0)) return false;
  double mj = m[j];
  if (!(w >= beta * fmin(mi, mj))) return false;
  double M = fmax(mi, mj);
  key.q = (2.0 * w > M) ? 0 : ((4.0 * w > M) ? 1 : 2);
  int lo = min(i, j), hi = max(i, j);
  key.h = mix64((uint64_t)lo * 0x9E3779B97F4A7C15ULL + (uint64_t)hi * 0xBF58476D1CE4E5B9ULL + salt);
  key.lo = lo;
  key.hi = hi;
  return true;
}

__global__ void k_row_max(int n, const int* __restrict__ rowptr, const int* __restrict__ col,
                          const double* __restrict__ val, double* __restrict__ m) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double mi = 0.0;
  for (int k = rowptr[i]; k < rowptr[i + 1]; ++k)
    if (col[k] != i) mi = fmax(mi, fmax(-val[k], 0.0));
  m[i] = mi;
}

// every unmatched vertex points to its best unmatched candidate neighbour (state = match[])
__global__ void k_propose(int n, const int* __restrict__ rowptr, const int* __restrict__ col,
                          const double* __restrict__ val, const double* __restrict__ m, double beta,
                          uint64_t salt, int* __restrict__ match, int* __restrict__ ptr,
                          const int* __restrict__ prev_added) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  if (prev_added && *prev_added == 0) return;  // the matching was already maximal a round ago (rounds are queued ahead)
  int best_j = -1;
  if (match[i] == -1) {
    EdgeKey best{};
    double mi = m[i];
    for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) {
      int j = col[k];
      EdgeKey key;
      if (!edge_candidate(i, j, val[k], m, mi, beta, salt, key)) continue;
      if (match[j] >= 0) continue;
      if (best_j < 0 || key_better(key, best)) {
        best = key;
        best_j = j;
      }
    }
    // no unmatched candidate left: there will be none in any later round either (the matched set only grows), so the
    // row retires (-2: still "unmatched" for every reader) and later rounds skip its edge scan
    if (best_j < 0) match[i] = -2;
  }
  ptr[i] = best_j;
}

__global__ void k_handshake(int n, const int* __restrict__ ptr, int* __restrict__ match,
                            int* __restrict__ added, const int* __restrict__ prev_added) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  if (prev_added && *prev_added == 0) return;
  int j = ptr[i];
  if (j >= 0 && ptr[j] == i) {
    match[i] = j;
    if (i < j) atomicAdd(added, 1);
  }
}

// root of every vertex after the singleton merge (one simultaneous step) + root flags
__global__ void k_roots(int n, const int* __restrict__ rowptr, const int* __restrict__ col,
                        const double* __restrict__ val, const double* __restrict__ m, double beta,
                        uint64_t salt, const int* __restrict__ match, int* __restrict__ root,
                        int* __restrict__ isroot) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int mi_ = match[i];
  int r;
  if (mi_ >= 0) {
    r = min(i, mi_);
  } else {
    r = i;
    int best_j = -1;
    EdgeKey best{};
    double mi = m[i];
    for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) {
      int j = col[k];
      EdgeKey key;
      if (!edge_candidate(i, j, val[k], m, mi, beta, salt, key)) continue;
      if (match[j] < 0) continue;  // only matched neighbours
      if (best_j < 0 || key_better(key, best)) {
        best = key;
        best_j = j;
      }
    }
    if (best_j >= 0) r = min(best_j, match[best_j]);
  }
  root[i] = r;
  isroot[i] = (r == i) ? 1 : 0;
}

__global__ void k_assign_agg(int n, const int* __restrict__ root, const int* __restrict__ id,
                             int* __restrict__ agg) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) agg[i] = id[root[i]];
}

__global__ void k_fill_int(int n, int* __restrict__ a, int v) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) a[i] = v;
}

__global__ void k_iota(int n, int* __restrict__ a) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) a[i] = i;
}

__global__ void k_max_int(int n, const int* __restrict__ a, int* __restrict__ out, int* __restrict__ neg) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int v = a[i];
  if (v < 0) *neg = 1;
  atomicMax(out, v);
}

// member lists of the aggregates, ascending fine index inside each aggregate
__global__ void k_count_members(int n, const int* __restrict__ agg, int* __restrict__ cnt,
                                int* __restrict__ slot) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) slot[i] = atomicAdd(&cnt[agg[i]], 1);
}
__global__ void k_fill_members(int n, const int* __restrict__ agg, const int* __restrict__ mptr,
                               const int* __restrict__ slot, int* __restrict__ mem) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) mem[mptr[agg[i]] + slot[i]] = i;
}
__global__ void k_sort_members(int nc, const int* __restrict__ mptr, int* __restrict__ mem) {
  int I = blockIdx.x * blockDim.x + threadIdx.x;
  if (I >= nc) return;
  int s = mptr[I], e = mptr[I + 1];
  for (int a = s + 1; a < e; ++a) {
    int v = mem[a];
    int b = a - 1;
    while (b >= s && mem[b] > v) {
      mem[b + 1] = mem[b];
      --b;
    }
    mem[b + 1] = v;
  }
}

// ------------------------------------------------------------------------------------------
// U4: Galerkin product with piecewise-constant P:  A_c[I,J] = sum_{i in I} sum_{j in J} a_ij
// one thread per coarse row keeps a sorted list of (J, sum) in a scratch segment; the sum of
// every (I,J) runs over ascending fine row, then ascending position (fixed order).
// ------------------------------------------------------------------------------------------
__global__ void k_rap_len(int nc, const int* __restrict__ mptr, const int* __restrict__ mem,
                          const int* __restrict__ rowptr, int* __restrict__ len) {
  int I = blockIdx.x * blockDim.x + threadIdx.x;
  if (I >= nc) return;
  int s = 0;
  for (int t = mptr[I]; t < mptr[I + 1]; ++t) {
    int i = mem[t];
    s += rowptr[i + 1] - rowptr[i];
  }
  len[I] = s;
}

// serial form (one lane): also the path of a coarse row whose segment does not fit the group's shared lists
__device__ void rap_row_serial(int I, const int* __restrict__ mptr, const int* __restrict__ mem,
                               const int* __restrict__ rowptr, const int* __restrict__ col,
                               const double* __restrict__ val, const int* __restrict__ agg, int* __restrict__ key,
                               double* __restrict__ acc, int* __restrict__ cnt) {
  int m = 0;  // entries in the sorted list
  for (int t = mptr[I]; t < mptr[I + 1]; ++t) {
    int i = mem[t];
    for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) {
      int J = agg[col[k]];
      double a = val[k];
      int p = m;  // find the slot from the back (columns arrive almost sorted)
      while (p > 0 && key[p - 1] > J) --p;
      if (p > 0 && key[p - 1] == J) {
        acc[p - 1] += a;
      } else {
        for (int q = m; q > p; --q) {
          key[q] = key[q - 1];
          acc[q] = acc[q - 1];
        }
        key[p] = J;
        acc[p] = a;
        ++m;
      }
    }
  }
  cnt[I] = m;
}

// G lanes per coarse row.  The entries (J, a) of the members' rows are listed in shared memory in the fixed order
// (ascending fine row, ascending position), ranked by a STABLE counting sort on J (every lane compares its entry with
// all others: the lists are short), and every distinct J is summed by one lane from its first entry on: the same
// additions in the same order as the serial form, so the values are bit-equal to it.
constexpr int RAP_THREADS = 128;
template <int G, int CAP>
__global__ void __launch_bounds__(RAP_THREADS)
    k_rap_rows(int nc, const int* __restrict__ mptr, const int* __restrict__ mem, const int* __restrict__ rowptr,
               const int* __restrict__ col, const double* __restrict__ val, const int* __restrict__ agg,
               const int* __restrict__ segptr, int* __restrict__ skey, double* __restrict__ sval,
               int* __restrict__ cnt) {
  constexpr int GROUPS = RAP_THREADS / G;
  __shared__ int uk[GROUPS][CAP], sk[GROUPS][CAP];
  __shared__ double uv[GROUPS][CAP], sv[GROUPS][CAP];
  __shared__ int mr0[GROUPS][G], mend[GROUPS][G];
  const int g = threadIdx.x / G, lane = threadIdx.x % G;
  constexpr unsigned LOW = (unsigned)((1ull << G) - 1ull);  // G lanes
  const int shift = (threadIdx.x % 32) / G * G;
  const unsigned gmask = LOW << shift;
  const int I = blockIdx.x * GROUPS + g;
  if (I >= nc) return;  // whole groups leave together
  const int seg = segptr[I], L = segptr[I + 1] - seg;
  if (L > CAP) {
    if (lane == 0) rap_row_serial(I, mptr, mem, rowptr, col, val, agg, skey + seg, sval + seg, cnt);
    return;
  }
  const int m0 = mptr[I], nm = mptr[I + 1] - m0;
  if (nm <= G) {
    // lane t holds member t's row start and its offset in the list: the entries of all members load at once
    int r0 = 0, len = 0;
    if (lane < nm) {
      const int i = mem[m0 + lane];
      r0 = rowptr[i];
      len = rowptr[i + 1] - r0;
    }
    int incl = len;
#pragma unroll
    for (int d = 1; d < G; d <<= 1) {
      const int v = __shfl_up_sync(gmask, incl, d, G);
      if (lane >= d) incl += v;
    }
    mr0[g][lane] = r0 - (incl - len);  // entry e of member t sits at mr0[t] + e
    mend[g][lane] = incl;             // one past member t's last entry
    __syncwarp(gmask);
    for (int e = lane; e < L; e += G) {
      int t = 0;
      while (mend[g][t] <= e) ++t;
      const int k = mr0[g][t] + e;
      uk[g][e] = agg[col[k]];
      uv[g][e] = val[k];
    }
  } else {
    int off = 0;
    for (int t = m0; t < m0 + nm; ++t) {
      const int i = mem[t], r0 = rowptr[i], len = rowptr[i + 1] - r0;
      for (int k = lane; k < len; k += G) {
        uk[g][off + k] = agg[col[r0 + k]];
        uv[g][off + k] = val[r0 + k];
      }
      off += len;
    }
  }
  __syncwarp(gmask);
  for (int e = lane; e < L; e += G) {
    const int J = uk[g][e];
    int r = 0;
    for (int f = 0; f < L; ++f) {
      const int K = uk[g][f];
      r += (K < J) | ((K == J) & (f < e));
    }
    sk[g][r] = J;
    sv[g][r] = uv[g][e];
  }
  __syncwarp(gmask);
  int base = 0;
  for (int r0 = 0; r0 < L; r0 += G) {  // uniform trip count inside the group
    const int r = r0 + lane;
    const bool head = r < L && (r == 0 || sk[g][r - 1] != sk[g][r]);
    const unsigned heads = (__ballot_sync(gmask, head) & gmask) >> shift;
    if (head) {
      const int J = sk[g][r];
      double a = sv[g][r];
      for (int q = r + 1; q < L && sk[g][q] == J; ++q) a += sv[g][q];
      const int pos = base + __popc(heads & ((1u << lane) - 1u));
      skey[seg + pos] = J;
      sval[seg + pos] = a;
    }
    base += __popc(heads);
  }
  if (lane == 0) cnt[I] = base;
}

__global__ void k_rap_compact(int nc, const int* __restrict__ segptr, const int* __restrict__ skey,
                              const double* __restrict__ sval, const int* __restrict__ crowptr,
                              int* __restrict__ ccol, double* __restrict__ cval) {
  int I = blockIdx.x * blockDim.x + threadIdx.x;
  if (I >= nc) return;
  int s = segptr[I], d = crowptr[I], m = crowptr[I + 1] - d;
  for (int t = 0; t < m; ++t) {
    ccol[d + t] = skey[s + t];
    cval[d + t] = sval[s + t];
  }
}

// U5: smoother diagonal
__global__ void k_dinv(int n, const int* __restrict__ rowptr, const int* __restrict__ col,
                       const double* __restrict__ val, int smoother, double omega, double* __restrict__ dinv) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double l1 = 0.0, aii = 0.0;
  for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) {
    l1 += fabs(val[k]);
    if (col[k] == i) aii = val[k];
  }
  dinv[i] = smoother == 1 ? omega / aii : 1.0 / l1;  // 0 and 2 (Chebyshev-accelerated L1-Jacobi): the l1 diagonal
}

// ------------------------------------------------------------------------------------------
// U6: dense LU with partial pivoting of the coarsest operator (one CTA)
// ------------------------------------------------------------------------------------------
__global__ void k_csr_to_dense(int n, const int* __restrict__ rowptr, const int* __restrict__ col,
                               const double* __restrict__ val, double* __restrict__ a) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) a[(size_t)i * n + col[k]] = val[k];
}

__global__ void __launch_bounds__(1024) k_dense_lu(int n, double* __restrict__ a, int* __restrict__ piv,
                                                   int* __restrict__ info) {
  __shared__ double s_val[32];
  __shared__ int s_idx[32];
  __shared__ double s_amax;
  __shared__ int s_p;
  const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, w = tid >> 5;
  // amax = max |a_ij|
  double mx = 0.0;
  for (size_t t = tid; t < (size_t)n * n; t += T) mx = fmax(mx, fabs(a[t]));
  for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if (lane == 0) s_val[w] = mx;
  __syncthreads();
  if (tid == 0) {
    double v = 0.0;
    for (int q = 0; q < (T + 31) / 32; ++q) v = fmax(v, s_val[q]);
    s_amax = v;
  }
  __syncthreads();
  const double amax = s_amax;
  for (int k = 0; k < n; ++k) {
    // pivot: first row i >= k with the largest |a_ik|
    double bv = -1.0;
    int bi = n;
    for (int i = k + tid; i < n; i += T) {
      double v = fabs(a[(size_t)i * n + k]);
      if (v > bv) {
        bv = v;
        bi = i;
      }
    }
    for (int o = 16; o > 0; o >>= 1) {
      double ov = __shfl_xor_sync(0xffffffffu, bv, o);
      int oi = __shfl_xor_sync(0xffffffffu, bi, o);
      if (ov > bv || (ov == bv && oi < bi)) {
        bv = ov;
        bi = oi;
      }
    }
    if (lane == 0) {
      s_val[w] = bv;
      s_idx[w] = bi;
    }
    __syncthreads();
    if (tid == 0) {
      double v = -1.0;
      int p = n;
      for (int q = 0; q < (T + 31) / 32; ++q)
        if (s_val[q] > v || (s_val[q] == v && s_idx[q] < p)) {
          v = s_val[q];
          p = s_idx[q];
        }
      if (!(v > 1e-300 * amax) || !(amax > 0.0)) {
        *info = 1;
        p = k;
      }
      piv[k] = p;
      s_p = p;
    }
    __syncthreads();
    const int p = s_p;
    if (p != k)
      for (int j = tid; j < n; j += T) {
        double t = a[(size_t)k * n + j];
        a[(size_t)k * n + j] = a[(size_t)p * n + j];
        a[(size_t)p * n + j] = t;
      }
    __syncthreads();
    const double akk = a[(size_t)k * n + k];
    for (int i = k + 1 + tid; i < n; i += T) a[(size_t)i * n + k] = a[(size_t)i * n + k] / akk;
    __syncthreads();
    const int mrem = n - k - 1;
    for (int64_t t = tid; t < (int64_t)mrem * mrem; t += T) {
      int i = k + 1 + (int)(t / mrem), j = k + 1 + (int)(t % mrem);
      a[(size_t)i * n + j] -= a[(size_t)i * n + k] * a[(size_t)k * n + j];
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------
// aggregate-contiguous renumbering
// ------------------------------------------------------------------------------------------
__global__ void k_perm_sizes(int nc, const int* __restrict__ mptr, const int* __restrict__ pos_next,
                             int* __restrict__ sizep) {
  int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a < nc) sizep[pos_next[a]] = mptr[a + 1] - mptr[a];
}

__global__ void k_perm_pos(int nc, const int* __restrict__ mptr, const int* __restrict__ mem,
                           const int* __restrict__ pos_next, const int* __restrict__ startp,
                           int* __restrict__ pos, int* __restrict__ inv, int* __restrict__ aggp) {
  int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= nc) return;
  int ap = pos_next[a];
  int base = startp[ap];
  for (int t = mptr[a]; t < mptr[a + 1]; ++t) {
    int i = mem[t];
    int p = base + (t - mptr[a]);
    pos[i] = p;
    inv[p] = i;
    aggp[p] = ap;
  }
}

__global__ void k_perm_rowlen(int n, const int* __restrict__ rowptr, const int* __restrict__ src_row,
                              int* __restrict__ len) {
  int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  int i = src_row[p];
  len[p] = rowptr[i + 1] - rowptr[i];
}

// row p of the output is row src_row[p] of the input with columns relabelled by col_map and
// re-sorted ascending
// G lanes per output row: the mapped columns are ranked in shared memory (a permutation keeps them distinct) and
// written in ascending order; a row longer than CAP is insertion-sorted in place by one lane
template <int G, int CAP>
__global__ void __launch_bounds__(128)
    k_perm_fill(int n, const int* __restrict__ rowptr, const int* __restrict__ col, const double* __restrict__ val,
                const int* __restrict__ src_row, const int* __restrict__ col_map,
                const int* __restrict__ rowptr_out, int* __restrict__ col_out, double* __restrict__ val_out) {
  constexpr int GROUPS = 128 / G;
  __shared__ int uk[GROUPS][CAP];
  __shared__ double uv[GROUPS][CAP];
  const int g = threadIdx.x / G, lane = threadIdx.x % G;
  constexpr unsigned LOW = (unsigned)((1ull << G) - 1ull);
  const unsigned gmask = LOW << ((threadIdx.x % 32) / G * G);
  const int p = blockIdx.x * GROUPS + g;
  if (p >= n) return;
  const int i = src_row[p];
  const int s = rowptr[i], len = rowptr[i + 1] - s, d = rowptr_out[p];
  if (len > CAP) {
    if (lane != 0) return;
    for (int m = 0; m < len; ++m) {
      int c = col_map[col[s + m]];
      double v = val[s + m];
      int q = m;
      while (q > 0 && col_out[d + q - 1] > c) {
        col_out[d + q] = col_out[d + q - 1];
        val_out[d + q] = val_out[d + q - 1];
        --q;
      }
      col_out[d + q] = c;
      val_out[d + q] = v;
    }
    return;
  }
  for (int k = lane; k < len; k += G) {
    uk[g][k] = col_map[col[s + k]];
    uv[g][k] = val[s + k];
  }
  __syncwarp(gmask);
  for (int e = lane; e < len; e += G) {
    const int c = uk[g][e];
    int r = 0;
    for (int f = 0; f < len; ++f) r += uk[g][f] < c;
    col_out[d + r] = c;
    val_out[d + r] = uv[g][e];
  }
}

__global__ void k_gather_double(int n, const double* __restrict__ src, const int* __restrict__ idx,
                                double* __restrict__ dst) {
  int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p < n) dst[p] = src[idx[p]];
}

// Row-tile partition by shared-memory bytes: a row weighs RT_ROW_WEIGHT bytes of staged row
// operands, a nonzero RT_NNZ_WEIGHT (value, 16-bit column, its share of the halo list and values).  Tile k starts at the first unit (aggregate, or row if
// unit_ptr == null) whose cumulative weight is at or beyond k * target.
constexpr int RT_ROW_WEIGHT = 24;
__device__ __forceinline__ int64_t tile_weight(const int* __restrict__ rowptr, int r, int nnz_w) {
  return nnz_w * (int64_t)rowptr[r] + (int64_t)RT_ROW_WEIGHT * r;
}
__global__ void k_blk_partition(int nblk, int target, int nnz_w, int nunits, const int* __restrict__ unit_ptr,
                                const int* __restrict__ rowptr, int n, int* __restrict__ blk_ptr) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k > nblk) return;
  if (k == nblk) {
    blk_ptr[k] = n;
    return;
  }
  int64_t want = (int64_t)k * target;
  int lo = 0, hi = nunits;  // smallest u in [0, nunits] with rowptr[start(u)] >= want
  while (lo < hi) {
    int mid = (lo + hi) >> 1;
    int r = unit_ptr ? unit_ptr[mid] : mid;
    if (tile_weight(rowptr, r, nnz_w) >= want)
      hi = mid;
    else
      lo = mid + 1;
  }
  blk_ptr[k] = lo == nunits ? n : (unit_ptr ? unit_ptr[lo] : lo);
}

// ------------------------------------------------------------------------------------------
// Tile packer (amg_tilepack.cuh): one CTA per tile.  Pass 1 (write == 0) sizes every tile: rows
// sorted by descending length (stable), slice widths, the sorted list of distinct out-of-tile
// columns; pass 2 (after a scan of the blob sizes) repeats that and writes the blob.
// info[0] = largest stage footprint (bytes), info[1] = a tile exceeds the packer's scratch
// ------------------------------------------------------------------------------------------
// ------------------------------------------------------------------------------------------
// Value dictionary of a level (amg_options::value_dict): the distinct fp64 values of its operator, if there are
// at most VD_MAX of them -- constant-coefficient stencils and their Galerkin sums hold a handful.  The tile blobs
// of such a level store an 8-bit code per entry instead of the value (3 bytes per entry instead of 10); the
// kernels look the value up in a 256-entry table in shared memory: the same fp64 value, bit for bit.
// Distinct values are collected in a small open-addressing hash table (the insertion stops at the first overflow:
// a level with all-different values costs a few thousand probes), then sorted ascending, so that the codes are a
// function of the value set alone.  Code 255 is 0.0: the padding slots of the tiles.
// ------------------------------------------------------------------------------------------
constexpr int VD_SLOTS = 1024, VD_MAX = 255;
constexpr unsigned long long VD_EMPTY = 0xFFFFFFFFFFFFFFFFull;  // (a NaN pattern: never a validated matrix value)
__global__ void k_vdict_insert(int nnz, const double* __restrict__ val, unsigned long long* table, int* count) {
  volatile int* over = count + 1;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < nnz; i += gridDim.x * blockDim.x) {
    if (*over) return;
    const unsigned long long key = (unsigned long long)__double_as_longlong(val[i]);
    unsigned h = (unsigned)(mix64(key) & (VD_SLOTS - 1));
    bool placed = false;
    // at most VD_MAX keys in VD_SLOTS slots: a probe sequence longer than 64 means the table is being flooded
    for (int probe = 0; probe < 64 && !placed; ++probe) {
      unsigned long long cur = *((volatile unsigned long long*)(table + h));
      if (cur == VD_EMPTY) {
        if (*over) return;
        cur = atomicCAS(table + h, VD_EMPTY, key);
        if (cur == VD_EMPTY) {
          if (atomicAdd(count, 1) + 1 > VD_MAX) *over = 1;
          placed = true;
        }
      }
      if (cur == key) placed = true;
      h = (h + 1) & (VD_SLOTS - 1);
    }
    if (!placed) {
      *over = 1;
      return;
    }
  }
}
// one CTA of VD_SLOTS threads: the keys sorted ascending as doubles -> dict[0 .. count), dict[255] = 0
__global__ void __launch_bounds__(VD_SLOTS) k_vdict_finalize(const unsigned long long* __restrict__ table,
                                                             const int* __restrict__ count, double* __restrict__ dict) {
  __shared__ double v[VD_SLOTS];
  const int tid = threadIdx.x;
  const unsigned long long key = table[tid];
  v[tid] = key == VD_EMPTY ? __longlong_as_double(0x7FF0000000000000ll) : __longlong_as_double((long long)key);
  __syncthreads();
  for (int k = 2; k <= VD_SLOTS; k <<= 1)
    for (int j = k >> 1; j > 0; j >>= 1) {
      const int p = tid ^ j;
      if (p > tid) {
        const double a = v[tid], b = v[p];
        const bool asc = (tid & k) == 0;
        if ((a > b) == asc) v[tid] = b, v[p] = a;
      }
      __syncthreads();
    }
  if (tid < 256) dict[tid] = (tid < *count && tid < VD_MAX) ? v[tid] : 0.0;
}
// code of a value: its position in the ascending dictionary (exact match by construction)
__device__ __forceinline__ unsigned char vdict_code(const double* dict, int ndict, double v) {
  int lo = 0, hi = ndict;  // first entry >= v
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (dict[mid] < v) lo = mid + 1;
    else hi = mid;
  }
  return (unsigned char)lo;
}

constexpr int PK_THREADS = 256;
constexpr int PK_MAX_LEN = 512;
__global__ void __launch_bounds__(PK_THREADS) k_pack_tiles(int ntiles, const int* __restrict__ blk_ptr,
                                                           const int* __restrict__ rowptr, const int* __restrict__ col,
                                                           const double* __restrict__ val, const int* __restrict__ agg,
                                                           int vb, int write, const int* __restrict__ blob_off16,
                                                           const int* __restrict__ halo_off, int* __restrict__ size16,
                                                           int* __restrict__ nhalo_out, int* __restrict__ info,
                                                           TileDesc* __restrict__ tiles, unsigned char* __restrict__ blob,
                                                           int* __restrict__ halo_idx, int* __restrict__ halo_cagg,
                                                           const double* __restrict__ vdict, int ndict) {
  __shared__ int ext[RT_MAX_NNZ];
  __shared__ int halo[RT_MAX_NNZ];
  __shared__ int len[RT_MAX_ROWS];
  __shared__ int srow[RT_MAX_ROWS];
  __shared__ int hist[PK_MAX_LEN + 1];
  __shared__ int sl_off[RT_MAX_ROWS / 32 + 1], sl_w[RT_MAX_ROWS / 32 + 1];
  __shared__ int cnts[PK_THREADS];
  __shared__ int s_cnt, s_nhalo, s_maxlen, s_nslots;
  const int t = blockIdx.x, tid = threadIdx.x;
  if (t >= ntiles) return;
  const int r0 = blk_ptr[t], r1 = blk_ptr[t + 1], nr = r1 - r0;
  TileDesc d;
  d.r0 = r0, d.nr = nr, d.I0 = 0, d.nA = 0, d.nsl = 0, d.nslots = 0, d.nhalo = 0, d.blob16 = 0;
  d.halo_off = 0, d.vb = vb, d.pad1 = d.pad2 = 0;
  if (nr <= 0) {
    if (tid == 0) {
      if (write) tiles[t] = d;
      else size16[t] = 0, nhalo_out[t] = 0;
    }
    return;
  }
  const int k0 = rowptr[r0], k1 = rowptr[r1];
  if (nr > RT_MAX_ROWS || k1 - k0 > RT_MAX_NNZ) {
    if (tid == 0) {
      info[1] = 1;
      if (!write) size16[t] = 0, nhalo_out[t] = 0;
    }
    return;
  }
  if (agg != nullptr) {
    d.I0 = agg[r0];
    d.nA = agg[r1 - 1] - d.I0 + 1;
  }
  if (tid == 0) s_cnt = 0, s_maxlen = 0;
  for (int q = tid; q <= PK_MAX_LEN; q += PK_THREADS) hist[q] = 0;
  __syncthreads();
  for (int lr = tid; lr < nr; lr += PK_THREADS) {
    const int l = rowptr[r0 + lr + 1] - rowptr[r0 + lr];
    len[lr] = l;
    atomicMax(&s_maxlen, l);
    if (l <= PK_MAX_LEN) atomicAdd(&hist[l], 1);
  }
  for (int k = k0 + tid; k < k1; k += PK_THREADS) {
    const int c = col[k];
    if (c < r0 || c >= r1) ext[atomicAdd(&s_cnt, 1)] = c;
  }
  __syncthreads();
  if (s_maxlen > PK_MAX_LEN) {
    if (tid == 0) {
      info[1] = 1;
      if (!write) size16[t] = 0, nhalo_out[t] = 0;
    }
    return;
  }
  const int nsl = (nr + 31) >> 5;
  if (tid == 0) {
    // stable counting sort by descending length: hist[l] = first sorted position of the rows of length l
    int acc = 0;
    for (int l = s_maxlen; l >= 0; --l) {
      const int c = hist[l];
      hist[l] = acc;
      acc += c;
    }
  }
  __syncthreads();
  // sorted position of a row = first position of its length + the rows of that length before it (every thread walks
  // len[] with the same index: broadcast reads)
  for (int lr = tid; lr < nr; lr += PK_THREADS) {
    const int l = len[lr];
    int before = 0;
    for (int q = 0; q < lr; ++q) before += (len[q] == l);
    srow[hist[l] + before] = lr;
  }
  __syncthreads();
  if (tid == 0) {  // slice widths = length of the slice's first row
    int off = 0;
    for (int j = 0; j < nsl; ++j) {
      const int w = len[srow[j * 32]];
      sl_off[j] = off;
      sl_w[j] = w;
      off += 32 * w;
    }
    sl_off[nsl] = off;
    s_nslots = off;
  }
  // sort the out-of-tile columns (bitonic, padded with INT_MAX), then keep the distinct ones
  const int cnt = s_cnt;
  int N = 1;
  while (N < cnt) N <<= 1;
  for (int i = cnt + tid; i < N; i += PK_THREADS) ext[i] = 0x7fffffff;
  __syncthreads();
  for (int k = 2; k <= N; k <<= 1)
    for (int j = k >> 1; j > 0; j >>= 1) {
      for (int i = tid; i < N; i += PK_THREADS) {
        const int p = i ^ j;
        if (p > i) {
          const int a = ext[i], b = ext[p];
          const bool asc = (i & k) == 0;
          if ((a > b) == asc) {
            ext[i] = b;
            ext[p] = a;
          }
        }
      }
      __syncthreads();
    }
  {
    const int chunk = (cnt + PK_THREADS - 1) / PK_THREADS;
    const int b = tid * chunk, e = min(cnt, b + chunk);
    int c = 0;
    for (int i = b; i < e; ++i) c += (i == 0 || ext[i] != ext[i - 1]);
    cnts[tid] = c;
    __syncthreads();
    if (tid == 0) {
      int acc = 0;
      for (int q = 0; q < PK_THREADS; ++q) {
        const int v = cnts[q];
        cnts[q] = acc;
        acc += v;
      }
      s_nhalo = acc;
    }
    __syncthreads();
    int o = cnts[tid];
    for (int i = b; i < e; ++i)
      if (i == 0 || ext[i] != ext[i - 1]) halo[o++] = ext[i];
  }
  __syncthreads();
  d.nsl = nsl, d.nslots = s_nslots, d.nhalo = s_nhalo;
  const BlobLayout p = tp_blob(d.nsl, d.nslots, vb);
  if (!write) {
    if (tid == 0) {
      size16[t] = p.end / 16;
      nhalo_out[t] = d.nhalo;
      atomicMax(&info[0], tp_stage_need(d));
      atomicMax(&info[2], tp_xslot_need(d));
    }
    return;
  }
  d.blob16 = (uint32_t)blob_off16[t];
  d.halo_off = halo_off[t];
  unsigned char* base = blob + (size_t)d.blob16 * 16u;
  if (tid == 0) tiles[t] = d;
  int2* o_sl = reinterpret_cast<int2*>(base);
  for (int j = tid; j < nsl; j += PK_THREADS) o_sl[j] = make_int2(sl_off[j], sl_w[j]);
  for (int h = tid; h < d.nhalo; h += PK_THREADS) {
    const int c = halo[h];
    halo_idx[d.halo_off + h] = c;
    halo_cagg[d.halo_off + h] = agg != nullptr ? agg[c] : 0;
  }
  unsigned short* o_perm = reinterpret_cast<unsigned short*>(base + p.o_perm);
  for (int s = tid; s < nsl * 32; s += PK_THREADS) o_perm[s] = s < nr ? (unsigned short)srow[s] : (unsigned short)0xFFFF;
  unsigned short* o_col = reinterpret_cast<unsigned short*>(base + p.o_col);
  double* o_val = reinterpret_cast<double*>(base + p.o_val);
  float* o_val32 = reinterpret_cast<float*>(base + p.o_val);  // vb == 4: mixed-precision hierarchy
  uint32_t* o_cw = reinterpret_cast<uint32_t*>(base + p.o_col);  // vb == 1: column | dictionary code << 16
  // tile-local column of every entry of the tile, one thread per entry (ext[] is free again: reused as u16[])
  unsigned short* c16s = reinterpret_cast<unsigned short*>(ext);
  __syncthreads();
  for (int e = tid; e < k1 - k0; e += PK_THREADS) {
    const int c = col[k0 + e];
    unsigned short c16;
    if (c >= r0 && c < r1) {
      c16 = (unsigned short)(c - r0);
    } else {
      int lo = 0, hi = d.nhalo;  // first entry >= c
      while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (halo[mid] < c) lo = mid + 1;
        else hi = mid;
      }
      c16 = (unsigned short)(nr + lo);
    }
    c16s[e] = c16;
  }
  __syncthreads();
  // One thread per row (sorted position s = slice j, lane): its entries in slots k = 0 .. w_j - 1, zero-padded past
  // the row's length; the stores of a warp for a fixed k are contiguous.
  // ORDER of a row's entries (any order is a valid row sum; this one is fixed by the pattern alone): the batched
  // kernel reads, per entry, the 64 bytes [8 right-hand sides] of the entry's column from shared memory, 16 lanes at
  // a time; the columns of a tile sit 64 bytes apart from a 128-byte aligned base (own rows: stage; halo columns:
  // x slot), so a column's CLASS = parity of its position there decides which half of the 128-byte bank line it
  // occupies.  Lane `lane` wants class (lane ^ k) & 1 at step k: then every 16-byte bank group is read by exactly 2
  // of the 16 lanes (the minimum).  Each row serves the wanted class from its remaining entries in ascending CSR
  // position, and falls back to the other class when that one is exhausted.
  for (int s = tid; s < nsl * 32; s += PK_THREADS) {
    const int j = s >> 5, lane = s & 31;
    const int off = sl_off[j] + lane, w = sl_w[j];
    int ln = 0, kk0 = 0;
    if (s < nr) {
      const int lr = srow[s];
      ln = len[lr];
      kk0 = rowptr[r0 + lr];
    }
    const unsigned short* rc = c16s + (kk0 - k0);
    auto cls = [&](int q) {
      const int c = rc[q];
      return (c < nr ? c : c - nr) & 1;
    };
    int cur[2] = {0, 0};  // next unserved entry of class 0 / 1
    while (cur[0] < ln && cls(cur[0]) != 0) ++cur[0];
    while (cur[1] < ln && cls(cur[1]) != 1) ++cur[1];
    for (int k = 0; k < w; ++k) {
      unsigned short c16 = 0;
      double v = 0.0;
      if (k < ln) {
        int t = (lane ^ k) & 1;
        if (cur[t] >= ln) t ^= 1;
        const int q = cur[t];
        c16 = rc[q];
        v = val[kk0 + q];
        int nx = q + 1;
        while (nx < ln && cls(nx) != t) ++nx;
        cur[t] = nx;
      }
      if (vb == 1) {
        o_cw[off + k * 32] = (uint32_t)c16 | ((uint32_t)(k < ln ? vdict_code(vdict, ndict, v) : (unsigned char)255) << 16);
        continue;
      }
      o_col[off + k * 32] = c16;
      if (vb == 4)
        o_val32[off + k * 32] = (float)v;
      else
        o_val[off + k * 32] = v;
    }
  }
  // tail of the u16 column section up to its 16-byte rounding
  if (vb != 1)
    for (int q = d.nslots + tid; q < tp_up(2 * d.nslots, 16) / 2; q += PK_THREADS) o_col[q] = 0;
}

__global__ void k_pad_tail(int nnz, int nnz_alloc, int* __restrict__ col, double* __restrict__ val) {
  int k = nnz + blockIdx.x * blockDim.x + threadIdx.x;
  if (k < nnz_alloc) {
    col[k] = 0;
    val[k] = 0.0;
  }
}

inline int grid_for(int n) { return n > 0 ? div_up(n, TPB) : 1; }

amg_status read_int(amg_handle_s* H, const int* d, int* h, cudaStream_t st) {
  AMG_CUDA_TRY(H, cudaMemcpyAsync(h, d, sizeof(int), cudaMemcpyDeviceToHost, st));
  AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
  return AMG_OK;
}

// ------------------------------------------------------------------------------------------
// CSR transpose on the device (NEXT-2; the paper calls cuSPARSE for it): count ->
// scan -> fill (atomic cursors: arbitrary order inside a row) -> per-row sort by column, which makes
// the result unique.  src[p] = position in the input the entry p came from: a value-only update
// re-transposes with one gather.
// ------------------------------------------------------------------------------------------
__global__ void k_tr_count(int nnz, const int* __restrict__ col, int* __restrict__ cnt) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k < nnz) atomicAdd(&cnt[col[k]], 1);
}
__global__ void k_tr_fill(int n, const int* __restrict__ rowptr, const int* __restrict__ col,
                          const int* __restrict__ tptr, int* __restrict__ cursor, int* __restrict__ tcol,
                          int* __restrict__ tsrc) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) {
    const int j = col[k];
    const int p = tptr[j] + atomicAdd(&cursor[j], 1);
    tcol[p] = i;
    tsrc[p] = k;
  }
}
__global__ void k_tr_sort(int n, const int* __restrict__ tptr, int* __restrict__ tcol, int* __restrict__ tsrc) {
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  const int s = tptr[j], e = tptr[j + 1];
  for (int a = s + 1; a < e; ++a) {
    const int c = tcol[a], k = tsrc[a];
    int b = a - 1;
    while (b >= s && tcol[b] > c) {
      tcol[b + 1] = tcol[b];
      tsrc[b + 1] = tsrc[b];
      --b;
    }
    tcol[b + 1] = c;
    tsrc[b + 1] = k;
  }
}
__global__ void k_gather_vals(int nnz, const double* __restrict__ val, const int* __restrict__ src,
                              double* __restrict__ out) {
  int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p < nnz) out[p] = val[src[p]];
}

// outputs are allocated here: trowptr[n+1], tcol / tval [nnz_alloc], tsrc[nnz]
amg_status transpose_csr(amg_handle_s* H, int n, int nnz, int nnz_alloc, const int* rowptr, const int* col,
                         const double* val, int** trowptr, int** tcol, double** tval, int** tsrc, cudaStream_t st) {
  int* cnt;
  AMG_ALLOC(H, cnt, int, n + 1, st);
  AMG_ALLOC(H, *trowptr, int, n + 1, st);
  AMG_ALLOC(H, *tcol, int, nnz_alloc, st);
  AMG_ALLOC(H, *tval, double, nnz_alloc, st);
  AMG_ALLOC(H, *tsrc, int, nnz, st);
  AMG_CUDA_TRY(H, cudaMemsetAsync(cnt, 0, sizeof(int) * (n + 1), st));
  k_tr_count<<<grid_for(nnz), TPB, 0, st>>>(nnz, col, cnt);
  AMG_CUDA_TRY(H, cudaGetLastError());
  AMG_TRY(amg_exclusive_scan(H, cnt, *trowptr, n, st));
  AMG_CUDA_TRY(H, cudaMemsetAsync(cnt, 0, sizeof(int) * (n + 1), st));
  k_tr_fill<<<grid_for(n), TPB, 0, st>>>(n, rowptr, col, *trowptr, cnt, *tcol, *tsrc);
  k_tr_sort<<<grid_for(n), TPB, 0, st>>>(n, *trowptr, *tcol, *tsrc);
  k_gather_vals<<<grid_for(nnz), TPB, 0, st>>>(nnz, val, *tsrc, *tval);
  if (nnz_alloc > nnz) k_pad_tail<<<1, 32, 0, st>>>(nnz, nnz_alloc, *tcol, *tval);
  AMG_CUDA_TRY(H, cudaGetLastError());
  amg_dev_free(H, cnt);
  return AMG_OK;
}

// S = (A + A^T) / 2 on the union of the two patterns (reading A1, nonsymmetric case: the strength of
// the pair {i,j} is w_ij = -(a_ij + a_ji)/2; commutative, so S is bitwise symmetric; a missing
// entry counts as 0).  Two sorted lists per row: ascending union.
__global__ void k_sym_rows(int n, const int* __restrict__ rp, const int* __restrict__ col,
                           const double* __restrict__ val, const int* __restrict__ trp,
                           const int* __restrict__ tcol, const double* __restrict__ tval,
                           const int* __restrict__ srp, int* __restrict__ scol, double* __restrict__ sval,
                           int* __restrict__ len) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int ka = rp[i], kt = trp[i], m = 0;
  const int ea = rp[i + 1], et = trp[i + 1];
  const int d = srp ? srp[i] : 0;
  while (ka < ea || kt < et) {
    const int ca = ka < ea ? col[ka] : 0x7fffffff, ct = kt < et ? tcol[kt] : 0x7fffffff;
    const int c = ca < ct ? ca : ct;
    double a = 0.0, t = 0.0;
    if (ca == c) a = val[ka++];
    if (ct == c) t = tval[kt++];
    if (srp) {
      scol[d + m] = c;
      sval[d + m] = (a + t) / 2;
    }
    ++m;
  }
  if (!srp) len[i] = m;
}

// natural-numbering CSR of one level while the hierarchy is being built
struct NatCsr {
  int n = 0, nnz = 0;
  int* rowptr = nullptr;
  int* col = nullptr;
  double* val = nullptr;
  int* agg = nullptr;   // natural aggregates (kept in Level::nat_agg)
  int* mptr = nullptr;  // member lists
  int* mem = nullptr;
  double* dinv = nullptr;
  int nc = 0;
};

__global__ void k_compose_agg(int n, int* __restrict__ agg, const int* __restrict__ agg2) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) agg[i] = agg2[agg[i]];
}

// U1-U3 on one matrix: *agg_out (allocated here), *nc_out.  Nonsymmetric handles match on S = (A + A^T)/2.
amg_status aggregate_csr(amg_handle_s* H, int n, int nnz, const int* rowptr, const int* col, const double* val,
                         uint64_t salt, int** agg_out, int* nc_out, int* rounds_out, cudaStream_t st) {
  const amg_options& o = H->opt;
  int *trp = nullptr, *tcol = nullptr, *tsrc = nullptr, *srp = nullptr, *scol = nullptr, *slen = nullptr;
  double *tval = nullptr, *sval = nullptr;
  if (!H->symmetric) {
    AMG_TRY(transpose_csr(H, n, nnz, nnz, rowptr, col, val, &trp, &tcol, &tval, &tsrc, st));
    AMG_ALLOC(H, slen, int, n, st);
    AMG_ALLOC(H, srp, int, n + 1, st);
    k_sym_rows<<<grid_for(n), TPB, 0, st>>>(n, rowptr, col, val, trp, tcol, tval, nullptr, nullptr, nullptr, slen);
    AMG_CUDA_TRY(H, cudaGetLastError());
    AMG_TRY(amg_exclusive_scan(H, slen, srp, n, st));
    int snnz = 0;
    AMG_TRY(read_int(H, srp + n, &snnz, st));
    AMG_ALLOC(H, scol, int, snnz, st);
    AMG_ALLOC(H, sval, double, snnz, st);
    k_sym_rows<<<grid_for(n), TPB, 0, st>>>(n, rowptr, col, val, trp, tcol, tval, srp, scol, sval, nullptr);
    AMG_CUDA_TRY(H, cudaGetLastError());
    rowptr = srp, col = scol, val = sval;
  }
  double* m;
  int *match, *ptr, *root, *isroot, *id, *added;
  AMG_ALLOC(H, m, double, n, st);
  AMG_ALLOC(H, match, int, n, st);
  AMG_ALLOC(H, ptr, int, n, st);
  AMG_ALLOC(H, root, int, n, st);
  AMG_ALLOC(H, isroot, int, n, st);
  AMG_ALLOC(H, id, int, n + 1, st);
  AMG_ALLOC(H, added, int, 8, st);
  const int g = grid_for(n);
  k_row_max<<<g, TPB, 0, st>>>(n, rowptr, col, val, m);
  k_fill_int<<<g, TPB, 0, st>>>(n, match, -1);
  // U1 rounds until one adds no pair.  MATCH_BATCH rounds are queued before the host looks at the counters (one
  // synchronisation per batch instead of one per round); a round queued behind the one that added nothing returns
  // at once on the device, so the matching and the reported round count are those of the round-by-round loop.
  constexpr int MATCH_BATCH = 6;
  int rounds = 0;
  for (bool done = false; !done;) {
    int nb = MATCH_BATCH;
    if (o.max_match_rounds > 0) nb = std::min(nb, o.max_match_rounds - rounds);
    if (nb <= 0) break;
    AMG_CUDA_TRY(H, cudaMemsetAsync(added + 1, 0, sizeof(int) * MATCH_BATCH, st));
    for (int r = 0; r < nb; ++r) {
      const int* prev = r > 0 ? added + r : nullptr;  // slot r + 1 counts round r of the batch
      k_propose<<<g, TPB, 0, st>>>(n, rowptr, col, val, m, o.strong_beta, salt, match, ptr, prev);
      k_handshake<<<g, TPB, 0, st>>>(n, ptr, match, added + r + 1, prev);
    }
    AMG_CUDA_TRY(H, cudaGetLastError());
    int h_added[MATCH_BATCH];
    AMG_CUDA_TRY(H, cudaMemcpyAsync(h_added, added + 1, sizeof(int) * nb, cudaMemcpyDeviceToHost, st));
    AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
    for (int r = 0; r < nb && !done; ++r) {
      ++rounds;
      done = h_added[r] == 0;
    }
  }
  *rounds_out = rounds;
  k_roots<<<g, TPB, 0, st>>>(n, rowptr, col, val, m, o.strong_beta, salt, match, root, isroot);
  AMG_CUDA_TRY(H, cudaGetLastError());
  AMG_TRY(amg_exclusive_scan(H, isroot, id, n, st));
  AMG_TRY(read_int(H, id + n, nc_out, st));
  AMG_ALLOC(H, *agg_out, int, n, st);
  k_assign_agg<<<g, TPB, 0, st>>>(n, root, id, *agg_out);
  AMG_CUDA_TRY(H, cudaGetLastError());
  for (void* q : {(void*)m, (void*)match, (void*)ptr, (void*)root, (void*)isroot, (void*)id, (void*)added, (void*)trp,
                  (void*)tcol, (void*)tval, (void*)tsrc, (void*)srp, (void*)scol, (void*)sval, (void*)slen})
    amg_dev_free(H, q);
  return AMG_OK;
}

amg_status build_members(amg_handle_s* H, NatCsr& N, cudaStream_t st);
amg_status galerkin_level(amg_handle_s* H, const NatCsr& N, NatCsr& C, cudaStream_t st);

// U1-U3 on one level: fills N.agg / N.nc.  agg_passes = 2: the intermediate Galerkin matrix is aggregated
// again (salt + 1000) and the two maps are composed (size-4 aggregates)
amg_status aggregate_level(amg_handle_s* H, NatCsr& N, uint64_t salt, int* rounds_out, cudaStream_t st) {
  AMG_TRY(aggregate_csr(H, N.n, N.nnz, N.rowptr, N.col, N.val, salt, &N.agg, &N.nc, rounds_out, st));
  for (int p = 1; p < H->opt.agg_passes; ++p) {
    NatCsr mid;
    AMG_TRY(build_members(H, N, st));
    AMG_TRY(galerkin_level(H, N, mid, st));
    int* agg2 = nullptr;
    int nc2 = 0, r2 = 0;
    AMG_TRY(aggregate_csr(H, mid.n, mid.nnz, mid.rowptr, mid.col, mid.val, salt + 1000ull * (uint64_t)p, &agg2, &nc2,
                          &r2, st));
    k_compose_agg<<<grid_for(N.n), TPB, 0, st>>>(N.n, N.agg, agg2);
    AMG_CUDA_TRY(H, cudaGetLastError());
    N.nc = nc2;
    if (r2 > *rounds_out) *rounds_out = r2;
    for (void* q : {(void*)agg2, (void*)mid.rowptr, (void*)mid.col, (void*)mid.val, (void*)N.mptr, (void*)N.mem})
      amg_dev_free(H, q);
    N.mptr = N.mem = nullptr;
  }
  return AMG_OK;
}

amg_status build_members(amg_handle_s* H, NatCsr& N, cudaStream_t st) {
  const int n = N.n, nc = N.nc;
  int *cnt, *slot;
  AMG_ALLOC(H, cnt, int, nc + 1, st);
  AMG_ALLOC(H, slot, int, n, st);
  AMG_ALLOC(H, N.mptr, int, nc + 1, st);
  AMG_ALLOC(H, N.mem, int, n, st);
  AMG_CUDA_TRY(H, cudaMemsetAsync(cnt, 0, sizeof(int) * (nc + 1), st));
  k_count_members<<<grid_for(n), TPB, 0, st>>>(n, N.agg, cnt, slot);
  AMG_CUDA_TRY(H, cudaGetLastError());
  AMG_TRY(amg_exclusive_scan(H, cnt, N.mptr, nc, st));
  k_fill_members<<<grid_for(n), TPB, 0, st>>>(n, N.agg, N.mptr, slot, N.mem);
  k_sort_members<<<grid_for(nc), TPB, 0, st>>>(nc, N.mptr, N.mem);
  AMG_CUDA_TRY(H, cudaGetLastError());
  amg_dev_free(H, cnt);
  amg_dev_free(H, slot);
  return AMG_OK;
}

// U4: C = Galerkin(N)
amg_status galerkin_level(amg_handle_s* H, const NatCsr& N, NatCsr& C, cudaStream_t st) {
  const int nc = N.nc;
  int *len, *segptr, *skey, *cnt;
  double* sval;
  AMG_ALLOC(H, len, int, nc, st);
  AMG_ALLOC(H, segptr, int, nc + 1, st);
  AMG_ALLOC(H, cnt, int, nc, st);
  AMG_ALLOC(H, skey, int, N.nnz, st);
  AMG_ALLOC(H, sval, double, N.nnz, st);
  k_rap_len<<<grid_for(nc), TPB, 0, st>>>(nc, N.mptr, N.mem, N.rowptr, len);
  AMG_CUDA_TRY(H, cudaGetLastError());
  AMG_TRY(amg_exclusive_scan(H, len, segptr, nc, st));
  if ((long long)N.nnz <= 24ll * nc)  // short merged rows (the fine levels): 8 lanes per coarse row
    k_rap_rows<8, 64><<<div_up(nc, RAP_THREADS / 8), RAP_THREADS, 0, st>>>(nc, N.mptr, N.mem, N.rowptr, N.col, N.val,
                                                                         N.agg, segptr, skey, sval, cnt);
  else
    k_rap_rows<32, 320><<<div_up(nc, RAP_THREADS / 32), RAP_THREADS, 0, st>>>(nc, N.mptr, N.mem, N.rowptr, N.col,
                                                                            N.val, N.agg, segptr, skey, sval, cnt);
  AMG_CUDA_TRY(H, cudaGetLastError());
  C.n = nc;
  AMG_ALLOC(H, C.rowptr, int, nc + 1, st);
  AMG_TRY(amg_exclusive_scan(H, cnt, C.rowptr, nc, st));
  AMG_TRY(read_int(H, C.rowptr + nc, &C.nnz, st));
  AMG_ALLOC(H, C.col, int, C.nnz, st);
  AMG_ALLOC(H, C.val, double, C.nnz, st);
  k_rap_compact<<<grid_for(nc), TPB, 0, st>>>(nc, segptr, skey, sval, C.rowptr, C.col, C.val);
  AMG_CUDA_TRY(H, cudaGetLastError());
  amg_dev_free(H, len);
  amg_dev_free(H, segptr);
  amg_dev_free(H, cnt);
  amg_dev_free(H, skey);
  amg_dev_free(H, sval);
  return AMG_OK;
}

// permuted copy of a natural CSR: output row p = input row src_row[p], columns mapped by col_map
amg_status permute_csr(amg_handle_s* H, int n, int nnz, const int* rowptr, const int* col, const double* val,
                       const int* src_row, const int* col_map, int* rowptr_out, int* col_out,
                       double* val_out, cudaStream_t st) {
  int* len;
  AMG_ALLOC(H, len, int, n, st);
  k_perm_rowlen<<<grid_for(n), TPB, 0, st>>>(n, rowptr, src_row, len);
  AMG_CUDA_TRY(H, cudaGetLastError());
  AMG_TRY(amg_exclusive_scan(H, len, rowptr_out, n, st));
  if ((long long)nnz <= 12ll * n)
    k_perm_fill<8, 64><<<div_up(n, 16), 128, 0, st>>>(n, rowptr, col, val, src_row, col_map, rowptr_out, col_out,
                                          val_out);
  else
    k_perm_fill<32, 320><<<div_up(n, 4), 128, 0, st>>>(n, rowptr, col, val, src_row, col_map, rowptr_out, col_out,
                                          val_out);
  AMG_CUDA_TRY(H, cudaGetLastError());
  amg_dev_free(H, len);
  (void)nnz;
  return AMG_OK;
}

// U6: dense LU with partial pivoting of a (coarsest) operator given in CSR; *lu / *piv allocated here if null
amg_status dense_lu_of(amg_handle_s* H, int n, const int* rowptr, const int* col, const double* val, double** lu,
                       int** piv, cudaStream_t st) {
  if (!*lu) AMG_ALLOC(H, *lu, double, (size_t)n * n, st);  // a warm resetup refactors in place
  if (!*piv) AMG_ALLOC(H, *piv, int, n, st);
  AMG_CUDA_TRY(H, cudaMemsetAsync(*lu, 0, sizeof(double) * (size_t)n * n, st));
  k_csr_to_dense<<<grid_for(n), TPB, 0, st>>>(n, rowptr, col, val, *lu);
  int* info;
  AMG_ALLOC(H, info, int, 1, st);
  AMG_CUDA_TRY(H, cudaMemsetAsync(info, 0, sizeof(int), st));
  k_dense_lu<<<1, n <= 64 ? 256 : 1024, 0, st>>>(n, *lu, *piv, info);
  AMG_CUDA_TRY(H, cudaGetLastError());
  int h_info = 0;
  AMG_TRY(read_int(H, info, &h_info, st));
  amg_dev_free(H, info);
  if (h_info) {
    H->err = "coarsest operator is singular";
    return AMG_ERR_COARSE_SINGULAR;
  }
  return AMG_OK;
}

// Value dictionary of a level, in two stream-ordered halves so that a warm resetup can queue all levels and
// synchronise once: vdict_collect (hash-set insertion; table and counters stay on the level) and, once the host has
// read the counters, vdict_finish (sort -> L.vdict[256]).
amg_status vdict_collect(amg_handle_s* H, Level& L, cudaStream_t st) {
  if (!L.vd_table) {
    AMG_ALLOC(H, L.vd_table, unsigned long long, VD_SLOTS, st);
    AMG_ALLOC(H, L.vd_count, int, 2, st);
  }
  AMG_CUDA_TRY(H, cudaMemsetAsync(L.vd_table, 0xFF, sizeof(unsigned long long) * VD_SLOTS, st));
  AMG_CUDA_TRY(H, cudaMemsetAsync(L.vd_count, 0, 2 * sizeof(int), st));
  int g = div_up(L.nnz, TPB * 8);
  if (g > H->sm_count * 8) g = H->sm_count * 8;
  if (g < 1) g = 1;
  k_vdict_insert<<<g, TPB, 0, st>>>(L.nnz, L.val, L.vd_table, L.vd_count);
  AMG_CUDA_TRY(H, cudaGetLastError());
  return AMG_OK;
}
// h_count = the level's two counters as read by the host; returns the number of distinct values, 0 = no dictionary
amg_status vdict_finish(amg_handle_s* H, Level& L, const int* h_count, int* ndict, cudaStream_t st) {
  *ndict = 0;
  if (h_count[1] || h_count[0] < 1 || h_count[0] > VD_MAX) return AMG_OK;
  if (!L.vdict) AMG_ALLOC(H, L.vdict, double, 256, st);
  k_vdict_finalize<<<1, VD_SLOTS, 0, st>>>(L.vd_table, L.vd_count, L.vdict);
  AMG_CUDA_TRY(H, cudaGetLastError());
  *ndict = h_count[0];
  return AMG_OK;
}
amg_status build_vdict(amg_handle_s* H, Level& L, cudaStream_t st) {
  L.ndict = 0;
  if (L.nnz <= 0) return AMG_OK;
  int h_count[2] = {0, 0};
  if (L.nnz > 16384) {
    // a cheap look at the first entries first: a level with all-different values (variable coefficients) is
    // recognised by one CTA instead of a full-grid insertion that floods the table
    if (!L.vd_table) {
      AMG_ALLOC(H, L.vd_table, unsigned long long, VD_SLOTS, st);
      AMG_ALLOC(H, L.vd_count, int, 2, st);
    }
    AMG_CUDA_TRY(H, cudaMemsetAsync(L.vd_table, 0xFF, sizeof(unsigned long long) * VD_SLOTS, st));
    AMG_CUDA_TRY(H, cudaMemsetAsync(L.vd_count, 0, 2 * sizeof(int), st));
    k_vdict_insert<<<1, 1024, 0, st>>>(8192, L.val, L.vd_table, L.vd_count);
    AMG_CUDA_TRY(H, cudaGetLastError());
    AMG_CUDA_TRY(H, cudaMemcpyAsync(h_count, L.vd_count, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
    AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
    if (h_count[1]) return AMG_OK;
  }
  AMG_TRY(vdict_collect(H, L, st));
  AMG_CUDA_TRY(H, cudaMemcpyAsync(h_count, L.vd_count, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
  AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
  return vdict_finish(H, L, h_count, &L.ndict, st);
}

// Row-tile partition by stage bytes, then the tile packer (amg_tilepack.cuh) for one operator of a
// level (A_l or A_l^T) in permuted numbering.  The byte model of the partition is approximate (the
// halo of a tile is only known once it is cut), so the target is rescaled until every tile fits a
// ring stage.  fast = 0: no partition fits (very long rows): the level runs the row-vector kernels.
struct TilePack {
  int* blk_ptr = nullptr;
  TileDesc* tiles = nullptr;
  unsigned char* blob = nullptr;
  int* halo_idx = nullptr;
  int* halo_cagg = nullptr;
  size_t blob_bytes = 0;
  int nblk = 0, fast = 0;
};

// *scale_io: the target scale that fitted the level above (the halo share grows from level to level, so the
// search starts a little above it instead of at 1: one attempt per level instead of two or three)
amg_status pack_tiles(amg_handle_s* H, int n, int nnz, const int* rowptr, const int* col, const double* val,
                      const int* agg, const int* agg_ptr, int nc, TilePack& P, cudaStream_t st,
                      double* scale_io = nullptr, int vb = 8, const double* vdict = nullptr, int ndict = 0) {
  const int nnz_w = vb == 1 ? 4 : 2 + vb;  // bytes a stored entry costs in a ring stage: 16-bit column + value, or column | code
  const int stage_cap = rt_stage_bytes(vb == 1), xslot_cap = rt_xslot_bytes(vb == 1);  // ring geometry of the level kind
  const int64_t total_w = nnz_w * (int64_t)nnz + (int64_t)RT_ROW_WEIGHT * n;
  double scale = scale_io ? (*scale_io * 1.12 < 1.0 ? *scale_io * 1.12 : 1.0) : 1.0;
  for (int attempt = 0; attempt < 6 && !P.fast; ++attempt) {
    const int target = (int)((stage_cap - TP_DESC_BYTES - 256) * scale);
    if (target < 512) break;
    if (P.blk_ptr) amg_dev_free(H, P.blk_ptr);
    if (P.tiles) amg_dev_free(H, P.tiles);
    P.blk_ptr = nullptr, P.tiles = nullptr;
    P.nblk = div_up(total_w, target);
    int *size16, *off16, *nh, *hoff, *info;
    AMG_ALLOC(H, P.blk_ptr, int, P.nblk + 1, st);
    AMG_ALLOC(H, P.tiles, TileDesc, P.nblk, st);
    AMG_ALLOC(H, size16, int, P.nblk + 1, st);
    AMG_ALLOC(H, off16, int, P.nblk + 1, st);
    AMG_ALLOC(H, nh, int, P.nblk + 1, st);
    AMG_ALLOC(H, hoff, int, P.nblk + 1, st);
    AMG_ALLOC(H, info, int, 4, st);
    AMG_CUDA_TRY(H, cudaMemsetAsync(info, 0, 4 * sizeof(int), st));
    k_blk_partition<<<grid_for(P.nblk + 1), TPB, 0, st>>>(P.nblk, target, nnz_w, agg_ptr ? nc : n, agg_ptr, rowptr, n,
                                                         P.blk_ptr);
    k_pack_tiles<<<P.nblk, PK_THREADS, 0, st>>>(P.nblk, P.blk_ptr, rowptr, col, val, agg, vb, 0, nullptr, nullptr, size16, nh,
                                               info, P.tiles, nullptr, nullptr, nullptr, vdict, ndict);
    AMG_CUDA_TRY(H, cudaGetLastError());
    int h_info[4];
    AMG_CUDA_TRY(H, cudaMemcpyAsync(h_info, info, 4 * sizeof(int), cudaMemcpyDeviceToHost, st));
    AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
    if (h_info[1]) {
      scale *= 0.5;
    } else if (h_info[0] > stage_cap || h_info[2] > xslot_cap) {
      const double f1 = (double)stage_cap / (double)h_info[0], f2 = (double)xslot_cap / (double)h_info[2];
      scale *= 0.96 * (f1 < f2 ? f1 : f2);
    } else {
      AMG_TRY(amg_exclusive_scan(H, size16, off16, P.nblk, st));
      AMG_TRY(amg_exclusive_scan(H, nh, hoff, P.nblk, st));
      int total16 = 0, total_h = 0;
      AMG_TRY(read_int(H, off16 + P.nblk, &total16, st));
      AMG_TRY(read_int(H, hoff + P.nblk, &total_h, st));
      P.blob_bytes = (size_t)total16 * 16u;
      P.blob = (unsigned char*)amg_dev_alloc(H, P.blob_bytes + 16, st);
      if (!P.blob) {
        H->err = "device allocation failed: tile blobs";
        return AMG_ERR_OOM;
      }
      AMG_ALLOC(H, P.halo_idx, int, total_h + 4, st);
      AMG_ALLOC(H, P.halo_cagg, int, total_h + 4, st);
      k_pack_tiles<<<P.nblk, PK_THREADS, 0, st>>>(P.nblk, P.blk_ptr, rowptr, col, val, agg, vb, 1, off16, hoff, size16, nh, info,
                                                 P.tiles, P.blob, P.halo_idx, P.halo_cagg, vdict, ndict);
      AMG_CUDA_TRY(H, cudaGetLastError());
      P.fast = 1;
      if (scale_io) *scale_io = scale;
    }
    amg_dev_free(H, size16);
    amg_dev_free(H, off16);
    amg_dev_free(H, nh);
    amg_dev_free(H, hoff);
    amg_dev_free(H, info);
  }
  if (!P.fast) {
    if (P.blk_ptr) amg_dev_free(H, P.blk_ptr);
    if (P.tiles) amg_dev_free(H, P.tiles);
    P.blk_ptr = nullptr, P.tiles = nullptr, P.nblk = 0;
  }
  return AMG_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// U7: the whole setup
// ------------------------------------------------------------------------------------------
amg_status amg_build_hierarchy(amg_handle_s* H, const int32_t* d_rowptr, const int32_t* d_col,
                               const double* d_val, int32_t nagg, const int32_t* const* h_d_aggs,
                               cudaStream_t st) {
  const double t_start = now_ms();
  const amg_options& o = H->opt;
  const int n0 = (int)H->n, nnz0 = (int)H->nnz;
  const bool imported = h_d_aggs != nullptr;

  // ---- validation ----
  {
    int h_ends[2] = {-1, -1};
    AMG_CUDA_TRY(H, cudaMemcpyAsync(&h_ends[0], d_rowptr, sizeof(int), cudaMemcpyDeviceToHost, st));
    AMG_CUDA_TRY(H, cudaMemcpyAsync(&h_ends[1], d_rowptr + n0, sizeof(int), cudaMemcpyDeviceToHost, st));
    AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
    if (h_ends[0] != 0 || h_ends[1] != nnz0) {
      H->err = "bad CSR: rowptr[0] != 0 or rowptr[n] != nnz";
      return AMG_ERR_BAD_CSR;
    }
    int* bad;
    AMG_ALLOC(H, bad, int, 2, st);
    AMG_CUDA_TRY(H, cudaMemsetAsync(bad, 0, 2 * sizeof(int), st));
    k_validate_csr<<<grid_for(n0), TPB, 0, st>>>(n0, nnz0, d_rowptr, d_col, d_val, bad);
    if (o.symmetric < 0) k_check_symmetric<<<grid_for(n0), TPB, 0, st>>>(n0, d_rowptr, d_col, d_val, bad + 1);
    AMG_CUDA_TRY(H, cudaGetLastError());
    int h_bad[2] = {0, 0};
    AMG_CUDA_TRY(H, cudaMemcpyAsync(h_bad, bad, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
    AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
    amg_dev_free(H, bad);
    if (h_bad[0]) {
      H->err = "bad CSR: rows must have ascending unique in-range columns and a positive diagonal";
      return AMG_ERR_BAD_CSR;
    }
    H->symmetric = o.symmetric < 0 ? (h_bad[1] ? 0 : 1) : o.symmetric;
  }

  // ---- natural-numbering hierarchy ----
  std::vector<NatCsr> nat(1);
  nat[0].n = n0;
  nat[0].nnz = nnz0;
  AMG_ALLOC(H, H->nat_rowptr, int, n0 + 1, st);
  AMG_ALLOC(H, H->nat_col, int, nnz0, st);
  AMG_CUDA_TRY(H, cudaMemcpyAsync(H->nat_rowptr, d_rowptr, sizeof(int) * (n0 + 1), cudaMemcpyDeviceToDevice, st));
  AMG_CUDA_TRY(H, cudaMemcpyAsync(H->nat_col, d_col, sizeof(int) * (size_t)nnz0, cudaMemcpyDeviceToDevice, st));
  nat[0].rowptr = H->nat_rowptr;
  nat[0].col = H->nat_col;
  nat[0].val = const_cast<double*>(d_val);  // read only during setup

  double t_agg = 0.0, t_rap = 0.0;
  int rounds_max = 0;
  std::vector<int> rounds_per_level;
  int l = 0;
  for (;;) {
    NatCsr& cur = nat[l];
    if (imported) {
      if (l >= nagg) break;
      // import: copy ids, nc = max + 1
      AMG_ALLOC(H, cur.agg, int, cur.n, st);
      AMG_CUDA_TRY(H, cudaMemcpyAsync(cur.agg, h_d_aggs[l], sizeof(int) * cur.n, cudaMemcpyDeviceToDevice, st));
      int* mx;
      AMG_ALLOC(H, mx, int, 2, st);
      AMG_CUDA_TRY(H, cudaMemsetAsync(mx, 0, 2 * sizeof(int), st));
      k_max_int<<<grid_for(cur.n), TPB, 0, st>>>(cur.n, cur.agg, mx, mx + 1);
      int h_mx[2];
      AMG_CUDA_TRY(H, cudaMemcpyAsync(h_mx, mx, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
      AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
      amg_dev_free(H, mx);
      if (h_mx[1]) {
        H->err = "imported aggregates contain a negative id";
        return AMG_ERR_INVALID_ARG;
      }
      cur.nc = h_mx[0] + 1;
      rounds_per_level.push_back(0);
    } else {
      if (cur.n <= o.coarse_max_rows || l == o.max_levels - 1) break;
      double t0 = now_ms();
      int rounds = 0;
      AMG_TRY(aggregate_level(H, cur, o.hash_seed + (uint64_t)l, &rounds, st));
      t_agg += now_ms() - t0;
      if ((double)cur.nc > 0.8 * (double)cur.n) {  // stall: this level is the coarsest
        amg_dev_free(H, cur.agg);
        cur.agg = nullptr;
        cur.nc = 0;
        break;
      }
      rounds_max = rounds > rounds_max ? rounds : rounds_max;
      rounds_per_level.push_back(rounds);
    }
    double t0 = now_ms();
    AMG_TRY(build_members(H, cur, st));
    {  // every id must be used (imported aggregates): no empty aggregate
      // checked implicitly by the Galerkin product: an empty aggregate gives an empty coarse row,
      // which fails the diagonal check below
    }
    AMG_ALLOC(H, cur.dinv, double, cur.n, st);
    k_dinv<<<grid_for(cur.n), TPB, 0, st>>>(cur.n, cur.rowptr, cur.col, cur.val, o.smoother, o.omega, cur.dinv);
    AMG_CUDA_TRY(H, cudaGetLastError());
    nat.emplace_back();
    AMG_TRY(galerkin_level(H, nat[l], nat[l + 1], st));
    t_rap += now_ms() - t0;
    ++l;
  }
  const int Lc = l;  // index of the coarsest level
  if (nat[Lc].n > MAX_DENSE) {
    H->err = "coarsening stalled above 4096 rows";
    return AMG_ERR_COARSEN_STALL;
  }
  if (imported) {  // imported aggregates with an unused id give a coarse row without diagonal
    int* bad;
    AMG_ALLOC(H, bad, int, 1, st);
    AMG_CUDA_TRY(H, cudaMemsetAsync(bad, 0, sizeof(int), st));
    for (int q = 1; q <= Lc; ++q)
      k_validate_csr<<<grid_for(nat[q].n), TPB, 0, st>>>(nat[q].n, nat[q].nnz, nat[q].rowptr, nat[q].col,
                                                        nat[q].val, bad);
    int h_bad = 0;
    AMG_TRY(read_int(H, bad, &h_bad, st));
    amg_dev_free(H, bad);
    if (h_bad) {
      H->err = "imported aggregates: every id in [0, nc) must be used and coarse diagonals must be positive";
      return AMG_ERR_INVALID_ARG;
    }
  }

  // ---- aggregate-contiguous renumbering, bottom-up ----
  const double t_reorder0 = now_ms();
  H->lv.assign(Lc + 1, Level());
  for (int q = 0; q <= Lc; ++q) {
    Level& L = H->lv[q];
    L.n = nat[q].n;
    L.nnz = nat[q].nnz;
    L.nc = q < Lc ? nat[q].nc : 0;
    L.nat_agg = nat[q].agg;
    L.match_rounds = q < (int)rounds_per_level.size() ? rounds_per_level[q] : 0;
    AMG_ALLOC(H, L.pos, int, L.n, st);
    AMG_ALLOC(H, L.inv, int, L.n, st);
  }
  {
    Level& L = H->lv[Lc];
    k_iota<<<grid_for(L.n), TPB, 0, st>>>(L.n, L.pos);
    k_iota<<<grid_for(L.n), TPB, 0, st>>>(L.n, L.inv);
  }
  for (int q = Lc - 1; q >= 0; --q) {
    Level& L = H->lv[q];
    const NatCsr& N = nat[q];
    int* sizep;
    AMG_ALLOC(H, sizep, int, L.nc, st);
    AMG_ALLOC(H, L.agg_ptr, int, L.nc + 1, st);
    AMG_ALLOC(H, L.agg, int, L.n, st);
    k_perm_sizes<<<grid_for(L.nc), TPB, 0, st>>>(L.nc, N.mptr, H->lv[q + 1].pos, sizep);
    AMG_CUDA_TRY(H, cudaGetLastError());
    AMG_TRY(amg_exclusive_scan(H, sizep, L.agg_ptr, L.nc, st));
    k_perm_pos<<<grid_for(L.nc), TPB, 0, st>>>(L.nc, N.mptr, N.mem, H->lv[q + 1].pos, L.agg_ptr, L.pos, L.inv,
                                              L.agg);
    AMG_CUDA_TRY(H, cudaGetLastError());
    amg_dev_free(H, sizep);
  }
  double pack_scale = 1.0;
  double pack_scale1 = 1.0;   // (levels stored as 8-bit codes have their own ring geometry: their own scale)
  for (int q = 0; q <= Lc; ++q) {
    Level& L = H->lv[q];
    const NatCsr& N = nat[q];
    L.nnz_alloc = ((L.nnz + 3) & ~3) + 4;
    AMG_ALLOC(H, L.rowptr, int, L.n + 1, st);
    AMG_ALLOC(H, L.col, int, L.nnz_alloc, st);
    AMG_ALLOC(H, L.val, double, L.nnz_alloc, st);
    AMG_TRY(permute_csr(H, L.n, L.nnz, N.rowptr, N.col, N.val, L.inv, L.pos, L.rowptr, L.col, L.val, st));
    k_pad_tail<<<1, 32, 0, st>>>(L.nnz, L.nnz_alloc, L.col, L.val);
    if (q < Lc) {
      AMG_ALLOC(H, L.dinv, double, L.n, st);
      k_gather_double<<<grid_for(L.n), TPB, 0, st>>>(L.n, N.dinv, L.inv, L.dinv);
    }
    AMG_CUDA_TRY(H, cudaGetLastError());
    L.fast = 0;
    L.v32 = (o.hierarchy_fp32 && q < Lc) ? 1 : 0;  // mixed-precision hierarchy: the V-cycle's operators in fp32
    if (!o.force_generic && L.n > 0) {
      if (o.value_dict && !o.hierarchy_fp32 && q < 64) AMG_TRY(build_vdict(H, L, st));  // (64: the warm path's counter array)
      TilePack P;
      AMG_TRY(pack_tiles(H, L.n, L.nnz, L.rowptr, L.col, L.val, q < Lc ? L.agg : nullptr, q < Lc ? L.agg_ptr : nullptr,
                         q < Lc ? L.nc : 0, P, st, L.ndict > 0 ? &pack_scale1 : &pack_scale, L.ndict > 0 ? 1 : (L.v32 ? 4 : 8),
                         L.vdict, L.ndict));
      L.blk_ptr = P.blk_ptr, L.tiles = P.tiles, L.blob = P.blob, L.halo_idx = P.halo_idx, L.halo_cagg = P.halo_cagg;
      L.blob_bytes = P.blob_bytes, L.nblk = P.nblk, L.fast = P.fast;
      if (L.v32 && q == 0) {  // the Krylov method's own SpMV keeps the fp64 operator
        TilePack PK;
        AMG_TRY(pack_tiles(H, L.n, L.nnz, L.rowptr, L.col, L.val, L.agg, L.agg_ptr, L.nc, PK, st, nullptr, 8));
        L.K.blk_ptr = PK.blk_ptr, L.K.tiles = PK.tiles, L.K.blob = PK.blob, L.K.halo_idx = PK.halo_idx;
        L.K.halo_cagg = PK.halo_cagg, L.K.blob_bytes = PK.blob_bytes, L.K.nblk = PK.nblk, L.K.fast = PK.fast;
      }
    }
    const double mean_len = L.n > 0 ? (double)L.nnz / L.n : 1.0;
    L.lpr = mean_len <= 6.0 ? 4 : (mean_len <= 12.0 ? 8 : (mean_len <= 24.0 ? 16 : 32));
    size_t mat_bytes = (size_t)L.nnz * 12 + (size_t)L.n * 4;
    L.stream_hint = (H->l2_bytes > 0 && mat_bytes > H->l2_bytes / 2) ? 1 : 0;
    // work vectors
    AMG_ALLOC(H, L.x, double, L.n, st);
    AMG_ALLOC(H, L.x2, double, L.n, st);
    if (q > 0) AMG_ALLOC(H, L.b, double, L.n, st);
    if (!L.fast && q < Lc) AMG_ALLOC(H, L.rtmp, double, L.n, st);
  }
  AMG_TRY(amg_build_sweep_diagonals(H, st));
  H->stats.reorder_ms = now_ms() - t_reorder0;

  // ---- coarsest dense LU ----
  const double t_lu0 = now_ms();
  {
    Level& L = H->lv[Lc];
    H->nL = L.n;
    AMG_TRY(dense_lu_of(H, L.n, L.rowptr, L.col, L.val, &H->lu, &H->piv, st));
  }
  H->stats.lu_ms = now_ms() - t_lu0;

  // ---- release the natural-numbering scratch ----
  AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
  for (int q = 0; q <= Lc; ++q) {
    NatCsr& N = nat[q];
    if (q > 0) {
      amg_dev_free(H, N.rowptr);
      amg_dev_free(H, N.col);
      amg_dev_free(H, N.val);
    }
    amg_dev_free(H, N.mptr);
    amg_dev_free(H, N.mem);
    amg_dev_free(H, N.dinv);
  }

  H->stats.aggregate_ms = t_agg;
  H->stats.galerkin_ms = t_rap;
  H->stats.match_rounds_max = rounds_max;
  H->stats.total_ms = now_ms() - t_start;
  return AMG_OK;
}

// NEXT-2 ("forms A^T ... then solves the adjoint system"): the
// transposed hierarchy IS the Galerkin hierarchy of A^T on the same aggregates ((P^T A P)^T =
// P^T A^T P), so every level operator is transposed in place (permuted numbering), tile-packed like
// the forward one, the coarsest A_L^T factored, and the dense tail of B^T assembled.
amg_status amg_ensure_transposed(amg_handle_s* H, cudaStream_t st) {
  if (H->have_T) return AMG_OK;
  const int Lc = (int)H->lv.size() - 1;
  for (int q = 0; q <= Lc; ++q) {
    Level& L = H->lv[q];
    LevelOpT& T = L.T;
    AMG_TRY(transpose_csr(H, L.n, L.nnz, L.nnz_alloc, L.rowptr, L.col, L.val, &T.rowptr, &T.col, &T.val, &T.src, st));
    if (!H->opt.force_generic && L.n > 0) {
      TilePack P;
      AMG_TRY(pack_tiles(H, L.n, L.nnz, T.rowptr, T.col, T.val, q < Lc ? L.agg : nullptr, q < Lc ? L.agg_ptr : nullptr,
                         q < Lc ? L.nc : 0, P, st, nullptr, L.ndict > 0 ? 1 : (L.v32 ? 4 : 8), L.vdict, L.ndict));
      T.blk_ptr = P.blk_ptr, T.tiles = P.tiles, T.blob = P.blob, T.halo_idx = P.halo_idx, T.halo_cagg = P.halo_cagg;
      T.blob_bytes = P.blob_bytes, T.nblk = P.nblk, T.fast = P.fast;
      if (L.v32 && q == 0) {  // fp64 blobs of A_0^T for the Krylov method's SpMV
        TilePack PK;
        AMG_TRY(pack_tiles(H, L.n, L.nnz, T.rowptr, T.col, T.val, L.agg, L.agg_ptr, L.nc, PK, st, nullptr, 8));
        L.KT.blk_ptr = PK.blk_ptr, L.KT.tiles = PK.tiles, L.KT.blob = PK.blob, L.KT.halo_idx = PK.halo_idx;
        L.KT.halo_cagg = PK.halo_cagg, L.KT.blob_bytes = PK.blob_bytes, L.KT.nblk = PK.nblk, L.KT.fast = PK.fast;
      }
    }
    if (!T.fast && !L.rtmp && q < Lc) AMG_ALLOC(H, L.rtmp, double, L.n, st);
  }
  {
    Level& L = H->lv[Lc];
    AMG_TRY(dense_lu_of(H, L.n, L.T.rowptr, L.T.col, L.T.val, &H->luT, &H->pivT, st));
  }
  H->have_T = true;
  AMG_TRY(amg_setup_tail(H, 1, st));
  return AMG_OK;
}

// natural-numbering CSR of a level, rebuilt from the permuted storage (parity hook)
amg_status amg_natural_level_csr(amg_handle_s* H, int level, int32_t* d_rowptr, int32_t* d_col,
                                 double* d_val, cudaStream_t st) {
  Level& L = H->lv[level];
  // natural row i = permuted row pos[i]; permuted column c -> natural inv[c]
  return permute_csr(H, L.n, L.nnz, L.rowptr, L.col, L.val, L.pos, L.inv, d_rowptr, d_col, d_val, st);
}

// ------------------------------------------------------------------------------------------
// NEXT-1, warm: amg_resetup_values(keep_aggregates = 1) on the KEPT hierarchy ("matrix
// coefficients are updated in place"; :285 "warm resetup-and-solve ... dominates").  Nothing
// structural is redone: aggregates, numbering, level patterns, tile partitions, halo lists, the
// slice / perm / column sections of the blobs, work vectors, CUDA graphs all stay.  Recomputed,
// each as one bandwidth-trivial pass: level-0 values (gather through src0), coarse values (numeric
// Galerkin: every coarse entry sums its fine contributions in ascending position, a fixed order),
// smoother diagonals, the value sections of the tile blobs, the coarsest LU, the dense tail, and
// the same for the transposed hierarchy.  The maps are built on the first warm resetup.
// ------------------------------------------------------------------------------------------
namespace {

// src0[k] for the permuted level-0 entry k = (row p, column c): position of (inv[p], inv[c]) in the caller's CSR
__global__ void k_build_src0(int n, const int* __restrict__ rowptr, const int* __restrict__ col,
                             const int* __restrict__ inv, const int* __restrict__ nat_rowptr,
                             const int* __restrict__ nat_col, int* __restrict__ src0) {
  int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const int i = inv[p];
  const int s = nat_rowptr[i], e = nat_rowptr[i + 1];
  for (int k = rowptr[p]; k < rowptr[p + 1]; ++k) {
    const int j = inv[col[k]];
    int lo = s, hi = e - 1, pos = s;
    while (lo <= hi) {
      const int mid = (lo + hi) >> 1;
      const int c = nat_col[mid];
      if (c == j) {
        pos = mid;
        break;
      }
      if (c < j) lo = mid + 1;
      else hi = mid - 1;
    }
    src0[k] = pos;
  }
}

// coarse entry of every fine entry: tgt[k] = position of (agg[i], agg[col[k]]) in the coarse CSR; cnt[tgt]++
__global__ void k_rap_target(int n, const int* __restrict__ rowptr, const int* __restrict__ col,
                             const int* __restrict__ agg, const int* __restrict__ crowptr,
                             const int* __restrict__ ccol, int* __restrict__ tgt, int* __restrict__ cnt) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int I = agg[i];
  const int s = crowptr[I], e = crowptr[I + 1];
  for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) {
    const int J = agg[col[k]];
    int lo = s, hi = e - 1, pos = s;
    while (lo <= hi) {
      const int mid = (lo + hi) >> 1;
      const int c = ccol[mid];
      if (c == J) {
        pos = mid;
        break;
      }
      if (c < J) lo = mid + 1;
      else hi = mid - 1;
    }
    tgt[k] = pos;
    atomicAdd(&cnt[pos], 1);
  }
}
__global__ void k_contrib_fill(int nnz, const int* __restrict__ tgt, const int* __restrict__ cptr,
                               int* __restrict__ cursor, int* __restrict__ cidx) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= nnz) return;
  const int t = tgt[k];
  cidx[cptr[t] + atomicAdd(&cursor[t], 1)] = k;
}
__global__ void k_contrib_sort(int m, const int* __restrict__ cptr, int* __restrict__ cidx) {
  int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= m) return;
  const int s = cptr[e], t = cptr[e + 1];
  for (int a = s + 1; a < t; ++a) {
    const int v = cidx[a];
    int b = a - 1;
    while (b >= s && cidx[b] > v) {
      cidx[b + 1] = cidx[b];
      --b;
    }
    cidx[b + 1] = v;
  }
}
// numeric Galerkin: cval[e] = sum of val[] over the contributions of e, ascending position
__global__ void k_rap_numeric(int m, const int* __restrict__ cptr, const int* __restrict__ cidx,
                              const double* __restrict__ val, double* __restrict__ cval) {
  int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= m) return;
  double s = 0.0;
  for (int t = cptr[e]; t < cptr[e + 1]; ++t) s += val[cidx[t]];
  cval[e] = s;
}

// value section of every tile blob from the level's CSR values (the slices / perm sections say where)
__global__ void __launch_bounds__(256) k_blob_refill(int ntiles, const TileDesc* __restrict__ tiles,
                                                     const int* __restrict__ rowptr, const int* __restrict__ col,
                                                     const double* __restrict__ val, const int* __restrict__ halo_idx,
                                                     unsigned char* __restrict__ blob, const double* __restrict__ vdict,
                                                     int ndict) {
  // the column section of the blob says which entry every slot holds (whatever order the packer chose): slot ->
  // tile-local column -> level column -> position in the CSR row (ascending unique columns: binary search)
  const int t = blockIdx.x;
  if (t >= ntiles) return;
  const TileDesc d = tiles[t];
  if (d.nr <= 0) return;
  unsigned char* base = blob + (size_t)d.blob16 * 16u;
  const BlobLayout p = tp_blob(d.nsl, d.nslots, d.vb);
  const int2* slices = reinterpret_cast<const int2*>(base);
  const unsigned short* perm = reinterpret_cast<const unsigned short*>(base + p.o_perm);
  const unsigned short* o_col = reinterpret_cast<const unsigned short*>(base + p.o_col);
  uint32_t* o_cw = reinterpret_cast<uint32_t*>(base + p.o_col);  // vb == 1: column | dictionary code << 16
  double* o_val = reinterpret_cast<double*>(base + p.o_val);
  float* o_val32 = reinterpret_cast<float*>(base + p.o_val);
  for (int j = 0; j < d.nsl; ++j) {
    const int2 sl = slices[j];
    for (int q = threadIdx.x; q < 32 * sl.y; q += blockDim.x) {
      const int k = q >> 5, lane = q & 31;
      const int lr = perm[j * 32 + lane];
      double v = 0.0;
      bool in_row = false;
      if (lr != 0xFFFF) {
        const int r = d.r0 + lr;
        const int s = rowptr[r], e = rowptr[r + 1];
        if (k < e - s) {
          in_row = true;
          const int c16 = d.vb == 1 ? (int)(o_cw[sl.x + q] & 0xFFFFu) : (int)o_col[sl.x + q];
          const int c = c16 < d.nr ? d.r0 + c16 : halo_idx[d.halo_off + c16 - d.nr];
          int lo = s, hi = e;  // first entry >= c
          while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (col[mid] < c) lo = mid + 1;
            else hi = mid;
          }
          v = val[lo];
        }
      }
      if (d.vb == 1)
        o_cw[sl.x + q] = (o_cw[sl.x + q] & 0xFFFFu) | ((uint32_t)(in_row ? vdict_code(vdict, ndict, v) : (unsigned char)255) << 16);
      else if (d.vb == 4)
        o_val32[sl.x + q] = (float)v;
      else
        o_val[sl.x + q] = v;
    }
  }
}

amg_status build_resetup_maps(amg_handle_s* H, cudaStream_t st) {
  const int Lc = (int)H->lv.size() - 1;
  AMG_TRY(amg_ensure_src0(H, st));
  for (int l = 0; l < Lc; ++l) {
    Level& L = H->lv[l];
    Level& C = H->lv[l + 1];
    int *tgt, *cnt;
    AMG_ALLOC(H, tgt, int, L.nnz, st);
    AMG_ALLOC(H, cnt, int, C.nnz + 1, st);
    AMG_ALLOC(H, L.contrib_ptr, int, C.nnz + 1, st);
    AMG_ALLOC(H, L.contrib_idx, int, L.nnz, st);
    AMG_CUDA_TRY(H, cudaMemsetAsync(cnt, 0, sizeof(int) * (C.nnz + 1), st));
    k_rap_target<<<grid_for(L.n), TPB, 0, st>>>(L.n, L.rowptr, L.col, L.agg, C.rowptr, C.col, tgt, cnt);
    AMG_CUDA_TRY(H, cudaGetLastError());
    AMG_TRY(amg_exclusive_scan(H, cnt, L.contrib_ptr, C.nnz, st));
    AMG_CUDA_TRY(H, cudaMemsetAsync(cnt, 0, sizeof(int) * (C.nnz + 1), st));
    k_contrib_fill<<<grid_for(L.nnz), TPB, 0, st>>>(L.nnz, tgt, L.contrib_ptr, cnt, L.contrib_idx);
    k_contrib_sort<<<grid_for(C.nnz), TPB, 0, st>>>(C.nnz, L.contrib_ptr, L.contrib_idx);
    AMG_CUDA_TRY(H, cudaGetLastError());
    amg_dev_free(H, tgt);
    amg_dev_free(H, cnt);
  }
  H->have_maps = true;
  return AMG_OK;
}

}  // namespace

namespace {
__global__ void k_scale_vec(int n, double w, const double* __restrict__ in, double* __restrict__ out) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = w * in[i];
}
}  // namespace

// Diagonals of the sweeps of a cycle.  Chebyshev-accelerated L1-Jacobi (smoother = 2, NEXT-4): spec(D_l1^-1 A) lies
// in (0, 1] (Gershgorin), so the nu sweeps of a smoothing step are Richardson steps x += tau_j D_l1^-1 (b - A x) with
// tau_j the reciprocal roots of the degree-nu Chebyshev polynomial of [1/ratio, 1] (ascending; post-sweeps reversed,
// so that B stays symmetric for nu1 = nu2).  tau_j * dinv is stored once per sweep: the kernels do not change.
amg_status amg_build_sweep_diagonals(amg_handle_s* H, cudaStream_t st) {
  const amg_options& o = H->opt;
  const int nu1 = o.pre_sweeps, nu2 = o.post_sweeps;
  const int Lc = (int)H->lv.size() - 1;
  auto weights = [&](int k) {
    std::vector<double> w(k > 0 ? k : 0);
    const double a = 1.0 / o.cheby_ratio, pi = 3.14159265358979323846;
    for (int j = 0; j < k; ++j) w[j] = 1.0 / ((1.0 + a) / 2 + (1.0 - a) / 2 * cos(pi * (2 * j + 1) / (2.0 * k)));
    return w;
  };
  const std::vector<double> wpre = weights(nu1), wpost = weights(nu2);
  for (int l = 0; l < Lc; ++l) {
    Level& L = H->lv[l];
    for (int s = 0; s < nu1 + nu2; ++s) {
      if (o.smoother != 2) {
        L.dsw[s] = L.dinv;
        continue;
      }
      const double w = s < nu1 ? wpre[s] : wpost[nu2 - 1 - (s - nu1)];
      if (!L.dsw[s] || L.dsw[s] == L.dinv) AMG_ALLOC(H, L.dsw[s], double, L.n, st);
      k_scale_vec<<<grid_for(L.n), TPB, 0, st>>>(L.n, w, L.dinv, L.dsw[s]);
    }
  }
  AMG_CUDA_TRY(H, cudaGetLastError());
  return AMG_OK;
}

// level 0: position in the caller's CSR of every entry of the permuted CSR (warm resetup, tile gradient)
amg_status amg_ensure_src0(amg_handle_s* H, cudaStream_t st) {
  Level& L0 = H->lv[0];
  if (L0.src0) return AMG_OK;
  AMG_ALLOC(H, L0.src0, int, L0.nnz, st);
  k_build_src0<<<grid_for(L0.n), TPB, 0, st>>>(L0.n, L0.rowptr, L0.col, L0.inv, H->nat_rowptr, H->nat_col, L0.src0);
  AMG_CUDA_TRY(H, cudaGetLastError());
  return AMG_OK;
}

amg_status amg_resetup_values_warm(amg_handle_s* H, const double* d_val, int* fallback, cudaStream_t st) {
  *fallback = 0;
  const amg_options& o = H->opt;
  const int n0 = (int)H->n, nnz0 = (int)H->nnz;
  const int Lc = (int)H->lv.size() - 1;
  // ---- the new values must keep the CSR valid; symmetric = -1 repeats the device check ----
  {
    int* bad;
    AMG_ALLOC(H, bad, int, 2, st);
    AMG_CUDA_TRY(H, cudaMemsetAsync(bad, 0, 2 * sizeof(int), st));
    k_validate_csr<<<grid_for(n0), TPB, 0, st>>>(n0, nnz0, H->nat_rowptr, H->nat_col, d_val, bad);
    if (o.symmetric < 0) k_check_symmetric<<<grid_for(n0), TPB, 0, st>>>(n0, H->nat_rowptr, H->nat_col, d_val, bad + 1);
    AMG_CUDA_TRY(H, cudaGetLastError());
    int h_bad[2] = {0, 0};
    AMG_CUDA_TRY(H, cudaMemcpyAsync(h_bad, bad, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
    AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
    amg_dev_free(H, bad);
    if (h_bad[0]) {
      H->err = "bad CSR: the new values must keep a positive diagonal in every row";
      return AMG_ERR_BAD_CSR;
    }
    const int sym = o.symmetric < 0 ? (h_bad[1] ? 0 : 1) : o.symmetric;
    if (sym != H->symmetric) {  // symmetric <-> nonsymmetric: the matching and the transposed hierarchy change
      *fallback = 1;
      return AMG_OK;
    }
  }
  const double t0 = now_ms();
  if (!H->have_maps) AMG_TRY(build_resetup_maps(H, st));
  // ---- values of every level: gather on level 0, numeric Galerkin below ----
  Level& L0 = H->lv[0];
  k_gather_vals<<<grid_for(L0.nnz), TPB, 0, st>>>(L0.nnz, d_val, L0.src0, L0.val);
  for (int l = 0; l < Lc; ++l) {
    Level& L = H->lv[l];
    Level& C = H->lv[l + 1];
    k_rap_numeric<<<grid_for(C.nnz), TPB, 0, st>>>(C.nnz, L.contrib_ptr, L.contrib_idx, L.val, C.val);
  }
  AMG_CUDA_TRY(H, cudaGetLastError());
  // ---- value dictionaries of the levels stored as 8-bit codes: the new values must fit one again (all levels
  // queued, one synchronisation) ----
  {
    int h_counts[64][2];
    int nd_levels = 0;
    for (int l = 0; l <= Lc && l < 64; ++l) {
      Level& L = H->lv[l];
      if (L.ndict <= 0) continue;
      AMG_TRY(vdict_collect(H, L, st));
      AMG_CUDA_TRY(H, cudaMemcpyAsync(h_counts[l], L.vd_count, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
      ++nd_levels;
    }
    if (nd_levels) AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
    for (int l = 0; l <= Lc && l < 64; ++l) {
      Level& L = H->lv[l];
      if (L.ndict <= 0) continue;
      int nd = 0;
      AMG_TRY(vdict_finish(H, L, h_counts[l], &nd, st));
      if (nd <= 0) {  // more than 255 distinct values now: the blobs need the fp64 layout
        *fallback = 1;
        return AMG_OK;
      }
      L.ndict = nd;
    }
  }
  // ---- smoother diagonals, blob value sections, transposed values ----
  for (int l = 0; l <= Lc; ++l) {
    Level& L = H->lv[l];
    if (l < Lc) k_dinv<<<grid_for(L.n), TPB, 0, st>>>(L.n, L.rowptr, L.col, L.val, o.smoother, o.omega, L.dinv);
    if (L.fast) k_blob_refill<<<L.nblk, 256, 0, st>>>(L.nblk, L.tiles, L.rowptr, L.col, L.val, L.halo_idx, L.blob, L.vdict, L.ndict);
    if (L.K.fast) k_blob_refill<<<L.K.nblk, 256, 0, st>>>(L.K.nblk, L.K.tiles, L.rowptr, L.col, L.val, L.K.halo_idx, L.K.blob, nullptr, 0);
    if (H->have_T) {
      k_gather_vals<<<grid_for(L.nnz), TPB, 0, st>>>(L.nnz, L.val, L.T.src, L.T.val);
      if (L.T.fast) k_blob_refill<<<L.T.nblk, 256, 0, st>>>(L.T.nblk, L.T.tiles, L.T.rowptr, L.T.col, L.T.val, L.T.halo_idx, L.T.blob, L.vdict, L.ndict);
      if (L.KT.fast) k_blob_refill<<<L.KT.nblk, 256, 0, st>>>(L.KT.nblk, L.KT.tiles, L.T.rowptr, L.T.col, L.T.val, L.KT.halo_idx, L.KT.blob, nullptr, 0);
    }
  }
  AMG_CUDA_TRY(H, cudaGetLastError());
  AMG_TRY(amg_build_sweep_diagonals(H, st));
  // ---- coarsest LU (factors rebuilt in place), dense tail ----
  {
    Level& L = H->lv[Lc];
    AMG_TRY(dense_lu_of(H, L.n, L.rowptr, L.col, L.val, &H->lu, &H->piv, st));
    if (H->have_T) AMG_TRY(dense_lu_of(H, L.n, L.T.rowptr, L.T.col, L.T.val, &H->luT, &H->pivT, st));
  }
  if (H->tail_dense_level >= 0) {
    AMG_TRY(amg_setup_tail(H, 0, st));
    if (H->have_T) AMG_TRY(amg_setup_tail(H, 1, st));
  }
  AMG_CUDA_TRY(H, cudaStreamSynchronize(st));
  H->stats.total_ms = now_ms() - t0;
  H->stats.aggregate_ms = H->stats.galerkin_ms = H->stats.reorder_ms = 0.0;
  return AMG_OK;
}
