// CPU ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.  See amg_oracle.h for scope, citations,
// pins and the "parity unpinned" list.  Plain C++17, fp64, std::vector CSR, no numerical
// library, no code shared with the CUDA path.  Every function below names the passage
// (PAPER.md line / SURVEY.md §8(c) step) it follows, in that passage's notation.
#include "amg_oracle.h"

#include <algorithm>
#include <cmath>
#include <climits>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

int g_threads = 1;

struct Csr {
  int n = 0;
  std::vector<int> rowptr, col;
  std::vector<double> val;
  int nnz() const { return rowptr.empty() ? 0 : rowptr[n]; }
};

struct Level {
  Csr A;                     // A_l
  Csr At;                    // A_l^T, built lazily for the nonsymmetric adjoint (O-7)
  Csr A32, At32;             // hierarchy_fp32: the same operators with every value rounded to fp32 (V-cycle only)
  std::vector<double> dinv;  // smoother diagonal (A7)
  std::vector<int> agg;      // agg_l[i] in [0, n_{l+1})
  std::vector<int> agg_ptr, agg_mem;  // members of every aggregate, ascending fine index
  int nc = 0;
  int rounds = 0;
};

}  // namespace

struct oracle_handle_s {
  oracle_options opt;
  std::vector<Level> lv;   // lv[0 … L]; lv[L] is the coarsest (only A used)
  std::vector<double> lu;  // dense LU of A_L (row-major, in place), unit lower
  std::vector<int> piv;
  std::vector<double> lut;  // dense LU of A_L^T
  std::vector<int> pivt;
  bool have_t = false;
  bool have_32 = false, have_t32 = false;
  bool have_lu = false;  // with imported aggregates the coarsest LU is factored at first use
  std::vector<double> hist;  // ||r_k|| / ||b|| of the last solve, k = 1 … iterations (PAPER.md:125 diagnostics)
};

namespace {

// ------------------------------------------------------------------------------------------
// basic kernels
// ------------------------------------------------------------------------------------------
void spmv(const Csr& A, const double* x, double* y) {
#pragma omp parallel for num_threads(g_threads) schedule(static) if (A.n > 20000)
  for (int i = 0; i < A.n; ++i) {
    double s = 0.0;
    for (int k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) s += A.val[k] * x[A.col[k]];
    y[i] = s;
  }
}

double dot(int n, const double* a, const double* b) {  // sequential: fixed summation order
  double s = 0.0;
  for (int i = 0; i < n; ++i) s += a[i] * b[i];
  return s;
}

Csr transpose(const Csr& A) {
  Csr T;
  T.n = A.n;
  T.rowptr.assign(A.n + 1, 0);
  T.col.resize(A.nnz());
  T.val.resize(A.nnz());
  for (int k = 0; k < A.nnz(); ++k) T.rowptr[A.col[k] + 1]++;
  for (int i = 0; i < A.n; ++i) T.rowptr[i + 1] += T.rowptr[i];
  std::vector<int> fill(T.rowptr.begin(), T.rowptr.end() - 1);
  for (int i = 0; i < A.n; ++i)
    for (int k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
      int p = fill[A.col[k]]++;
      T.col[p] = i;  // ascending i => ascending columns in every row of T
      T.val[p] = A.val[k];
    }
  return T;
}

// S = (A + A^T) / 2 on the union of the two patterns (A1, nonsymmetric case: the strength of the
// pair {i,j} is w_ij = -(a_ij + a_ji)/2; the sum is commutative, so S is bitwise symmetric and
// S(A) == S(A^T); a missing entry counts as 0).  For a bitwise symmetric A, S == A bitwise.
Csr symmetrise(const Csr& A) {
  Csr T = transpose(A);
  Csr S;
  S.n = A.n;
  S.rowptr.assign(A.n + 1, 0);
  for (int i = 0; i < A.n; ++i) {
    int ka = A.rowptr[i], ea = A.rowptr[i + 1], kt = T.rowptr[i], et = T.rowptr[i + 1];
    while (ka < ea || kt < et) {  // two sorted lists: ascending union
      int ca = ka < ea ? A.col[ka] : INT32_MAX, ct = kt < et ? T.col[kt] : INT32_MAX;
      int c = std::min(ca, ct);
      double a = 0.0, t = 0.0;
      if (ca == c) a = A.val[ka++];
      if (ct == c) t = T.val[kt++];
      S.col.push_back(c);
      S.val.push_back((a + t) / 2);
    }
    S.rowptr[i + 1] = (int)S.col.size();
  }
  return S;
}

// ------------------------------------------------------------------------------------------
// O-2  Aggregate(A, salt): deterministic pairwise matching (SURVEY.md §8(c) O-2, A1 … A5)
// ------------------------------------------------------------------------------------------
inline uint64_t mix64(uint64_t z) {  // A4
  z ^= z >> 30;
  z *= 0xBF58476D1CE4E5B9ULL;
  z ^= z >> 27;
  z *= 0x94D049BB133111EBULL;
  z ^= z >> 31;
  return z;
}
inline uint64_t edge_hash(int i, int j, uint64_t salt) {  // symmetric in (i, j)
  uint64_t lo = (uint64_t)std::min(i, j), hi = (uint64_t)std::max(i, j);
  return mix64(lo * 0x9E3779B97F4A7C15ULL + hi * 0xBF58476D1CE4E5B9ULL + salt);
}

struct Key {  // key(i,j) = (-q, h, -lo, -hi), larger is better
  int q;
  uint64_t h;
  int lo, hi;
};
inline bool better(const Key& a, const Key& b) {  // a > b in the lexicographic order
  if (a.q != b.q) return a.q < b.q;
  if (a.h != b.h) return a.h > b.h;
  if (a.lo != b.lo) return a.lo < b.lo;
  return a.hi < b.hi;
}

// m_i = max_{j != i} max(w_ij, 0),  w_ij = -a_ij  (A1)
std::vector<double> row_maxima(const Csr& A) {
  std::vector<double> m(A.n, 0.0);
  for (int i = 0; i < A.n; ++i) {
    double mi = 0.0;
    for (int k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k)
      if (A.col[k] != i) mi = std::max(mi, std::max(-A.val[k], 0.0));
    m[i] = mi;
  }
  return m;
}

// candidate edge test (A2) and bucket (A3) for the entry k of row i
inline bool candidate(const Csr& A, const std::vector<double>& m, double beta, int i, int k,
                      Key* key, uint64_t salt) {
  int j = A.col[k];
  if (j == i) return false;
  double w = -A.val[k];
  if (!(w > 0.0)) return false;
  if (!(w >= beta * std::min(m[i], m[j]))) return false;
  double M = std::max(m[i], m[j]);
  key->q = (2.0 * w > M) ? 0 : ((4.0 * w > M) ? 1 : 2);
  key->h = edge_hash(i, j, salt);
  key->lo = std::min(i, j);
  key->hi = std::max(i, j);
  return true;
}

// handshake rounds to the fix-point (the definition)
int match_handshake(const Csr& A, const std::vector<double>& m, double beta, uint64_t salt,
                    int max_rounds, std::vector<int>& match) {
  int n = A.n;
  match.assign(n, -1);
  std::vector<int> ptr(n);
  int rounds = 0;
  for (;;) {
    if (max_rounds > 0 && rounds >= max_rounds) break;
    // every unmatched i points to its best unmatched candidate neighbour (state at round start)
    for (int i = 0; i < n; ++i) {
      ptr[i] = -1;
      if (match[i] >= 0) continue;
      Key best{};
      for (int k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
        Key key;
        if (!candidate(A, m, beta, i, k, &key, salt)) continue;
        if (match[A.col[k]] >= 0) continue;
        if (ptr[i] < 0 || better(key, best)) {
          best = key;
          ptr[i] = A.col[k];
        }
      }
    }
    int added = 0;
    for (int i = 0; i < n; ++i) {
      int j = ptr[i];
      if (j >= 0 && ptr[j] == i) {
        match[i] = j;
        ++added;
      }
    }
    ++rounds;
    if (added == 0) break;
  }
  return rounds;
}

// greedy matching over candidate edges by descending key (independent second code, pin P8)
int match_greedy(const Csr& A, const std::vector<double>& m, double beta, uint64_t salt,
                 std::vector<int>& match) {
  struct E {
    Key key;
    int i, j;
  };
  std::vector<E> edges;
  for (int i = 0; i < A.n; ++i)
    for (int k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
      Key key;
      if (A.col[k] > i && candidate(A, m, beta, i, k, &key, salt)) edges.push_back({key, i, A.col[k]});
    }
  std::sort(edges.begin(), edges.end(), [](const E& a, const E& b) { return better(a.key, b.key); });
  match.assign(A.n, -1);
  for (const E& e : edges)
    if (match[e.i] < 0 && match[e.j] < 0) {
      match[e.i] = e.j;
      match[e.j] = e.i;
    }
  return 0;
}

// roots, singleton merge (A5), numbering by ascending root
int number_aggregates(const Csr& A, const std::vector<double>& m, double beta, uint64_t salt,
                      const std::vector<int>& match, std::vector<int>& agg) {
  int n = A.n;
  std::vector<int> root(n);
  for (int i = 0; i < n; ++i) root[i] = match[i] >= 0 ? std::min(i, match[i]) : i;
  std::vector<int> root2(root);
  for (int i = 0; i < n; ++i) {  // one simultaneous step: reads only `match` / `root`
    if (match[i] >= 0) continue;
    int jbest = -1;
    Key best{};
    for (int k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
      Key key;
      if (!candidate(A, m, beta, i, k, &key, salt)) continue;
      if (match[A.col[k]] < 0) continue;  // only matched neighbours
      if (jbest < 0 || better(key, best)) {
        best = key;
        jbest = A.col[k];
      }
    }
    if (jbest >= 0) root2[i] = root[jbest];
  }
  std::vector<int> id(n, -1);
  int nc = 0;
  for (int i = 0; i < n; ++i)
    if (root2[i] == i) id[i] = nc++;
  agg.resize(n);
  for (int i = 0; i < n; ++i) agg[i] = id[root2[i]];
  return nc;
}

// symmetric != 0: w_ij = -a_ij read from row i (A1; the generators make a_ij == a_ji bitwise);
// symmetric == 0: the matching runs on S = (A + A^T)/2 (A1, nonsymmetric case)
int aggregate(const Csr& A0, double beta, uint64_t salt, int max_rounds, int mode, int symmetric,
              std::vector<int>& match, std::vector<int>& agg, int* rounds) {
  Csr S;
  if (!symmetric) S = symmetrise(A0);
  const Csr& A = symmetric ? A0 : S;
  std::vector<double> m = row_maxima(A);
  *rounds = mode == 0 ? match_handshake(A, m, beta, salt, max_rounds, match)
                      : match_greedy(A, m, beta, salt, match);
  return number_aggregates(A, m, beta, salt, match, agg);
}

void member_lists(const std::vector<int>& agg, int nc, std::vector<int>& ptr, std::vector<int>& mem) {
  int n = (int)agg.size();
  ptr.assign(nc + 1, 0);
  for (int i = 0; i < n; ++i) ptr[agg[i] + 1]++;
  for (int I = 0; I < nc; ++I) ptr[I + 1] += ptr[I];
  mem.resize(n);
  std::vector<int> fill(ptr.begin(), ptr.end() - 1);
  for (int i = 0; i < n; ++i) mem[fill[agg[i]]++] = i;  // ascending fine index inside each aggregate
}

// ------------------------------------------------------------------------------------------
// O-3  Galerkin(A, agg): A_c[I,J] = sum_{agg(i)=I} sum_{agg(j)=J} a_ij  (piecewise-constant P)
// columns ascending, explicit zeros kept, summation in ascending fine row then position (A8)
// ------------------------------------------------------------------------------------------
Csr galerkin(const Csr& A, const std::vector<int>& agg, int nc) {
  std::vector<int> ptr, mem;
  member_lists(agg, nc, ptr, mem);
  Csr C;
  C.n = nc;
  C.rowptr.assign(nc + 1, 0);
  std::vector<int> where(nc, -1);  // position of coarse column J in the current row's list
  std::vector<int> cols;
  std::vector<double> vals;
  std::vector<std::pair<int, double>> row;
  for (int I = 0; I < nc; ++I) {
    cols.clear();
    vals.clear();
    for (int t = ptr[I]; t < ptr[I + 1]; ++t) {
      int i = mem[t];
      for (int k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
        int J = agg[A.col[k]];
        if (where[J] < 0) {
          where[J] = (int)cols.size();
          cols.push_back(J);
          vals.push_back(A.val[k]);
        } else {
          vals[where[J]] += A.val[k];
        }
      }
    }
    row.clear();
    for (size_t t = 0; t < cols.size(); ++t) {
      row.emplace_back(cols[t], vals[t]);
      where[cols[t]] = -1;
    }
    std::sort(row.begin(), row.end(), [](auto& a, auto& b) { return a.first < b.first; });
    for (auto& e : row) {
      C.col.push_back(e.first);
      C.val.push_back(e.second);
    }
    C.rowptr[I + 1] = (int)C.col.size();
  }
  return C;
}

// smoother diagonal (A7): L1: 1 / sum_j |a_ij| ; damped Jacobi: omega / a_ii
std::vector<double> smoother_diag(const Csr& A, int smoother, double omega) {
  std::vector<double> d(A.n);
  for (int i = 0; i < A.n; ++i) {
    double l1 = 0.0, aii = 0.0;
    for (int k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
      l1 += std::fabs(A.val[k]);
      if (A.col[k] == i) aii = A.val[k];
    }
    d[i] = smoother == 1 ? omega / aii : 1.0 / l1;  // 0 and 2 (Chebyshev-accelerated L1-Jacobi): the l1 diagonal
  }
  return d;
}

// Chebyshev-accelerated L1-Jacobi (smoother = 2, NEXT-4).  spec(D_l1^-1 A) lies in (0, 1] for the M-matrix-like
// operators of the method (Gershgorin), so no eigenvalue estimate is needed: the k sweeps of one smoothing step are
// Richardson steps x += tau_j D_l1^-1 (b - A x) whose weights are the reciprocals of the roots of the degree-k
// Chebyshev polynomial of the interval [1/ratio, 1]:  r_j = (1+a)/2 + (1-a)/2 cos(pi (2j+1) / (2k)), a = 1/ratio.
// The product of the k error factors (1 - tau_j mu) is the polynomial of degree k with p(0) = 1 of least maximum
// on [a, 1]:  max |p| = 1 / T_k((1+a)/(1-a)).  j ascending: weights ascending (the mildest step first).
std::vector<double> cheby_weights(int k, double ratio) {
  std::vector<double> w(k > 0 ? k : 0);
  const double a = 1.0 / ratio, pi = 3.14159265358979323846;
  for (int j = 0; j < k; ++j) w[j] = 1.0 / ((1.0 + a) / 2 + (1.0 - a) / 2 * std::cos(pi * (2 * j + 1) / (2.0 * k)));
  return w;
}

// dense LU with partial pivoting, in place, row-major; returns false if singular (O-1)
bool dense_lu(int n, std::vector<double>& a, std::vector<int>& piv) {
  piv.resize(n);
  double amax = 0.0;
  for (double v : a) amax = std::max(amax, std::fabs(v));
  for (int k = 0; k < n; ++k) {
    int p = k;
    double best = std::fabs(a[(size_t)k * n + k]);
    for (int i = k + 1; i < n; ++i) {
      double v = std::fabs(a[(size_t)i * n + k]);
      if (v > best) {
        best = v;
        p = i;
      }
    }
    if (!(best > 1e-300 * amax) || !(amax > 0.0)) return false;
    piv[k] = p;
    if (p != k)
      for (int j = 0; j < n; ++j) std::swap(a[(size_t)k * n + j], a[(size_t)p * n + j]);
    double akk = a[(size_t)k * n + k];
    for (int i = k + 1; i < n; ++i) {
      double l = a[(size_t)i * n + k] / akk;
      a[(size_t)i * n + k] = l;
      for (int j = k + 1; j < n; ++j) a[(size_t)i * n + j] -= l * a[(size_t)k * n + j];
    }
  }
  return true;
}

void dense_lu_solve(int n, const std::vector<double>& a, const std::vector<int>& piv,
                    const double* b, double* x) {
  // dense_lu exchanges WHOLE rows (the multipliers of the earlier columns move with them), so the
  // factors are those of P A with P = the product of all exchanges: P is applied to b first, then
  // L y = P b and U x = y  (O-1: "factor A_L = P L U"; pinned by test_dense_lu_row_swaps)
  for (int i = 0; i < n; ++i) x[i] = b[i];
  for (int k = 0; k < n; ++k)
    if (piv[k] != k) std::swap(x[k], x[piv[k]]);
  for (int k = 0; k < n; ++k)
    for (int i = k + 1; i < n; ++i) x[i] -= a[(size_t)i * n + k] * x[k];
  for (int i = n - 1; i >= 0; --i) {
    double s = x[i];
    for (int j = i + 1; j < n; ++j) s -= a[(size_t)i * n + j] * x[j];
    x[i] = s / a[(size_t)i * n + i];
  }
}

std::vector<double> to_dense(const Csr& A) {
  std::vector<double> d((size_t)A.n * A.n, 0.0);
  for (int i = 0; i < A.n; ++i)
    for (int k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) d[(size_t)i * A.n + A.col[k]] = A.val[k];
  return d;
}

int check_csr(int n, const int* rowptr, const int* col, const double* val) {
  if (n <= 0 || rowptr[0] != 0) return ORACLE_ERR_BAD_CSR;
  for (int i = 0; i < n; ++i) {
    if (rowptr[i + 1] < rowptr[i]) return ORACLE_ERR_BAD_CSR;
    bool diag = false;
    for (int k = rowptr[i]; k < rowptr[i + 1]; ++k) {
      if (col[k] < 0 || col[k] >= n) return ORACLE_ERR_BAD_CSR;
      if (k > rowptr[i] && col[k] <= col[k - 1]) return ORACLE_ERR_BAD_CSR;
      if (col[k] == i) diag = val[k] > 0.0;
    }
    if (!diag) return ORACLE_ERR_BAD_CSR;
  }
  return ORACLE_OK;
}

// ------------------------------------------------------------------------------------------
// O-1  Setup
// ------------------------------------------------------------------------------------------
int ensure_lu(oracle_handle_s* H) {  // factor A_L = P L U densely with partial pivoting
  if (H->have_lu) return ORACLE_OK;
  const Csr& AL = H->lv.back().A;
  if (AL.n > 4096) return ORACLE_ERR_COARSEN_STALL;
  H->lu = to_dense(AL);
  if (!dense_lu(AL.n, H->lu, H->piv)) return ORACLE_ERR_COARSE_SINGULAR;
  H->have_lu = true;
  return ORACLE_OK;
}

int setup(oracle_handle_s* H, Csr A0, int nagg, const int32_t* const* aggs) {
  const oracle_options& o = H->opt;
  H->lv.clear();
  H->lv.emplace_back();
  H->lv[0].A = std::move(A0);
  int l = 0;
  for (;;) {
    Level& cur = H->lv[l];
    int nl = cur.A.n;
    std::vector<int> agg;
    int nc;
    if (aggs) {
      if (l >= nagg) break;
      agg.assign(aggs[l], aggs[l] + nl);
      nc = 0;
      for (int v : agg) {
        if (v < 0) return ORACLE_ERR_INVALID_ARG;
        nc = std::max(nc, v + 1);
      }
    } else {
      if (nl <= o.coarse_max_rows || l == o.max_levels - 1) break;
      std::vector<int> match;
      nc = aggregate(cur.A, o.strong_beta, o.hash_seed + (uint64_t)l, o.max_match_rounds, 0,
                     o.symmetric, match, agg, &cur.rounds);
      // agg_passes > 1 (O-1): aggregate the intermediate Galerkin matrix again and compose
      // (pass p uses the salt hash_seed + l + 1000 p; size-4 aggregates for agg_passes = 2)
      for (int p = 1; p < o.agg_passes; ++p) {
        Csr mid = galerkin(cur.A, agg, nc);
        std::vector<int> match2, agg2;
        int r2 = 0;
        int nc2 = aggregate(mid, o.strong_beta, o.hash_seed + (uint64_t)l + 1000ull * (uint64_t)p,
                            o.max_match_rounds, 0, o.symmetric, match2, agg2, &r2);
        for (int i = 0; i < nl; ++i) agg[i] = agg2[agg[i]];
        nc = nc2;
        cur.rounds = std::max(cur.rounds, r2);
      }
      if ((double)nc > 0.8 * (double)nl) break;  // stall => this level is the coarsest (A6)
    }
    cur.agg = agg;
    cur.nc = nc;
    member_lists(cur.agg, nc, cur.agg_ptr, cur.agg_mem);
    cur.dinv = smoother_diag(cur.A, o.smoother, o.omega);
    Csr C = galerkin(cur.A, cur.agg, nc);
    H->lv.emplace_back();
    H->lv[l + 1].A = std::move(C);
    ++l;
  }
  if (aggs) return ORACLE_OK;  // imported hierarchy: LU deferred to ensure_lu()
  return ensure_lu(H);
}

// ------------------------------------------------------------------------------------------
// O-4  z = B r = Vcycle(0, r); zero guess on every level, V(nu1, nu2), gamma  (A9)
// `T` selects the transposed hierarchy (B^T) for the nonsymmetric adjoint (O-7)
// ------------------------------------------------------------------------------------------
void jacobi_sweep(const Csr& A, const std::vector<double>& dinv, const double* b, const double* x,
                  double* xout, double w = 1.0) {  // all rows from the old x; w: Chebyshev weight of the sweep
#pragma omp parallel for num_threads(g_threads) schedule(static) if (A.n > 20000)
  for (int i = 0; i < A.n; ++i) {
    double s = 0.0;
    for (int k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) s += A.val[k] * x[A.col[k]];
    xout[i] = x[i] + (w * dinv[i]) * (b[i] - s);
  }
}

void residual_restrict(const Csr& A, const Level& L, const double* b, const double* x, double* rc) {
#pragma omp parallel for num_threads(g_threads) schedule(static) if (A.n > 20000)
  for (int I = 0; I < L.nc; ++I) {
    double acc = 0.0;
    for (int t = L.agg_ptr[I]; t < L.agg_ptr[I + 1]; ++t) {
      int i = L.agg_mem[t];
      double s = 0.0;
      for (int k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) s += A.val[k] * x[A.col[k]];
      acc += b[i] - s;
    }
    rc[I] = acc;
  }
}

void vcycle(const oracle_handle_s* H, int l, bool T, const double* b, double* x) {
  int Lc = (int)H->lv.size() - 1;
  const Level& lev = H->lv[l];
  // hierarchy_fp32 (NEXT-4): inside the V-cycle the sparse level operators are the fp64 ones
  // rounded to fp32, used in fp64 arithmetic; dinv, the coarsest LU and every vector stay fp64
  const bool f32 = H->opt.hierarchy_fp32 != 0 && l < Lc;
  const Csr& A = T ? (f32 ? lev.At32 : lev.At) : (f32 ? lev.A32 : lev.A);
  int n = A.n;
  if (l == Lc) {
    dense_lu_solve(n, T ? H->lut : H->lu, T ? H->pivt : H->piv, b, x);
    return;
  }
  const oracle_options& o = H->opt;
  std::vector<double> tmp(n);
  const std::vector<double> wpre = o.smoother == 2 ? cheby_weights(o.pre_sweeps, o.cheby_ratio)
                                                   : std::vector<double>(o.pre_sweeps > 0 ? o.pre_sweeps : 0, 1.0);
  const std::vector<double> wpost = o.smoother == 2 ? cheby_weights(o.post_sweeps, o.cheby_ratio)
                                                    : std::vector<double>(o.post_sweeps > 0 ? o.post_sweeps : 0, 1.0);
  if (o.pre_sweeps > 0) {
    for (int i = 0; i < n; ++i) x[i] = (wpre[0] * lev.dinv[i]) * b[i];  // sweep 1 of nu1 from a zero guess
    for (int s = 1; s < o.pre_sweeps; ++s) {
      jacobi_sweep(A, lev.dinv, b, x, tmp.data(), wpre[s]);
      std::memcpy(x, tmp.data(), sizeof(double) * n);
    }
  } else {
    for (int i = 0; i < n; ++i) x[i] = 0.0;
  }
  std::vector<double> rc(lev.nc), ec(lev.nc);
  residual_restrict(A, lev, b, x, rc.data());
  vcycle(H, l + 1, T, rc.data(), ec.data());
  for (int i = 0; i < n; ++i) x[i] = x[i] + o.coarse_scale * ec[lev.agg[i]];
  for (int s = 0; s < o.post_sweeps; ++s) {  // Chebyshev: the weights in reverse order (B stays symmetric for nu1 = nu2)
    jacobi_sweep(A, lev.dinv, b, x, tmp.data(), wpost[o.post_sweeps - 1 - s]);
    std::memcpy(x, tmp.data(), sizeof(double) * n);
  }
}

void apply_precond(const oracle_handle_s* H, int precond, bool T, const double* r, double* z) {
  if (precond)
    vcycle(H, 0, T, r, z);
  else
    std::memcpy(z, r, sizeof(double) * H->lv[0].A.n);
}

// ------------------------------------------------------------------------------------------
// O-5  PCG (textbook, x0 = 0, recurrence residual, Euclidean norm; A10)
// ------------------------------------------------------------------------------------------
void pcg(oracle_handle_s* H, const Csr& A, bool T, const double* b, double* x, double rtol,
         int maxit, int precond, oracle_info* info) {
  int n = A.n;
  H->hist.clear();
  std::vector<double> r(b, b + n), z(n), p(n), q(n);
  for (int i = 0; i < n; ++i) x[i] = 0.0;
  double nb = std::sqrt(dot(n, b, b));
  info->b_norm = nb;
  info->iterations = 0;
  info->rel_residual = 0.0;
  info->status = ORACLE_CONVERGED;
  if (nb == 0.0) return;
  apply_precond(H, precond, T, r.data(), z.data());
  p = z;
  double rho = dot(n, r.data(), z.data());
  info->status = ORACLE_MAXIT;
  info->rel_residual = 1.0;
  for (int k = 1; k <= maxit; ++k) {
    spmv(A, p.data(), q.data());
    double sigma = dot(n, p.data(), q.data());
    if (!(sigma > 0.0)) {
      info->status = std::isfinite(sigma) ? ORACLE_BREAKDOWN : ORACLE_NONFINITE;
      break;
    }
    double alpha = rho / sigma;
    for (int i = 0; i < n; ++i) x[i] += alpha * p[i];
    for (int i = 0; i < n; ++i) r[i] -= alpha * q[i];
    double nr = std::sqrt(dot(n, r.data(), r.data()));
    info->iterations = k;
    info->rel_residual = nr / nb;
    H->hist.push_back(nr / nb);
    if (!std::isfinite(nr)) {
      info->status = ORACLE_NONFINITE;
      break;
    }
    if (nr <= rtol * nb) {
      info->status = ORACLE_CONVERGED;
      break;
    }
    apply_precond(H, precond, T, r.data(), z.data());
    double rho1 = dot(n, r.data(), z.data());
    double beta = rho1 / rho;
    for (int i = 0; i < n; ++i) p[i] = z[i] + beta * p[i];
    rho = rho1;
  }
}

// ------------------------------------------------------------------------------------------
// O-6  right-preconditioned BiCGSTAB (x0 = 0, rhat = r0 = b; A11)
// ------------------------------------------------------------------------------------------
void bicgstab(oracle_handle_s* H, const Csr& A, bool T, const double* b, double* x,
              double rtol, int maxit, int precond, oracle_info* info) {
  int n = A.n;
  H->hist.clear();
  std::vector<double> r(b, b + n), rhat(b, b + n), p(n, 0.0), v(n, 0.0), s(n), t(n), ph(n), sh(n);
  for (int i = 0; i < n; ++i) x[i] = 0.0;
  double nb = std::sqrt(dot(n, b, b));
  info->b_norm = nb;
  info->iterations = 0;
  info->rel_residual = 0.0;
  info->status = ORACLE_CONVERGED;
  if (nb == 0.0) return;
  double rho = 1.0, alpha = 1.0, omega = 1.0;
  info->status = ORACLE_MAXIT;
  info->rel_residual = 1.0;
  for (int k = 1; k <= maxit; ++k) {
    double rho1 = dot(n, rhat.data(), r.data());
    if (rho1 == 0.0 || !std::isfinite(rho1)) {
      info->status = std::isfinite(rho1) ? ORACLE_BREAKDOWN : ORACLE_NONFINITE;
      break;
    }
    double beta = (rho1 / rho) * (alpha / omega);
    rho = rho1;
    for (int i = 0; i < n; ++i) p[i] = r[i] + beta * (p[i] - omega * v[i]);
    apply_precond(H, precond, T, p.data(), ph.data());
    spmv(A, ph.data(), v.data());
    double rv = dot(n, rhat.data(), v.data());
    if (rv == 0.0 || !std::isfinite(rv)) {
      info->status = std::isfinite(rv) ? ORACLE_BREAKDOWN : ORACLE_NONFINITE;
      break;
    }
    alpha = rho / rv;
    for (int i = 0; i < n; ++i) s[i] = r[i] - alpha * v[i];
    double ns = std::sqrt(dot(n, s.data(), s.data()));
    info->iterations = k;
    if (ns <= rtol * nb) {  // half-step exit reports the current k (A11)
      for (int i = 0; i < n; ++i) x[i] += alpha * ph[i];
      info->rel_residual = ns / nb;
      info->status = ORACLE_CONVERGED;
      H->hist.push_back(ns / nb);
      break;
    }
    apply_precond(H, precond, T, s.data(), sh.data());
    spmv(A, sh.data(), t.data());
    double ts = dot(n, t.data(), s.data());
    double tt = dot(n, t.data(), t.data());
    omega = ts / tt;
    for (int i = 0; i < n; ++i) x[i] += alpha * ph[i] + omega * sh[i];
    for (int i = 0; i < n; ++i) r[i] = s[i] - omega * t[i];
    double nr = std::sqrt(dot(n, r.data(), r.data()));
    info->rel_residual = nr / nb;
    H->hist.push_back(nr / nb);
    if (!std::isfinite(nr)) {
      info->status = ORACLE_NONFINITE;
      break;
    }
    if (nr <= rtol * nb) {
      info->status = ORACLE_CONVERGED;
      break;
    }
    if (omega == 0.0) {
      info->status = ORACLE_BREAKDOWN;
      break;
    }
  }
}

Csr rounded_to_fp32(const Csr& A) {
  Csr R = A;
  for (double& v : R.val) v = (double)(float)v;
  return R;
}

void ensure_fp32(oracle_handle_s* H) {
  if (!H->opt.hierarchy_fp32) return;
  if (!H->have_32) {
    for (Level& L : H->lv) L.A32 = rounded_to_fp32(L.A);
    H->have_32 = true;
  }
  if (H->have_t && !H->have_t32) {
    for (Level& L : H->lv) L.At32 = rounded_to_fp32(L.At);
    H->have_t32 = true;
  }
}

void ensure_transposed(oracle_handle_s* H) {
  if (H->have_t) return;
  for (Level& L : H->lv) L.At = transpose(L.A);  // (P^T A P)^T = P^T A^T P on the same aggregates
  int Lc = (int)H->lv.size() - 1;
  H->lut = to_dense(H->lv[Lc].At);
  dense_lu(H->lv[Lc].At.n, H->lut, H->pivt);
  H->have_t = true;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------
extern "C" {

void oracle_options_default(oracle_options* o) {
  o->pre_sweeps = 2;
  o->post_sweeps = 2;
  o->smoother = 0;
  o->coarse_max_rows = 64;
  o->max_levels = 32;
  o->max_match_rounds = 0;
  o->omega = 2.0 / 3.0;
  o->strong_beta = 0.25;
  o->coarse_scale = 1.0;
  o->hash_seed = 0;
  o->agg_passes = 1;
  o->symmetric = 1;
  o->hierarchy_fp32 = 0;
  o->cheby_ratio = 6.0;
}

void oracle_set_threads(int nthreads) { g_threads = nthreads > 0 ? nthreads : 1; }
int oracle_get_threads(void) { return g_threads; }

static int setup_common(oracle_handle* out, int32_t n, const int32_t* rowptr, const int32_t* col,
                        const double* val, const oracle_options* opt, int32_t nagg,
                        const int32_t* const* aggs) {
  if (!out) return ORACLE_ERR_INVALID_ARG;
  *out = nullptr;
  if (!rowptr || !col || !val || n <= 0) return ORACLE_ERR_INVALID_ARG;
  int rc = check_csr(n, rowptr, col, val);
  if (rc) return rc;
  oracle_handle_s* H = new oracle_handle_s;
  if (opt)
    H->opt = *opt;
  else
    oracle_options_default(&H->opt);
  Csr A;
  A.n = n;
  A.rowptr.assign(rowptr, rowptr + n + 1);
  A.col.assign(col, col + rowptr[n]);
  A.val.assign(val, val + rowptr[n]);
  rc = setup(H, std::move(A), nagg, aggs);
  if (rc) {
    delete H;
    return rc;
  }
  *out = H;
  return ORACLE_OK;
}

int oracle_setup(oracle_handle* out, int32_t n, const int32_t* rowptr, const int32_t* col,
                 const double* val, const oracle_options* opt) {
  return setup_common(out, n, rowptr, col, val, opt, 0, nullptr);
}

int oracle_setup_with_aggregates(oracle_handle* out, int32_t n, const int32_t* rowptr,
                                 const int32_t* col, const double* val, const oracle_options* opt,
                                 int32_t nagg, const int32_t* const* aggs) {
  if (nagg < 0 || (nagg > 0 && !aggs)) return ORACLE_ERR_INVALID_ARG;
  static const int32_t* const none[1] = {nullptr};
  return setup_common(out, n, rowptr, col, val, opt, nagg, nagg > 0 ? aggs : none);
}

void oracle_destroy(oracle_handle h) { delete h; }

int oracle_num_levels(oracle_handle h) { return h ? (int)h->lv.size() : ORACLE_ERR_INVALID_ARG; }

int oracle_level_info(oracle_handle h, int32_t level, int32_t* rows, int32_t* nnz) {
  if (!h || level < 0 || level >= (int)h->lv.size()) return ORACLE_ERR_INVALID_ARG;
  if (rows) *rows = h->lv[level].A.n;
  if (nnz) *nnz = h->lv[level].A.nnz();
  return ORACLE_OK;
}

int oracle_get_aggregates(oracle_handle h, int32_t level, int32_t* agg) {
  if (!h || level < 0 || level >= (int)h->lv.size() - 1 || !agg) return ORACLE_ERR_INVALID_ARG;
  std::copy(h->lv[level].agg.begin(), h->lv[level].agg.end(), agg);
  return ORACLE_OK;
}

int oracle_get_level_csr(oracle_handle h, int32_t level, int32_t* rowptr, int32_t* col, double* val) {
  if (!h || level < 0 || level >= (int)h->lv.size()) return ORACLE_ERR_INVALID_ARG;
  const Csr& A = h->lv[level].A;
  if (rowptr) std::copy(A.rowptr.begin(), A.rowptr.end(), rowptr);
  if (col) std::copy(A.col.begin(), A.col.end(), col);
  if (val) std::copy(A.val.begin(), A.val.end(), val);
  return ORACLE_OK;
}

int oracle_get_dinv(oracle_handle h, int32_t level, double* dinv) {
  if (!h || level < 0 || level >= (int)h->lv.size() - 1 || !dinv) return ORACLE_ERR_INVALID_ARG;
  std::copy(h->lv[level].dinv.begin(), h->lv[level].dinv.end(), dinv);
  return ORACLE_OK;
}

int oracle_match_rounds(oracle_handle h, int32_t level) {
  if (!h || level < 0 || level >= (int)h->lv.size() - 1) return ORACLE_ERR_INVALID_ARG;
  return h->lv[level].rounds;
}

int oracle_aggregate(int32_t n, const int32_t* rowptr, const int32_t* col, const double* val,
                     double beta, uint64_t salt, int32_t max_rounds, int32_t mode, int32_t symmetric,
                     int32_t* match, int32_t* agg, int32_t* nc, int32_t* rounds) {
  if (n <= 0 || !rowptr || !col || !val || !nc) return ORACLE_ERR_INVALID_ARG;
  Csr A;
  A.n = n;
  A.rowptr.assign(rowptr, rowptr + n + 1);
  A.col.assign(col, col + rowptr[n]);
  A.val.assign(val, val + rowptr[n]);
  std::vector<int> m, a;
  int r = 0;
  *nc = aggregate(A, beta, salt, max_rounds, mode, symmetric, m, a, &r);
  if (match) std::copy(m.begin(), m.end(), match);
  if (agg) std::copy(a.begin(), a.end(), agg);
  if (rounds) *rounds = r;
  return ORACLE_OK;
}

int oracle_galerkin(int32_t n, const int32_t* rowptr, const int32_t* col, const double* val,
                    const int32_t* agg, int32_t nc, int32_t* crowptr, int32_t* ccol, double* cval,
                    int32_t* cnnz) {
  if (n <= 0 || !rowptr || !col || !val || !agg || nc <= 0) return ORACLE_ERR_INVALID_ARG;
  Csr A;
  A.n = n;
  A.rowptr.assign(rowptr, rowptr + n + 1);
  A.col.assign(col, col + rowptr[n]);
  A.val.assign(val, val + rowptr[n]);
  std::vector<int> a(agg, agg + n);
  Csr C = galerkin(A, a, nc);
  if (cnnz) *cnnz = C.nnz();
  if (crowptr) {
    std::copy(C.rowptr.begin(), C.rowptr.end(), crowptr);
    std::copy(C.col.begin(), C.col.end(), ccol);
    std::copy(C.val.begin(), C.val.end(), cval);
  }
  return ORACLE_OK;
}

int oracle_spmv(oracle_handle h, int32_t level, const double* x, double* y) {
  if (!h || level < 0 || level >= (int)h->lv.size()) return ORACLE_ERR_INVALID_ARG;
  spmv(h->lv[level].A, x, y);
  return ORACLE_OK;
}

int oracle_smooth(oracle_handle h, int32_t level, const double* b, const double* x, double* xout) {
  if (!h || level < 0 || level >= (int)h->lv.size() - 1) return ORACLE_ERR_INVALID_ARG;
  jacobi_sweep(h->lv[level].A, h->lv[level].dinv, b, x, xout);
  return ORACLE_OK;
}

int oracle_residual_restrict(oracle_handle h, int32_t level, const double* b, const double* x,
                             double* rc) {
  if (!h || level < 0 || level >= (int)h->lv.size() - 1) return ORACLE_ERR_INVALID_ARG;
  residual_restrict(h->lv[level].A, h->lv[level], b, x, rc);
  return ORACLE_OK;
}

int oracle_vcycle(oracle_handle h, int32_t level, const double* r, double* z) {
  if (!h || level < 0 || level >= (int)h->lv.size()) return ORACLE_ERR_INVALID_ARG;
  if (int rc = ensure_lu(h)) return rc;
  ensure_fp32(h);
  vcycle(h, level, false, r, z);
  return ORACLE_OK;
}

int oracle_vcycle_transpose(oracle_handle h, int32_t level, const double* r, double* z) {
  if (!h || level < 0 || level >= (int)h->lv.size()) return ORACLE_ERR_INVALID_ARG;
  if (int rc = ensure_lu(h)) return rc;
  ensure_transposed(h);
  ensure_fp32(h);
  vcycle(h, level, true, r, z);
  return ORACLE_OK;
}

int oracle_solve(oracle_handle h, const double* b, double* x, double rtol, int32_t maxit,
                 int32_t krylov, int32_t precond, oracle_info* info) {
  if (!h || !b || !x || !info || maxit < 0) return ORACLE_ERR_INVALID_ARG;
  if (precond)
    if (int rc = ensure_lu(h)) return rc;
  ensure_fp32(h);
  if (krylov == 0)
    pcg(h, h->lv[0].A, false, b, x, rtol, maxit, precond, info);
  else
    bicgstab(h, h->lv[0].A, false, b, x, rtol, maxit, precond, info);
  return ORACLE_OK;
}

int oracle_solve_transpose(oracle_handle h, const double* g, double* lambda, double rtol,
                           int32_t maxit, int32_t krylov, int32_t precond, int32_t symmetric,
                           oracle_info* info) {
  if (!h || !g || !lambda || !info || maxit < 0) return ORACLE_ERR_INVALID_ARG;
  if (symmetric) return oracle_solve(h, g, lambda, rtol, maxit, krylov, precond, info);
  if (precond)
    if (int rc = ensure_lu(h)) return rc;
  ensure_transposed(h);
  ensure_fp32(h);
  if (krylov == 0)
    pcg(h, h->lv[0].At, true, g, lambda, rtol, maxit, precond, info);
  else
    bicgstab(h, h->lv[0].At, true, g, lambda, rtol, maxit, precond, info);
  return ORACLE_OK;
}

int oracle_cheby_weights(int32_t k, double ratio, double* w) {
  if (k < 0 || !(ratio > 1.0) || (k > 0 && !w)) return ORACLE_ERR_INVALID_ARG;
  const std::vector<double> v = cheby_weights(k, ratio);
  std::copy(v.begin(), v.end(), w);
  return ORACLE_OK;
}

int oracle_get_residual_history(oracle_handle h, double* out, int32_t cap) {
  if (!h) return ORACLE_ERR_INVALID_ARG;
  int m = (int)h->hist.size();
  if (out)
    for (int k = 0; k < m && k < cap; ++k) out[k] = h->hist[k];
  return m;
}

int oracle_grad_values(oracle_handle h, const double* lambda, const double* x, int32_t nrhs,
                       int64_t ld, double* gA, int32_t accumulate) {
  if (!h || !lambda || !x || !gA || nrhs < 0) return ORACLE_ERR_INVALID_ARG;
  const Csr& A = h->lv[0].A;
  for (int i = 0; i < A.n; ++i)
    for (int k = A.rowptr[i]; k < A.rowptr[i + 1]; ++k) {
      double s = 0.0;
      for (int b = 0; b < nrhs; ++b) s += lambda[(size_t)b * ld + i] * x[(size_t)b * ld + A.col[k]];
      gA[k] = accumulate ? gA[k] - s : -s;
    }
  return ORACLE_OK;
}

}  // extern "C"
