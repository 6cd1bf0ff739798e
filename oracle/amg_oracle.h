/* CPU ORACLE — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 implementation of the hot path of arxiv/paper_2606_09001 ("JAX-AMG"):
 * the aggregation-AMG-preconditioned CG / BiCGSTAB solve of A x = b (§2.1), the
 * adjoint solve A^T lambda = dL/dx (Eq. 1) and the gradients dL/dA = -lambda x^T
 * on the sparsity pattern, dL/db = lambda (Eq. 2).  The paper delegates every
 * numerical kernel to NVIDIA AmgX and states none of the algorithm; the
 * algorithm followed here step by step is the reading fixed in SURVEY.md §8(c) (O-1 … O-8,
 * readings A1 … A22, restated in DESIGN.md).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this library.  It shares no code, header, table or constant generator with the CUDA
 * library in paper_2606_09001_b200/csrc (which never includes this file).
 *
 * All pointers are HOST pointers.  Indices int32, values fp64.  Every function returns 0 on
 * success, a negative code otherwise (see ORACLE_ERR_*).
 *
 * Pins (tests/test_oracle_pins.py; SURVEY.md §8(c) P1 … P12): closed-form Laplacian eigenpairs,
 * CG finite termination and the Chebyshev bound, dense LU (numpy) on tiny systems, exact
 * Galerkin stencils, V-cycle symmetry/definiteness, smoother error factors, structural
 * aggregation invariants + handshake == greedy, manufactured solutions, central finite
 * differences for the adjoint gradient, the paper's §3.1 and §3.2 worked examples.
 * Parity unpinned: the absolute iteration counts on the five BASELINE.json configurations
 * (they depend on the readings A1 … A9; only oracle-vs-GPU parity is defined for them).
 */
#ifndef AMG_ORACLE_H
#define AMG_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORACLE_OK 0
#define ORACLE_ERR_INVALID_ARG (-1)
#define ORACLE_ERR_BAD_CSR (-2)
#define ORACLE_ERR_COARSE_SINGULAR (-3)
#define ORACLE_ERR_COARSEN_STALL (-4)

/* status of a solve ("convergence status") */
#define ORACLE_CONVERGED 0
#define ORACLE_MAXIT 1
#define ORACLE_BREAKDOWN 2
#define ORACLE_NONFINITE 3

typedef struct {
  int32_t pre_sweeps;       /* nu1, default 2 (BASELINE.json cfg 1)                         */
  int32_t post_sweeps;      /* nu2, default 2                                               */
  int32_t smoother;         /* 0 = L1-Jacobi  d_i = sum_j |a_ij|  (A7);  1 = damped Jacobi;
                               2 = Chebyshev-accelerated L1-Jacobi (NEXT-4): the nu sweeps of a smoothing step are
                               x += tau_j D_l1^-1 (b - A x) with tau_j the reciprocal roots of the degree-nu Chebyshev
                               polynomial of [1/cheby_ratio, 1]; post-sweeps in reverse order                 */
  int32_t coarse_max_rows;  /* stop coarsening at n_l <= this; default 64 (A6)              */
  int32_t max_levels;       /* default 32                                                   */
  int32_t max_match_rounds; /* 0 = until fix-point                                          */
  double omega;             /* damped Jacobi weight, default 2/3                            */
  double strong_beta;       /* beta, default 0.25 (A2)                                      */
  double coarse_scale;      /* gamma, default 1.0 (A9)                                      */
  uint64_t hash_seed;       /* tie-break salt; level l uses hash_seed + l (A4)              */
  int32_t agg_passes;       /* 1 = pairwise; 2 = the intermediate Galerkin matrix is aggregated
                               again and the maps composed (size-4 aggregates; O-1, NEXT-4);
                               pass p uses the salt hash_seed + l + 1000 p.  default 1       */
  int32_t symmetric;        /* 1 (default): w_ij = -a_ij read from row i (A1);  0: the matching
                               of every level runs on (A_l + A_l^T)/2, union pattern (A1,
                               nonsymmetric case; bitwise equal to 1 for a bitwise symmetric A) */
  int32_t hierarchy_fp32;   /* 1: mixed-precision hierarchy (NEXT-4; "single and double precision"):
                               inside the V-cycle every sparse level operator A_l, l < L, is the fp64 operator with
                               each value rounded to fp32, used in fp64 arithmetic; dinv, the coarsest LU, the Krylov
                               operator A, all vectors and all sums stay fp64.  default 0                        */
  int32_t pad0;
  double cheby_ratio;       /* smoother = 2: the smoothing interval of spec(D_l1^-1 A) is [1/cheby_ratio, 1]; default 6 */
} oracle_options;

typedef struct {
  int32_t iterations;  /* number of passes of the Krylov loop (A11)                  */
  int32_t status;      /* ORACLE_CONVERGED …                                         */
  double rel_residual; /* recurrence ||r||_2 / ||b||_2 at exit (A10)                 */
  double b_norm;       /* ||b||_2                                                    */
} oracle_info;

typedef struct oracle_handle_s* oracle_handle;

void oracle_options_default(oracle_options* o);
void oracle_set_threads(int nthreads); /* OpenMP threads for row loops; dots stay sequential */
int oracle_get_threads(void);

/* O-1: build the hierarchy.  The CSR must have ascending unique columns and a positive
 * diagonal entry in every row. */
int oracle_setup(oracle_handle* out, int32_t n, const int32_t* rowptr, const int32_t* col,
                 const double* val, const oracle_options* opt);
/* Same, but levels 0 … nagg-1 use the given aggregate arrays (aggs[l] has rows(l) entries,
 * ids contiguous 0 … nc-1) instead of O-2.  Coarsening stops after nagg levels. */
int oracle_setup_with_aggregates(oracle_handle* out, int32_t n, const int32_t* rowptr,
                                 const int32_t* col, const double* val,
                                 const oracle_options* opt, int32_t nagg,
                                 const int32_t* const* aggs);
void oracle_destroy(oracle_handle h);

int oracle_num_levels(oracle_handle h);                                  /* L+1 */
int oracle_level_info(oracle_handle h, int32_t level, int32_t* rows, int32_t* nnz);
int oracle_get_aggregates(oracle_handle h, int32_t level, int32_t* agg); /* level < L */
int oracle_get_level_csr(oracle_handle h, int32_t level, int32_t* rowptr, int32_t* col,
                         double* val);
int oracle_get_dinv(oracle_handle h, int32_t level, double* dinv);       /* level < L */
int oracle_match_rounds(oracle_handle h, int32_t level);                 /* rounds O-2 needed */

/* O-2 on its own.  mode 0 = handshake rounds (the definition), mode 1 = greedy matching over
 * candidate edges sorted by descending key (must give the same result on a bitwise
 * symmetric matrix; pin P8).  match[i] = partner or -1; agg[i] in [0, *nc). */
int oracle_aggregate(int32_t n, const int32_t* rowptr, const int32_t* col, const double* val,
                     double beta, uint64_t salt, int32_t max_rounds, int32_t mode, int32_t symmetric,
                     int32_t* match, int32_t* agg, int32_t* nc, int32_t* rounds);
/* O-3 on its own: sizes the output (call with crowptr=NULL to get *cnnz only). */
int oracle_galerkin(int32_t n, const int32_t* rowptr, const int32_t* col, const double* val,
                    const int32_t* agg, int32_t nc, int32_t* crowptr, int32_t* ccol,
                    double* cval, int32_t* cnnz);

/* y = A_level x */
int oracle_spmv(oracle_handle h, int32_t level, const double* x, double* y);
/* one smoother sweep on a level: xout = x + dinv o (b - A x) */
int oracle_smooth(oracle_handle h, int32_t level, const double* b, const double* x, double* xout);
/* rc[I] = sum_{i in I} (b - A_level x)_i */
int oracle_residual_restrict(oracle_handle h, int32_t level, const double* b, const double* x,
                             double* rc);
/* O-4: z = B r, one V-cycle from a zero guess, starting at `level` (0 = the preconditioner) */
int oracle_vcycle(oracle_handle h, int32_t level, const double* r, double* z);

/* O-7: z = B^T r, the same cycle on the transposed level operators A_l^T (same aggregates, same
 * dinv, LU of A_L^T): exactly the transpose of the linear map of oracle_vcycle when nu1 = nu2. */
int oracle_vcycle_transpose(oracle_handle h, int32_t level, const double* r, double* z);

/* smoother = 2: the k sweep weights tau_0 <= ... <= tau_{k-1} of one smoothing step (pre-sweeps in this order,
 * post-sweeps reversed). */
int oracle_cheby_weights(int32_t k, double ratio, double* w);

/* O-5 / O-6.  krylov: 0 = PCG, 1 = right-preconditioned BiCGSTAB.  precond: 1 = AMG V-cycle,
 * 0 = identity.  x0 = 0.  x is output only. */
int oracle_solve(oracle_handle h, const double* b, double* x, double rtol, int32_t maxit,
                 int32_t krylov, int32_t precond, oracle_info* info);
/* O-7: A^T lambda = g.  `symmetric` = 1: identical to oracle_solve on A.
 * symmetric = 0: operator A^T, preconditioner B^T (transposed level operators, same
 * aggregates, same dinv), BiCGSTAB or PCG as requested. */
int oracle_solve_transpose(oracle_handle h, const double* g, double* lambda, double rtol,
                           int32_t maxit, int32_t krylov, int32_t precond, int32_t symmetric,
                           oracle_info* info);
/* ||r_k||_2 / ||b||_2 of the last oracle_solve / oracle_solve_transpose on this handle for
 * k = 1 … iterations (the value the convergence test of iteration k saw).
 * Returns the number of entries; copies at most `cap` of them into `out` (may be NULL). */
int oracle_get_residual_history(oracle_handle h, double* out, int32_t cap);

/* O-8: gA[k] (+)= - sum_b lambda_b[i] x_b[col[k]],  rowptr[i] <= k < rowptr[i+1];  columns of
 * Lambda / X are ld apart. */
int oracle_grad_values(oracle_handle h, const double* lambda, const double* x, int32_t nrhs,
                       int64_t ld, double* gA, int32_t accumulate);

#ifdef __cplusplus
}
#endif
#endif
