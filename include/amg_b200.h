/* amg_b200 — C ABI of the B200-native AMG-preconditioned Krylov solve with adjoint gradients.
 *
 * What it computes (arxiv/paper_2606_09001, "JAX-AMG"; citations are PAPER.md lines):
 *   - the solve  A x = b  of a sparse PDE system in CSR by a Krylov method with an
 *     aggregation-AMG preconditioner (§2.1 "jaxamg.solve", default BiCGSTAB + AMG;
 *     :277 CG), returning iteration count, final residual and convergence status (:125);
 *   - the adjoint solve  A^T lambda = dL/dx  (:87 Eq. 1) on the SAME cached hierarchy;
 *   - the gradients  dL/dA = -lambda x^T  restricted to the stored entries and  dL/db = lambda
 *     (:93 Eq. 2; :186 "gradients with respect to the matrix entries");
 *   - the cached setup: one handle = one cache entry of the paper's solver cache (:103, :121),
 *     reused for any number of right-hand sides (:116, :287 reuse_setup).
 * The paper delegates the numerical algorithm to NVIDIA AmgX and states none of it; the
 * algorithm implemented here is the reading fixed in SURVEY.md §8(c) and DESIGN.md:
 * deterministic pairwise aggregation (handshake matching with a 3-bucket + hash key), Galerkin
 * coarse operators with piecewise-constant prolongation, V(nu1,nu2) cycles with L1-/damped-
 * Jacobi smoothing from a zero guess on every level, dense LU on the coarsest level, PCG or
 * right-preconditioned BiCGSTAB with x0 = 0, stop on the recurrence residual
 * ||r||_2 <= rtol * ||b||_2.
 *
 * Everything is fp64 values / int32 indices, single GPU (sm_100a).  No torch types cross this
 * boundary: plain pointers and sizes.
 *
 * POINTERS.  Arguments prefixed d_ are DEVICE pointers, h_ are HOST pointers; `opt`, `info`,
 * `out` scalars are host pointers.  The caller owns every buffer it passes; the library never
 * frees or reallocates them and copies what it needs during amg_setup (the CSR arrays may be
 * released after amg_setup returns).  Library-owned memory (hierarchy, work vectors, setup
 * temporaries) comes from the device's default stream-ordered memory pool (cudaMallocAsync,
 * release threshold raised so that repeated setups reuse it), or from the allocator hook if
 * one is installed, and is released by amg_destroy.
 *
 * STREAMS.  Every call enqueues its work on `cuda_stream` (a cudaStream_t passed as void*;
 * NULL = the legacy default stream).  A solve is: one init kernel, one graph whose conditional
 * WHILE node repeats the iteration until the device-side convergence test says stop, one output
 * kernel -- nothing of the loop involves the host.  With info != NULL the call then waits for
 * the stream and reports; with info == NULL it returns at once (fully asynchronous).  Hooks,
 * gradients and amg_get_aggregates are stream-ordered and do not synchronise.  Graphs are
 * captured on an internal stream and launched into `cuda_stream`.
 *
 * ERRORS.  Every function returns amg_status; no exception crosses the ABI.  On a failed
 * amg_setup *out is NULL and amg_last_error(NULL) holds a message (thread-local).
 * Non-convergence is NOT an error: it is reported in amg_info.status.
 *
 * NUMBERING.  Internally every level is stored in an aggregate-contiguous order (DESIGN.md
 * §layout); vectors are permuted at this boundary.  All arrays crossing the ABI — b, x, g,
 * lambda, gA, aggregates, level CSR — are in the caller's (natural) numbering.
 *
 * THREADS.  Distinct handles may be used concurrently from distinct host threads on distinct
 * streams; one handle runs one call at a time.
 */
#ifndef AMG_B200_H
#define AMG_B200_H
#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define AMG_API __attribute__((visibility("default")))
#else
#define AMG_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct amg_handle_s* amg_handle;

typedef enum {
  AMG_OK = 0,
  AMG_ERR_INVALID_ARG = 1,
  AMG_ERR_BAD_CSR = 2,          /* rowptr not monotone / col out of range or unsorted / no positive diagonal */
  AMG_ERR_CUDA = 3,
  AMG_ERR_OOM = 4,
  AMG_ERR_COARSE_SINGULAR = 5,  /* dense LU of the coarsest operator found a zero pivot */
  AMG_ERR_COARSEN_STALL = 6,    /* coarsening stalled above 4096 rows */
  AMG_ERR_UNSUPPORTED = 7
} amg_status;

typedef enum { AMG_CONVERGED = 0, AMG_MAXIT = 1, AMG_BREAKDOWN = 2, AMG_NONFINITE = 3 } amg_conv;

/* Filled by amg_options_default(); struct_size guards ABI growth. */
typedef struct {
  int32_t struct_size;
  int32_t krylov;           /* 0 = PCG, 1 = right-preconditioned BiCGSTAB (paper default)   */
  int32_t symmetric;        /* -1 (default) = check on the device at setup, bitwise a_ij == a_ji, one cheap kernel;
                                1 = caller asserts A == A^T (no check; no transposition for the adjoint, :95, :114);
                                0 = not symmetric: the matching of every level runs on (A_l + A_l^T)/2 and
                                    amg_solve_transpose uses the transposed hierarchy            */
  int32_t agg_passes;       /* 1 = pairwise aggregation (default); 2 = the intermediate Galerkin matrix is
                               aggregated again and the maps composed (size-4 aggregates); pass p of level l
                               uses the salt hash_seed + l + 1000 p                                          */
  int32_t pre_sweeps;       /* nu1, default 2                                                            */
  int32_t post_sweeps;      /* nu2, default 2                                                            */
  int32_t smoother;         /* 0 = L1-Jacobi (d_i = sum_j |a_ij|), 1 = damped Jacobi (omega / a_ii),
                               2 = Chebyshev-accelerated L1-Jacobi: the nu sweeps of a smoothing step are
                                   x += tau_j D_l1^-1 (b - A x), tau_j the reciprocal roots of the degree-nu Chebyshev
                                   polynomial of [1/cheby_ratio, 1] (spec(D_l1^-1 A) lies in (0, 1]); post-sweeps in
                                   reverse order                                                          */
  int32_t coarse_max_rows;  /* stop coarsening at n_l <= this (default 64); dense LU there               */
  int32_t max_levels;       /* default 32                                                                */
  int32_t max_match_rounds; /* 0 = handshake rounds until the fix-point                                  */
  int32_t force_generic;    /* 1 = use the row-vector fallback kernels on every level (tests)            */
  int32_t use_graph;        /* 1 = replay one Krylov iteration as a CUDA graph (default), 0 = plain launches */
  int32_t tail_dense_rows;  /* the V-cycle from the first level with at most this many rows down to the
                               coarsest solve is applied as ONE dense operator assembled at setup (the same
                               linear map); default 2304, 0 = off                            */
  int32_t use_pdl;          /* 1 = the kernels of a captured iteration are chained by programmatic dependent
                               launches (a kernel becomes resident while its predecessor drains); default 1 */
  int32_t split_prolong_rows; /* levels with at least this many rows apply the coarse correction x += gamma P e_c
                               as its own unit-stride pass instead of fusing it into the first post-sweep
                               (the fused sweep gathers two values per halo column); default 800000, 0 = never */
  int32_t use_while;        /* 1 = the whole Krylov loop is ONE graph launch: a conditional WHILE node whose body is one
                               iteration, the loop condition set on the device from the convergence flag (no host
                               polling, no surplus iteration); default 1; falls back to replaying the iteration
                               graph under host control if the driver refuses the node; 0 = host-controlled loop   */
  double omega;             /* damped Jacobi weight, default 2/3                                         */
  double strong_beta;       /* strength threshold beta, default 0.25                                     */
  double coarse_scale;      /* gamma: x += gamma * P e_c, default 1.0                                    */
  uint64_t hash_seed;       /* tie-break salt of the matching; level l uses hash_seed + l                */
  int32_t hierarchy_fp32;   /* 1 = mixed-precision hierarchy: inside the V-cycle every sparse level operator
                               A_l, l < L, is stored with fp32 values (6 bytes per entry instead of 10) and used in fp64
                               arithmetic; dinv, the coarsest LU, the Krylov operator A (level 0 keeps an fp64 copy), all
                               vectors and all sums stay fp64.  The solve still converges to rtol in fp64.  In this mode
                               the per-level hooks (amg_level_op) see the rounded operators.  default 0            */
  int32_t value_dict;       /* 1 (default) = value dictionary: a level whose operator holds at most 255 distinct fp64 values
                               (constant-coefficient stencils and their Galerkin sums) is stored in the tile blobs as
                               8-bit codes into a table of those values -- 3 bytes per entry instead of 10, the values and
                               every result bit-identical; other levels keep fp64 values.  Ignored with hierarchy_fp32 = 1 */
  double cheby_ratio;       /* smoother = 2: smoothing interval [1/cheby_ratio, 1]; default 6                    */
} amg_options;

typedef struct {
  int32_t iterations;   /* passes of the Krylov loop                                                     */
  int32_t status;       /* amg_conv                                                                      */
  double rel_residual;  /* recurrence ||r||_2 / ||b||_2 at exit                                          */
  double b_norm;        /* ||b||_2                                                                       */
} amg_info;

/* Timings of the last amg_setup, for the report ("timed separately", BASELINE.json). */
typedef struct {
  double total_ms;      /* host wall clock of amg_setup                                                  */
  double aggregate_ms;  /* U1-U3 over all levels                                                         */
  double galerkin_ms;   /* U4 over all levels                                                            */
  double reorder_ms;    /* aggregate-contiguous renumbering of the hierarchy                             */
  double lu_ms;         /* U6                                                                            */
  int32_t match_rounds_max;
  int32_t reserved;
} amg_setup_stats;

AMG_API amg_status amg_options_default(amg_options* opt);

/* Optional: route library-owned device memory through the caller's allocator (e.g. torch's
 * caching allocator).  A handle keeps the allocator that was installed when it was created.  Pass NULLs
 * to restore the stream-ordered pool.  free_fn may be called while work that uses the block is still queued
 * on the stream the block was allocated on: the allocator must be stream-ordered on that stream (torch's
 * caching allocator, cudaFreeAsync) or synchronise itself (cudaFree). */
AMG_API amg_status amg_set_allocator(void* (*alloc_fn)(size_t bytes, void* cuda_stream, void* user),
                             void (*free_fn)(void* ptr, void* user), void* user);

/* U1-U7: validate the CSR (ascending unique columns, positive diagonal in every row), build
 * and cache the hierarchy.  d_rowptr int32[n+1], d_col int32[nnz], d_val double[nnz]. */
AMG_API amg_status amg_setup(amg_handle* out, int64_t n, int64_t nnz, const int32_t* d_rowptr,
                     const int32_t* d_col, const double* d_val, const amg_options* opt,
                     void* cuda_stream);

/* Test hook: same, but levels 0..nagg-1 use the given aggregate arrays (h_d_aggs is a HOST
 * array of nagg DEVICE pointers; aggs[l] has rows(l) int32 ids in [0, nc_l), every id used)
 * instead of the built-in matching; coarsening stops after nagg levels. */
AMG_API amg_status amg_setup_with_aggregates(amg_handle* out, int64_t n, int64_t nnz,
                                     const int32_t* d_rowptr, const int32_t* d_col,
                                     const double* d_val, const amg_options* opt, int32_t nagg,
                                     const int32_t* const* h_d_aggs, void* cuda_stream);

/* Warm resetup (the paper's cache-hit path: "matrix coefficients are updated in
 * place" and the setup is repeated on the new values; the operation its Fig. 3 benchmarks, :285).
 * d_val double[nnz]: new values on the SAME pattern as the amg_setup call (device pointer, read
 * only during the call, not borrowed).  keep_aggregates = 1: the aggregates of the current
 * hierarchy are kept (no matching: Galerkin products, smoother diagonals, tile blobs, coarse LU
 * and the dense tail operator are recomputed); 0: everything is rebuilt, the result equals a cold
 * amg_setup on the new values.  The handle stays valid; on an error it keeps its old hierarchy. */
AMG_API amg_status amg_resetup_values(amg_handle h, const double* d_val, int32_t keep_aggregates,
                                      void* cuda_stream);

AMG_API amg_status amg_destroy(amg_handle h);

/* S1-S9: solve A x = b from x0 = 0 with the Krylov method of the options (a nonsymmetric handle
 * always uses BiCGSTAB: PCG needs A = A^T); x is output only.  ||b|| = 0 gives x = 0, 0 iterations,
 * converged.  info == NULL: nothing is reported and the call does not wait for the end of the solve
 * (it returns with at most the last iteration and the output kernel still in the stream; x is
 * valid in stream order). */
AMG_API amg_status amg_solve(amg_handle h, const double* d_b, double* d_x, double rtol, int32_t maxit,
                     amg_info* info, void* cuda_stream);
/* Same with an explicit Krylov method (0 PCG, 1 BiCGSTAB) and preconditioner switch
 * (1 = AMG V-cycle, 0 = identity: plain CG / BiCGSTAB as in PAPER.md:277). */
AMG_API amg_status amg_solve_ex(amg_handle h, const double* d_b, double* d_x, double rtol, int32_t maxit,
                        int32_t krylov, int32_t precond, amg_info* info, void* cuda_stream);
/* G1: A^T lambda = g on the same hierarchy (Eq. 1).  Symmetric handle: the transposition is
 * skipped and this is amg_solve on A.  Nonsymmetric handle ("forms
 * A^T ... then solves the adjoint system"): right-preconditioned BiCGSTAB on A^T with the
 * preconditioner B^T -- the same V-cycle on the transposed level operators A_l^T (= the Galerkin
 * hierarchy of A^T on the same aggregates), same smoother diagonals, LU of A_L^T; the transposed
 * operators are built on the device at setup (hand-written CSR transpose) and tile-packed like
 * the forward ones. */
AMG_API amg_status amg_solve_transpose(amg_handle h, const double* d_g, double* d_lambda, double rtol,
                               int32_t maxit, amg_info* info, void* cuda_stream);
/* S10: nrhs independent solves on one hierarchy; column s of B / X starts at s * ld.
 * transpose = 1 solves the adjoint systems.  infos: host array of nrhs entries or NULL. */
AMG_API amg_status amg_solve_batched(amg_handle h, int32_t transpose, const double* d_B, double* d_X,
                             int32_t nrhs, int64_t ld, double rtol, int32_t maxit, amg_info* infos,
                             void* cuda_stream);
/* End-to-end variant with HOST buffers: copies b to the device, solves, copies x back. */
AMG_API amg_status amg_solve_host(amg_handle h, const double* h_b, double* h_x, double rtol,
                          int32_t maxit, amg_info* info, void* cuda_stream);

/* G2: gA[k] (+)= - sum_{s < nrhs} lambda_s[i] * x_s[col[k]]  for rowptr[i] <= k < rowptr[i+1]
 * on the pattern given to amg_setup (Eq. 2; each stored entry is its own parameter).
 * Column s of Lambda / X starts at s * ld.  accumulate = 0 overwrites gA.
 * G3: dL/db = lambda is the caller's lambda itself (no call). */
AMG_API amg_status amg_grad_values(amg_handle h, const double* d_lambda, const double* d_x, int32_t nrhs,
                           int64_t ld, double* d_gA, int32_t accumulate, void* cuda_stream);

/* G2 without any allocation and without a handle (for callers under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same result as amg_grad_values (Eq. 2),
 *   gA[k] (+)= - sum_{s < nrhs} lambda_s[i] * x_s[col[k]]  for rowptr[i] <= k < rowptr[i+1],
 * on the pattern the CALLER passes: d_rowptr int32[n + 1], d_col int32[nnz], d_gA f64[nnz], d_lambda / d_x
 * f64 with column s at s * ld (ld >= n); all DEVICE pointers owned by the caller, on the current device.
 * The interleaved copy of X that the batched kernel gathers from lives in a file-scope static device array of
 * AMG_NOALLOC_MAX_DOUBLES values (8 MiB; every GPU that loads the library holds it until the process exits).
 * Limits: n * nrhs <= AMG_NOALLOC_MAX_DOUBLES and nrhs <= 94, else AMG_ERR_UNSUPPORTED with a message in
 * amg_last_error(NULL); null pointers / ld < n: AMG_ERR_INVALID_ARG.  The call enqueues two kernels on
 * cuda_stream and returns; it calls no cudaMalloc, cudaFree or allocating library routine and does not
 * synchronise.  Every call on a device shares the one array, which keeps the previous call's contents (each
 * call overwrites what it reads, nothing needs clearing): calls that OVERLAP on the GPU -- different streams, or
 * several host threads on one device -- race on it; order them on one stream or with events. */
#define AMG_NOALLOC_MAX_DOUBLES (1 << 20)
AMG_API amg_status amg_grad_values_noalloc(int64_t n, int64_t nnz, const int32_t* d_rowptr, const int32_t* d_col,
                                           const double* d_lambda, const double* d_x, int32_t nrhs, int64_t ld,
                                           double* d_gA, int32_t accumulate, void* cuda_stream);

/* z = B r: one V-cycle from a zero guess (the preconditioner; also the V-cycle timing hook). */
AMG_API amg_status amg_apply_preconditioner(amg_handle h, const double* d_r, double* d_z,
                                    void* cuda_stream);

/* ---- introspection / parity hooks (natural numbering) ---- */
AMG_API amg_status amg_get_num_levels(amg_handle h, int32_t* num_levels);
AMG_API amg_status amg_get_level_info(amg_handle h, int32_t level, int64_t* rows, int64_t* nnz);
AMG_API amg_status amg_get_aggregates(amg_handle h, int32_t level, int32_t* d_agg_out, void* cuda_stream);
/* Diagnostics: ||r_k||_2 / ||b||_2 for k = 1 .. iterations of the last solve on this handle
 * that was called with info != NULL -- the value the convergence test of iteration k saw (BiCGSTAB: ||s|| of a
 * half-step exit, else ||r||).  *count = number of entries; at most `cap` are copied to the HOST array h_out. */
AMG_API amg_status amg_get_residual_history(amg_handle h, double* h_out, int32_t cap, int32_t* count,
                                            void* cuda_stream);
/* Diagnostics file ("optional file-based output provides detailed AMG hierarchy statistics and
 * per-iteration residual histories"): writes a plain-text report to `path` (HOST string) -- per level rows, nonzeros,
 * entries per row, aggregation rounds, kernel path, tiles; grid / operator complexity; the options in force; the
 * setup timings; the residual history of the last reporting solve.  Synchronises `cuda_stream`. */
AMG_API amg_status amg_write_report(amg_handle h, const char* path, void* cuda_stream);
/* 1 / 0: what the setup decided (the caller's flag, or the result of the device check for -1). */
AMG_API amg_status amg_get_symmetric(amg_handle h, int32_t* symmetric);
AMG_API amg_status amg_get_level_csr(amg_handle h, int32_t level, int32_t* d_rowptr, int32_t* d_col,
                             double* d_val, void* cuda_stream);
AMG_API amg_status amg_get_setup_stats(amg_handle h, amg_setup_stats* stats);
/* 1 if `level` runs the row-block streaming kernels, 0 if the row-vector fallback. */
AMG_API amg_status amg_get_level_path(amg_handle h, int32_t level, int32_t* fast_path);
/* Algorithmic bytes of: which = 0 one level-0 SpMV, 1 one V-cycle,
 * 2 one PCG iteration (SpMV + vector ops + V-cycle), 3 one BiCGSTAB iteration,
 * 4 one level-0 smoother sweep.  Stored sizes (not algorithmic): 10 = bytes of the tile blobs of all levels the
 * V-cycle streams, 11 = of level 0 alone, 12 = number of levels stored as 8-bit codes (value_dict). */
AMG_API amg_status amg_get_algorithmic_bytes(amg_handle h, int32_t which, double* bytes);

/* Kernel launches enqueued by the last amg_solve* / amg_level_op / amg_grad_values call on this
 * handle (graph replays count their kernel nodes); the caller's evidence for "gpu_launches". */
AMG_API amg_status amg_get_last_launches(amg_handle h, int64_t* launches);

/* Per-kernel hooks on one level, vectors in that level's natural numbering:
 *   op 0: y = A_l x                               (d_in0 = x,           d_out rows(l))
 *   op 1: xout = x + dinv o (b - A_l x)           (d_in0 = x, d_in1 = b, d_out rows(l))
 *   op 2: rc = R (b - A_l x)                      (d_in0 = x, d_in1 = b, d_out rows(l+1))
 *   op 3: xout = x + gamma * P e_c                (d_in0 = x, d_in1 = e_c rows(l+1), d_out rows(l))
 *   op 4: two fused sweeps from zero: x2 of b     (d_in1 = b,           d_out rows(l))
 *   op 5: V-cycle started at level l              (d_in1 = b,           d_out rows(l))
 *   op 6: xout = x~ + dinv o (b - A_l x~), x~ = x + gamma * P e_c
 *                                                 (d_in0 = x, d_in1 = [b rows(l) | e_c rows(l+1)], d_out rows(l))
 *   op 7: y = A_l^T x   (nonsymmetric handles)    (d_in0 = x,           d_out rows(l))
 *   op 8: transposed V-cycle started at level l   (d_in1 = b,           d_out rows(l))
 * The calls are stream-ordered (no synchronisation).
 * `reps` > 1 repeats the kernel back to back (timing); results are those of one application.  For op 1
 * on level 0 the repetitions rotate over three internal copies of the operands (x, b, dinv, out: 12
 * level-0 vectors), so that no operand of a launch is still in L2 from the launch before. */
AMG_API amg_status amg_level_op(amg_handle h, int32_t level, int32_t op, const double* d_in0,
                        const double* d_in1, double* d_out, int32_t reps, void* cuda_stream);

/* ---- keyed LRU cache of hierarchies ("LRU cache of solver handles keyed by a hash of the
 * sparsity pattern"; :121; :287 reuse_setup) ----
 * amg_cache_get looks the matrix up by a 64-bit hash of (n, nnz, rowptr, col, options), computed on the device.
 *   miss: amg_setup; the handle is inserted and the least recently used one beyond `capacity` is destroyed.
 *   hit:  on_hit = 0 the cached handle is returned as it is (same values: reuse_setup);
 *         on_hit = 1 amg_resetup_values(h, d_val, keep_aggregates = 0): "coefficients are updated in place and
 *                    the setup is repeated"; on_hit = 2 the same with the aggregates kept.
 * The handles belong to the cache (amg_cache_destroy destroys them; never call amg_destroy on one); a handle
 * stays valid until it is evicted.  *hit (may be NULL) reports which case it was.  One call at a time per cache
 * (an internal mutex serialises them). */
typedef struct amg_cache_s* amg_cache;
AMG_API amg_status amg_cache_create(amg_cache* out, int32_t capacity);
AMG_API amg_status amg_cache_get(amg_cache c, int64_t n, int64_t nnz, const int32_t* d_rowptr, const int32_t* d_col,
                                 const double* d_val, const amg_options* opt, int32_t on_hit, amg_handle* out,
                                 int32_t* hit, void* cuda_stream);
AMG_API amg_status amg_cache_stats(amg_cache c, int64_t* entries, int64_t* hits, int64_t* misses,
                                   int64_t* evictions);
AMG_API amg_status amg_cache_destroy(amg_cache c);

/* Message of the last error on this handle; NULL handle: last failed setup on this thread. */
AMG_API const char* amg_last_error(amg_handle h);

#ifdef __cplusplus
}
#endif
#endif
