"""Writes tests/golden/full_size_*.txt: what the CPU oracle (and only the oracle) computes on the
full-size BASELINE.json configurations that are too slow to re-run inside the GPU test suite.

    python tests/golden/make_full_size_golden.py [cfg4] [cfg5] [cfg2] [tuned]    (about 90 minutes on 8 cores)

"tuned" writes the same files with the suffix _tuned for the solver options bench.py runs these configurations with
(size-4 aggregation, Chebyshev-weighted L1-Jacobi, gamma = 1.6; oracle options of the same names).

Every solve runs ONCE to rtol 1e-13 ("converged", reading A12); the iteration count at the timed
tolerance 1e-8 is read off the oracle's residual history (the iterates do not depend on rtol).

cfg 4 (192^3 variable-coefficient diffusion, permuted rows; BASELINE.json configs[3]) -> full_size_oracle.txt
    level shapes, iterations / recurrence residual at 1e-8, and the converged x at NS sampled rows.
cfg 5 (same matrix; configs[4]), right-hand sides s = 0, 7, 15 of the 16 (SURVEY.md §8(d) allows the
    subsample) -> full_size_cfg5.txt
    forward solve A x_s = b_s, adjoint solve A^T lambda_s = x_s - x_target,s (A symmetric: same operator),
    iterations at 1e-8 of both, x_s / lambda_s at NS sampled rows, and the single-column gradient
    gA_s[k] = -lambda_s[row(k)] x_s[col(k)] (Eq. 2 on the pattern) at NS sampled entries.
cfg 2 (2D Poisson 1024^2, 8 manufactured right-hand sides on one hierarchy; configs[1]) -> full_size_cfg2.txt
    iterations at 1e-8 and the converged x at NS2 sampled rows for each of the 8.

Sample positions come from numpy's PCG64 with the seeds below; the GPU test draws the same ones.
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2606_09001_b200 import inputs  # noqa: E402  (seeded generators only: no method arithmetic)

NS, NS2 = 10000, 4096
SEED_ROWS, SEED_ENTRIES = 9001, 9002
CFG5_COLUMNS = (0, 7, 15)
RTOL_TIMED, RTOL_CONVERGED, MAXIT = 1e-8, 1e-13, 600
OPTS, SUFFIX = {}, ""   # "tuned": the options of bench.py
TUNED = dict(smoother=2, agg_passes=2, coarse_scale=1.6)


def sample_rows(n, count=NS):
    return np.random.default_rng(SEED_ROWS).integers(0, n, count)


def sample_entries(nnz, count=NS):
    return np.random.default_rng(SEED_ENTRIES).integers(0, nnz, count)


def its_at(hist, rtol):
    """first k (1-based) with ||r_k|| <= rtol ||b||, and that residual"""
    k = int(np.argmax(hist <= rtol))
    assert hist[k] <= rtol
    return k + 1, float(hist[k])


def fmt(v):
    return " ".join(f"{x:.17g}" for x in np.asarray(v, dtype=np.float64))


def converged_solve(o, b):
    t = time.time()
    x, info = o.solve(b, RTOL_CONVERGED, MAXIT, 0, 1)
    hist = o.residual_history()
    k8, r8 = its_at(hist, RTOL_TIMED)
    return x, info, k8, r8, time.time() - t


def write(name, lines):
    with open(os.path.join(HERE, name), "w") as f:
        f.write("\n".join(lines) + "\n")
    print(f"wrote {name} ({len(lines)} lines)", flush=True)


def cfg4_and_5(do4, do5):
    A = inputs.config_matrix(4, 192)
    t = time.time()
    o = oracle.Oracle(A.rowptr, A.col, A.val, **OPTS)
    ts = time.time() - t
    rows_s, ent_s = sample_rows(A.n), sample_entries(A.nnz)
    row_of = np.searchsorted(A.rowptr, ent_s, side="right") - 1
    if do4:
        b = inputs.config_rhs(4, A.n)
        x, info, k8, r8, tv = converged_solve(o, b)
        shapes = [o.level_info(l) for l in range(o.num_levels)]
        out = ["# written by tests/golden/make_full_size_golden.py (CPU oracle only); cfg 4 = BASELINE.json configs[3]" +
               (f"; oracle options {OPTS}" if OPTS else ""),
               f"# oracle setup {ts:.0f} s, solve to 1e-13 {tv:.0f} s ({info.iterations} iterations) on {os.cpu_count()} cores",
               f"cfg4_192 iterations {k8}", f"cfg4_192 rel_residual {r8:.17g}", f"cfg4_192 levels {o.num_levels}",
               "cfg4_192 rows " + " ".join(str(r) for r, _ in shapes),
               "cfg4_192 nnz " + " ".join(str(z) for _, z in shapes),
               f"cfg4_192 converged_iterations {info.iterations}", f"cfg4_192 converged_status {info.status}",
               f"cfg4_192 sample_rows_seed {SEED_ROWS} {NS}",
               "cfg4_192 x_converged " + fmt(x[rows_s])]
        write(f"full_size_oracle{SUFFIX}.txt", out)
    if do5:
        out = ["# written by tests/golden/make_full_size_golden.py (CPU oracle only); cfg 5 = BASELINE.json configs[4],",
               f"# right-hand sides {CFG5_COLUMNS} of 16; x, lambda at rows rng({SEED_ROWS}).integers(0, n, {NS}),",
               f"# gA_s = -lambda_s[row(k)] x_s[col(k)] at entries rng({SEED_ENTRIES}).integers(0, nnz, {NS})"]
        for s in CFG5_COLUMNS:
            b = inputs.config_rhs(5, A.n, s)
            x, info, k8, r8, tv = converged_solve(o, b)
            g = x - inputs.config_target(A.n, s)
            lam, info_a, k8a, r8a, tva = converged_solve(o, g)  # symmetric: A^T lambda = g is A lambda = g
            gA = o.grad_values(lam, x)
            out += [f"# rhs {s}: forward {tv:.0f} s ({info.iterations} its), adjoint {tva:.0f} s ({info_a.iterations} its)",
                    f"cfg5_rhs{s} iterations {k8}", f"cfg5_rhs{s} rel_residual {r8:.17g}",
                    f"cfg5_rhs{s} converged_status {info.status}",
                    f"cfg5_rhs{s} adjoint_iterations {k8a}", f"cfg5_rhs{s} adjoint_rel_residual {r8a:.17g}",
                    f"cfg5_rhs{s} adjoint_converged_status {info_a.status}",
                    f"cfg5_rhs{s} x_converged " + fmt(x[rows_s]),
                    f"cfg5_rhs{s} lambda_converged " + fmt(lam[rows_s]),
                    f"cfg5_rhs{s} gA " + fmt(gA[ent_s])]
            assert np.array_equal(gA[ent_s], -(lam[row_of] * x[A.col[ent_s]]))
            write(f"full_size_cfg5{SUFFIX}.txt", out)  # keep what is done so far
    o.close()


def cfg2():
    A = inputs.config_matrix(2, 1024)
    Asp = A.to_scipy()
    t = time.time()
    o = oracle.Oracle(A.rowptr, A.col, A.val, **OPTS)
    ts = time.time() - t
    rows_s = sample_rows(A.n, NS2)
    shapes = [o.level_info(l) for l in range(o.num_levels)]
    out = ["# written by tests/golden/make_full_size_golden.py (CPU oracle only); cfg 2 = BASELINE.json configs[1]:",
           f"# 8 right-hand sides b_s = A x_true,s on one hierarchy (oracle setup {ts:.0f} s); x at rows rng({SEED_ROWS}).integers(0, n, {NS2})",
           f"cfg2_1024 levels {o.num_levels}",
           "cfg2_1024 rows " + " ".join(str(r) for r, _ in shapes),
           "cfg2_1024 nnz " + " ".join(str(z) for _, z in shapes)]
    for s in range(8):
        b = Asp @ inputs.config_rhs(2, A.n, s)
        x, info, k8, r8, tv = converged_solve(o, b)
        out += [f"# rhs {s}: {tv:.0f} s ({info.iterations} its)",
                f"cfg2_rhs{s} iterations {k8}", f"cfg2_rhs{s} rel_residual {r8:.17g}",
                f"cfg2_rhs{s} converged_status {info.status}",
                f"cfg2_rhs{s} x_converged " + fmt(x[rows_s])]
    o.close()
    write(f"full_size_cfg2{SUFFIX}.txt", out)


def main():
    global OPTS, SUFFIX
    which = set(sys.argv[1:])
    if "tuned" in which:
        OPTS, SUFFIX = dict(TUNED), "_tuned"
        which.discard("tuned")
    which = which or {"cfg4", "cfg5", "cfg2"}
    oracle.build()
    oracle.set_threads(os.cpu_count() or 1)
    if "cfg2" in which:
        cfg2()
    if which & {"cfg4", "cfg5"}:
        cfg4_and_5("cfg4" in which, "cfg5" in which)


if __name__ == "__main__":
    main()
