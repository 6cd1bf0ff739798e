"""Full-size BASELINE.json configurations 2, 4 and 5 on the GPU against STORED oracle results
(tests/golden/full_size_*.txt, written by tests/golden/make_full_size_golden.py, which calls only
oracle/ and the seeded generators; the oracle needs ~3 minutes per 192^3 solve).

  cfg 2  1024^2 Poisson, 8 manufactured right-hand sides on ONE hierarchy through amg_solve_batched
  cfg 4  192^3 variable-coefficient diffusion, permuted rows: levels, iterations, converged x
  cfg 5  the same matrix: amg_solve_batched with 16 right-hand sides forward and 16 adjoint, the
         fused 16-column amg_grad_values over the 49.3 M-entry pattern; x, lambda, gA of columns
         0, 7, 15 against the oracle's (SURVEY.md §8(d) allows the subsample)

Bars (BASELINE.json north_star): level shapes exact; iterations at 1e-8 within +-2; host fp64 residual
<= 1e-8; x / lambda against the oracle's CONVERGED samples <= 1e-6 (both sides near convergence, A12:
GPU at 1e-11, oracle at 1e-13); gradient <= 1e-5.
"""
import os

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

from paper_2606_09001_b200 import inputs  # noqa: E402

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
# "default": the library defaults (BASELINE.json configs[0]'s pairwise aggregation, plain L1-Jacobi);
# "tuned": the solver options bench.py measures these configurations with (stored oracle results with suffix _tuned)
MODES = {"default": ("", {}), "tuned": ("_tuned", dict(smoother=2, agg_passes=2, coarse_scale=1.6))}
NS, NS2 = 10000, 4096            # as in make_full_size_golden.py
SEED_ROWS, SEED_ENTRIES = 9001, 9002


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / max(np.linalg.norm(np.asarray(b)), 1e-300))


def golden(name):
    g = {}
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            key, field, *vals = line.split()
            g[(key, field)] = vals
    return g


def gi(g, key, field):
    return int(g[(key, field)][0])


def gv(g, key, field):
    return np.array([float(v) for v in g[(key, field)]])


@pytest.fixture(scope="module")
def B():
    from paper_2606_09001_b200 import binding

    assert torch.cuda.is_available()
    binding.load_library()
    return binding


@pytest.mark.parametrize("mode", list(MODES))
def test_full_size_cfg2_eight_right_hand_sides_on_one_hierarchy(B, mode):
    suffix, opts = MODES[mode]
    g = golden(f"full_size_cfg2{suffix}.txt")
    A = inputs.config_matrix(2)
    Asp = A.to_scipy()
    n = A.n
    s = B.AmgSolver(A.rowptr, A.col, A.val, **opts)
    try:
        rows = [int(v) for v in g[("cfg2_1024", "rows")]]
        nnzs = [int(v) for v in g[("cfg2_1024", "nnz")]]
        assert [s.level_info(l) for l in range(s.num_levels)] == list(zip(rows, nnzs))
        xt = np.stack([inputs.config_rhs(2, n, k) for k in range(8)])
        Bh = np.stack([Asp @ xt[k] for k in range(8)])
        Bd = torch.as_tensor(Bh).cuda().contiguous()
        X = torch.empty_like(Bd)
        infos = B.amg_solve_batched(s.h, 0, Bd, X, 8, n, 1e-8, 1000)
        Xh = X.cpu().numpy()
        for k in range(8):
            assert infos[k].status == 0
            assert abs(infos[k].iterations - gi(g, f"cfg2_rhs{k}", "iterations")) <= 2, k
            assert np.linalg.norm(Bh[k] - Asp @ Xh[k]) <= 1e-8 * np.linalg.norm(Bh[k])
        # near convergence: the oracle's converged x at the sampled rows, and the manufactured solution (P9)
        infos = B.amg_solve_batched(s.h, 0, Bd, X, 8, n, 1e-11, 1000)
        Xh = X.cpu().numpy()
        rows_s = np.random.default_rng(SEED_ROWS).integers(0, n, NS2)
        for k in range(8):
            assert infos[k].status == 0
            assert rel(Xh[k][rows_s], gv(g, f"cfg2_rhs{k}", "x_converged")) <= 1e-6
            assert rel(Xh[k], xt[k]) <= 1e-6
    finally:
        s.close()


@pytest.fixture(scope="module", params=list(MODES))
def full45(B, request):
    suffix, opts = MODES[request.param]
    A = inputs.config_matrix(4)
    s = B.AmgSolver(A.rowptr, A.col, A.val, **opts)
    yield A, A.to_scipy(), s, suffix
    s.close()


def test_full_size_cfg4_against_stored_oracle(full45):
    A, Asp, s, suffix = full45
    g = golden(f"full_size_oracle{suffix}.txt")
    b = inputs.config_rhs(4, A.n)
    assert s.num_levels == gi(g, "cfg4_192", "levels")
    rows = [int(v) for v in g[("cfg4_192", "rows")]]
    nnzs = [int(v) for v in g[("cfg4_192", "nnz")]]
    assert [s.level_info(l) for l in range(s.num_levels)] == list(zip(rows, nnzs))  # integer work: exact
    xg, ig = s.solve(b, 1e-8, 1000, 0)
    assert ig.status == 0 and abs(ig.iterations - gi(g, "cfg4_192", "iterations")) <= 2
    # (not a north_star bar: the recurrence residual at the stopping iteration agrees to the rounding-order differences of
    # the dot products amplified by ~30-70 iterations: 2e-5 with the library defaults, 3e-3 with the over-corrected cycle)
    assert abs(ig.rel_residual - float(g[("cfg4_192", "rel_residual")][0])) <= 2e-2 * ig.rel_residual
    assert np.linalg.norm(b - Asp @ xg.cpu().numpy()) <= 1e-8 * np.linalg.norm(b)
    xg, ig = s.solve(b, 1e-11, 1000, 0)
    rows_s = np.random.default_rng(SEED_ROWS).integers(0, A.n, NS)
    assert ig.status == 0 and rel(xg.cpu().numpy()[rows_s], gv(g, "cfg4_192", "x_converged")) <= 1e-6


def test_full_size_cfg5_batch_of_16_forward_adjoint_gradient(full45, B):
    A, Asp, s, suffix = full45
    g = golden(f"full_size_cfg5{suffix}.txt")
    n, nnz, R = A.n, A.nnz, 16
    cols = (0, 7, 15)
    Bh = np.stack([inputs.config_rhs(5, n, k) for k in range(R)])
    Th = np.stack([inputs.config_target(n, k) for k in range(R)])
    Bd = torch.as_tensor(Bh).cuda().contiguous()
    Td = torch.as_tensor(Th).cuda().contiguous()
    X = torch.empty_like(Bd)
    # ---- 16 forward solves at the timed tolerance: iterations, residuals ----
    infos = B.amg_solve_batched(s.h, 0, Bd, X, R, n, 1e-8, 1000)
    assert all(i.status == 0 for i in infos)
    for k in cols:
        assert abs(infos[k].iterations - gi(g, f"cfg5_rhs{k}", "iterations")) <= 2, k
        xk = X[k].cpu().numpy()
        assert np.linalg.norm(Bh[k] - Asp @ xk) <= 1e-8 * np.linalg.norm(Bh[k])
    its = [i.iterations for i in infos]
    assert max(its) - min(its) <= 6  # same matrix, same kind of right-hand side
    # ---- near convergence (A12): 16 forward + 16 adjoint + the fused gradient ----
    infos = B.amg_solve_batched(s.h, 0, Bd, X, R, n, 1e-11, 1000)
    assert all(i.status == 0 for i in infos)
    G = (X - Td).contiguous()                      # dL/dx of L = 1/2 sum_s ||x_s - x_target,s||^2
    Lam = torch.empty_like(G)
    infos_a = B.amg_solve_batched(s.h, 1, G, Lam, R, n, 1e-11, 1000)
    assert all(i.status == 0 for i in infos_a)
    gA = torch.empty(nnz, dtype=torch.float64, device="cuda")
    B.amg_grad_values(s.h, Lam, X, R, n, gA, 0)
    rows_s = np.random.default_rng(SEED_ROWS).integers(0, n, NS)
    ent_s = np.random.default_rng(SEED_ENTRIES).integers(0, nnz, NS)
    g1 = torch.empty(nnz, dtype=torch.float64, device="cuda")
    for k in cols:
        assert rel(X[k].cpu().numpy()[rows_s], gv(g, f"cfg5_rhs{k}", "x_converged")) <= 1e-6, k
        assert rel(Lam[k].cpu().numpy()[rows_s], gv(g, f"cfg5_rhs{k}", "lambda_converged")) <= 1e-6, k
        B.amg_grad_values(s.h, Lam[k].contiguous(), X[k].contiguous(), 1, n, g1, 0)   # Eq. 2, one column
        assert rel(g1.cpu().numpy()[ent_s], gv(g, f"cfg5_rhs{k}", "gA")) <= 1e-5, k
    # adjoint at the timed tolerance: iterations of the three oracle columns
    Lam8 = torch.empty_like(G)
    infos_a8 = B.amg_solve_batched(s.h, 1, G, Lam8, R, n, 1e-8, 1000)
    for k in cols:
        assert abs(infos_a8[k].iterations - gi(g, f"cfg5_rhs{k}", "adjoint_iterations")) <= 2, k
        gk = G[k].cpu().numpy()
        assert np.linalg.norm(gk - Asp.T @ Lam8[k].cpu().numpy()) <= 1e-8 * np.linalg.norm(gk)
    del Lam8
    # the fused 16-column gradient over the 49.3 M-entry pattern: (i) three columns packed against the sum of
    # the oracle's three single-column gradients; (ii) all 16: sampled entries recomputed one by one on the
    # host from the definition gA[k] = -sum_s lambda_s[row(k)] x_s[col(k)] (the oracle solved 3 of the 16)
    X3 = torch.stack([X[k] for k in cols]).contiguous()
    L3 = torch.stack([Lam[k] for k in cols]).contiguous()
    B.amg_grad_values(s.h, L3, X3, 3, n, g1, 0)
    want3 = sum(gv(g, f"cfg5_rhs{k}", "gA") for k in cols)
    assert rel(g1.cpu().numpy()[ent_s], want3) <= 1e-5
    ks = np.random.default_rng(8).integers(0, nnz, 200000)
    rows_of = np.searchsorted(A.rowptr, ks, side="right") - 1
    cols_of = A.col[ks]
    Xh, Lh = X.cpu().numpy(), Lam.cpu().numpy()
    want = -np.einsum("sk,sk->k", Lh[:, rows_of], Xh[:, cols_of])
    got = gA.cpu().numpy()[ks]
    assert np.max(np.abs(got - want)) <= 1e-13 * np.max(np.abs(want))
    # accumulate = 1 over two halves equals the fused call to rounding
    B.amg_grad_values(s.h, Lam[:8].contiguous(), X[:8].contiguous(), 8, n, g1, 0)
    B.amg_grad_values(s.h, Lam[8:].contiguous(), X[8:].contiguous(), 8, n, g1, 1)
    assert rel(g1.cpu().numpy()[ks], got) <= 1e-13
    # adjoint identity per column (P10 (iii)): g.x = lambda.b
    for k in cols:
        gk, xk, lk = G[k].cpu().numpy(), Xh[k], Lh[k]
        assert abs(gk @ xk - lk @ Bh[k]) <= 1e-8 * np.linalg.norm(gk) * np.linalg.norm(xk)
