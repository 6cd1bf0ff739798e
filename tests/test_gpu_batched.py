"""GPU parity of the batched multi-right-hand-side kernels ("the
matrix is shared across the batch"): amg_solve_batched with >= 4 columns runs ONE operator pass for 8
interleaved right-hand sides with per-column Krylov scalars and convergence masks.  Every column is
compared with the oracle's solve of that column on the identical hierarchy: iterations +-2, host fp64
residual <= 1e-8, x against the converged solution <= 1e-6 (A12).
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

from paper_2606_09001_b200 import inputs  # noqa: E402


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / max(np.linalg.norm(np.asarray(b)), 1e-300))


@pytest.fixture(scope="module")
def B():
    from paper_2606_09001_b200 import binding

    assert torch.cuda.is_available()
    binding.load_library()
    return binding


def rhs_columns(A, nrhs, seed):
    """Columns that converge at different iteration counts: random, smooth (A * ones), a single spike, a zero
    column, a scaled copy -- the masks of finished columns are exercised."""
    rng = np.random.default_rng(seed)
    Asp = A.to_scipy()
    cols = []
    for k in range(nrhs):
        kind = k % 5
        if kind == 0:
            cols.append(rng.uniform(-1, 1, A.n))
        elif kind == 1:
            cols.append(Asp @ np.ones(A.n))
        elif kind == 2:
            e = np.zeros(A.n)
            e[rng.integers(0, A.n)] = 1.0
            cols.append(e)
        elif kind == 3:
            cols.append(np.zeros(A.n) if k == 3 else 1e6 * rng.standard_normal(A.n))
        else:
            cols.append(Asp @ rng.standard_normal(A.n))
    return np.stack(cols)


@pytest.mark.parametrize("opts", [dict(), dict(use_graph=0), dict(use_pdl=0), dict(tail_dense_rows=300)])
@pytest.mark.parametrize("case,nrhs", [((3, 40), 8), ((4, 28), 13), ((2, 96), 16), ((3, 24), 5)])
def test_batched_solve_matches_the_oracle_column_by_column(oracle_mod, B, case, nrhs, opts):
    cfg, edge = case
    A = inputs.config_matrix(cfg, edge)
    Asp = A.to_scipy()
    n = A.n
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val)
    s = B.AmgSolver(A.rowptr, A.col, A.val, **opts)
    try:
        Bh = rhs_columns(A, nrhs, 100 + nrhs)
        Bd = torch.as_tensor(Bh).cuda().contiguous()
        X = torch.full_like(Bd, float("nan"))
        infos = B.amg_solve_batched(s.h, 0, Bd, X, nrhs, n, 1e-8, 500)
        launches = B.amg_get_last_launches(s.h)
        Xh = X.cpu().numpy()
        its_o = []
        for k in range(nrhs):
            xo, io = o.solve(Bh[k], 1e-8, 500, 0, 1)
            its_o.append(io.iterations)
            assert infos[k].status == io.status == 0, k
            assert abs(infos[k].iterations - io.iterations) <= 2, (k, infos[k].iterations, io.iterations)
            bn = np.linalg.norm(Bh[k])
            assert abs(infos[k].b_norm - bn) <= 1e-12 * max(bn, 1e-300)
            if bn == 0.0:
                assert infos[k].iterations == 0 and not Xh[k].any()
                continue
            assert np.linalg.norm(Bh[k] - Asp @ Xh[k]) <= 1e-8 * bn, k
            assert infos[k].rel_residual <= 1e-8
        assert len(set(its_o)) >= 3  # the columns really finish at different iterations
        assert launches > 0
        # near convergence (A12): every column against the oracle's converged solution
        infos = B.amg_solve_batched(s.h, 0, Bd, X, nrhs, n, 1e-11, 500)
        Xh = X.cpu().numpy()
        for k in range(nrhs):
            if not Bh[k].any():
                continue
            xo, io = o.solve(Bh[k], 1e-13, 500, 0, 1)
            assert infos[k].status == 0 and rel(Xh[k], xo) <= 1e-6, k
        # the adjoint batch of a symmetric matrix is the same batch: bitwise
        XT = torch.empty_like(Bd)
        B.amg_solve_batched(s.h, 1, Bd, XT, nrhs, n, 1e-11, 500)
        assert torch.equal(X, XT)
        # determinism, and independence of a column from its neighbours: column 0 alone in another batch
        B2 = Bd.clone()
        B2[1:] = torch.flip(Bd[1:], dims=[0])
        X2 = torch.empty_like(Bd)
        B.amg_solve_batched(s.h, 0, B2, X2, nrhs, n, 1e-11, 500)
        assert torch.equal(X2[0], X[0])
        # maxit stop: every unfinished column reports MAXIT after exactly 3 iterations
        infos = B.amg_solve_batched(s.h, 0, Bd, X, nrhs, n, 1e-30, 3)
        for k in range(nrhs):
            if Bh[k].any():
                assert infos[k].status == 1 and infos[k].iterations == 3
    finally:
        s.close()
        o.close()


@pytest.mark.parametrize("sweeps", [(1, 1), (3, 2), (1, 3), (2, 1)])
def test_batched_cycle_with_other_sweep_counts(oracle_mod, B, sweeps):
    nu1, nu2 = sweeps
    A = inputs.config_matrix(3, 32)
    n = A.n
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, pre_sweeps=nu1, post_sweeps=nu2)
    s = B.AmgSolver(A.rowptr, A.col, A.val, pre_sweeps=nu1, post_sweeps=nu2)
    try:
        Bh = np.stack([inputs.config_rhs(5, n, k) for k in range(8)])
        Bd = torch.as_tensor(Bh).cuda().contiguous()
        X = torch.empty_like(Bd)
        # a fixed number of iterations: the iterates agree with the oracle's whatever the symmetry of B
        infos = B.amg_solve_batched(s.h, 0, Bd, X, 8, n, 1e-30, 6)
        for k in (0, 3, 7):
            xo, io = o.solve(Bh[k], 1e-30, 6, 0, 1)
            assert infos[k].iterations == io.iterations == 6
            assert rel(X[k].cpu().numpy(), xo) <= 1e-9
            assert abs(infos[k].rel_residual - io.rel_residual) <= 1e-8 * io.rel_residual
    finally:
        s.close()
        o.close()


def test_batched_path_is_the_one_that_runs(B):
    """>= 4 columns on a default symmetric handle take the batched kernels (fewer launches than a loop of
    single solves); force_generic or BiCGSTAB handles loop."""
    A = inputs.config_matrix(3, 40)
    n = A.n
    Bd = torch.as_tensor(np.stack([inputs.config_rhs(5, n, k) for k in range(8)])).cuda().contiguous()
    X = torch.empty_like(Bd)
    counts = {}
    for name, opts in [("batched", dict()), ("loop", dict(krylov=1))]:
        s = B.AmgSolver(A.rowptr, A.col, A.val, **opts)
        infos = B.amg_solve_batched(s.h, 0, Bd, X, 8, n, 1e-8, 500)
        assert all(i.status == 0 for i in infos)
        counts[name] = B.amg_get_last_launches(s.h)
        s.close()
    s = B.AmgSolver(A.rowptr, A.col, A.val)
    one = 0
    x = torch.empty(n, dtype=torch.float64, device="cuda")
    B.amg_solve(s.h, Bd[0].contiguous(), x, 1e-8, 500)
    one = B.amg_get_last_launches(s.h)
    s.close()
    assert counts["batched"] < 2 * one  # 8 columns for about the launches of one solve


def test_batched_work_vectors_need_no_initialisation(B):
    """Regression: the search direction p is not initialised; beta = 0 must give p = z exactly whatever the
    buffer held.  The library's memory is routed through torch's allocator, whose cached blocks are NaN."""
    import ctypes as C

    lib = B.load_library()
    ALLOC = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p)
    FREE = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)
    a_cb = ALLOC(lambda nbytes, stream, user: torch.cuda.caching_allocator_alloc(int(nbytes), device=0, stream=stream or 0))
    f_cb = FREE(lambda p, user: torch.cuda.caching_allocator_delete(p))
    A = inputs.config_matrix(3, 32)
    n = A.n
    Bd = torch.as_tensor(np.stack([inputs.config_rhs(5, n, k) for k in range(8)])).cuda().contiguous()
    X = torch.empty_like(Bd)
    poison = [torch.full((n * 8,), float("nan"), dtype=torch.float64, device="cuda") for _ in range(24)]
    del poison  # back into torch's cache, still NaN
    assert lib.amg_set_allocator(a_cb, f_cb, None) == 0
    try:
        s = B.AmgSolver(A.rowptr, A.col, A.val)
        infos = B.amg_solve_batched(s.h, 0, Bd, X, 8, n, 1e-8, 500)
        assert all(i.status == 0 and i.iterations > 5 for i in infos)
        assert bool(torch.isfinite(X).all())
        s.close()
    finally:
        lib.amg_set_allocator(None, None, None)
