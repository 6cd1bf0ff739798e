"""GPU parity of the nonsymmetric path ("for nonsymmetric systems,
the backward pass forms A^T ... then solves the adjoint system"; Eq. 1 at :87): device CSR transpose,
symmetrised strength (reading A1), transposed hierarchy, BiCGSTAB adjoint with B^T -- against the CPU
oracle (oracle_solve_transpose with symmetric = 0, pinned by P10), through the C ABI.

Also the GPU twins of the oracle pins of round 2: dense LU that needs row exchanges, the singleton
merge target, the stall rule.
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


def csr_of(rp, cl, vl):
    import scipy.sparse as sp

    n = len(rp) - 1
    return sp.csr_matrix((vl, cl, rp), shape=(n, n))


NONSYM = {
    "channel_12x20x16": lambda: inputs.stretched_channel_csr((12, 20, 16), 2.0),      # 3840 rows, a few tiles
    "channel_24x40x32": lambda: inputs.stretched_channel_csr((24, 40, 32), 2.2),      # 30720 rows, ~120 tiles on level 0
}


@pytest.mark.parametrize("opts", [dict(), dict(force_generic=1), dict(tail_dense_rows=0), dict(use_graph=0)])
@pytest.mark.parametrize("name", list(NONSYM))
def test_nonsymmetric_hierarchy_and_adjoint(oracle_mod, B, name, opts):
    A = NONSYM[name]()
    Asp = A.to_scipy()
    n = A.n
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, symmetric=0)
    s = B.AmgSolver(A.rowptr, A.col, A.val, **opts)  # default symmetric = -1: detected on the device
    try:
        assert s.symmetric == 0
        # identical hierarchy: aggregates from the matching on (A + A^T)/2, bit-exact
        assert s.num_levels == o.num_levels
        for l in range(s.num_levels - 1):
            assert np.array_equal(s.aggregates(l).cpu().numpy(), o.aggregates(l)), f"level {l}"
        rng = np.random.default_rng(31)
        for l in range(s.num_levels):
            rows, nnz = s.level_info(l)
            rp, cl, vl = o.level_csr(l)
            assert (rows, nnz) == (len(rp) - 1, len(cl))
            Al = csr_of(rp, cl, vl)
            x = rng.standard_normal(rows)
            # y = A_l x and y = A_l^T x (device transpose + its tile blobs), every level
            assert rel(s.level_op(l, 0, x, None, rows).cpu().numpy(), Al @ x) <= 1e-13
            assert rel(s.level_op(l, 7, x, None, rows).cpu().numpy(), Al.T @ x) <= 1e-13
            # the transposed V-cycle from every level: z = B_l^T b
            assert rel(s.level_op(l, 8, None, x, rows).cpu().numpy(), o.vcycle_transpose(x, l)) <= 1e-12
            assert rel(s.level_op(l, 5, None, x, rows).cpu().numpy(), o.vcycle(x, l)) <= 1e-12
        # forward: amg_solve picks BiCGSTAB on a nonsymmetric handle
        b = inputs.rhs_uniform(n, 77)
        xb = torch.empty(n, dtype=torch.float64, device="cuda")
        ig = B.amg_solve(s.h, torch.as_tensor(b).cuda(), xb, 1e-8, 500)
        xo, io = o.solve(b, 1e-8, 500, 1, 1)
        assert ig.status == io.status == 0 and abs(ig.iterations - io.iterations) <= 2
        assert np.linalg.norm(b - Asp @ xb.cpu().numpy()) <= 1e-8 * np.linalg.norm(b)
        # adjoint: A^T lambda = g with B^T (Eq. 1)
        g = inputs.rhs_uniform(n, 78)
        lam, il = s.solve_transpose(g, 1e-8, 500)
        lo, ilo = o.solve_transpose(g, 1e-8, 500, 1, 1, 0)
        assert il.status == ilo.status == 0 and abs(il.iterations - ilo.iterations) <= 2
        assert np.linalg.norm(g - Asp.T @ lam.cpu().numpy()) <= 1e-8 * np.linalg.norm(g)
        # parity near convergence (A12): x, lambda, gA against the oracle's converged results
        xg, _ = s.solve(b, 1e-11, 500, 1)
        lg, _ = s.solve_transpose(g, 1e-11, 500)
        xo, _ = o.solve(b, 1e-13, 500, 1, 1)
        lo, _ = o.solve_transpose(g, 1e-13, 500, 1, 1, 0)
        assert rel(xg.cpu().numpy(), xo) <= 1e-6 and rel(lg.cpu().numpy(), lo) <= 1e-6
        gA = s.grad_values(lg, xg).cpu().numpy()
        assert rel(gA, o.grad_values(lo, xo)) <= 1e-5
        # the adjoint identity g.x = lambda.b (pin P10 (iii)) on the GPU results
        xg_, lg_ = xg.cpu().numpy(), lg.cpu().numpy()
        Ag = np.linalg.norm(g) * np.linalg.norm(xg_)
        xg2, _ = s.solve(b, 1e-11, 500, 1)
        assert abs(g @ xg_ - lg_ @ b) <= 1e-8 * Ag
        assert torch.equal(xg, xg2)  # determinism of the BiCGSTAB path
    finally:
        s.close()
        o.close()


def test_default_options_on_nonsymmetric_matrix_solve_the_transposed_system(oracle_mod, B):
    """with default options a nonsymmetric A must not silently give A lambda = g."""
    A = inputs.stretched_channel_csr((8, 12, 10), 2.0)
    D = A.to_dense()
    assert not np.allclose(D, D.T)
    s = B.AmgSolver(A.rowptr, A.col, A.val)
    g = inputs.rhs_uniform(A.n, 5)
    lam, info = s.solve_transpose(g, 1e-12, 500)
    assert info.status == 0 and s.symmetric == 0
    assert np.allclose(lam.cpu().numpy(), np.linalg.solve(D.T, g), rtol=1e-8, atol=1e-10)
    assert not np.allclose(lam.cpu().numpy(), np.linalg.solve(D, g), rtol=1e-3)
    # the same values flagged symmetric by the caller: the caller's assertion is taken at its word
    s.close()
    # a warm resetup repeats the device check: symmetric values -> nonsymmetric values on one pattern
    S = inputs.poisson_csr((8, 12, 10))
    assert np.array_equal(S.col, A.col)
    s = B.AmgSolver(S.rowptr, S.col, S.val)
    assert s.symmetric == 1
    s.resetup_values(A.val, keep_aggregates=False)
    assert s.symmetric == 0
    lam, info = s.solve_transpose(g, 1e-12, 500)
    assert np.allclose(lam.cpu().numpy(), np.linalg.solve(D.T, g), rtol=1e-8, atol=1e-10)
    s.close()


def test_nonsymmetric_pattern(oracle_mod, B):
    """Structurally nonsymmetric matrix (entries without a transposed partner): the union pattern of
    (A + A^T)/2 and the transpose kernels on rows of unequal length."""
    rng = np.random.default_rng(41)
    A = inputs.poisson_csr((18, 18))
    D = A.to_dense()
    n = A.n
    for _ in range(150):  # one-sided couplings
        i, j = rng.integers(0, n, 2)
        if i != j and D[i, j] == 0.0 and D[j, i] == 0.0:
            D[i, j] = -rng.uniform(0.05, 0.8)
            D[i, i] += 1.0
    import scipy.sparse as sp

    M = sp.csr_matrix(D)
    M.sort_indices()
    rp, cl, vl = M.indptr.astype(np.int32), M.indices.astype(np.int32), M.data.copy()
    o = oracle_mod.Oracle(rp, cl, vl, symmetric=0)
    s = B.AmgSolver(rp, cl, vl)
    try:
        assert s.symmetric == 0 and s.num_levels == o.num_levels
        for l in range(s.num_levels - 1):
            assert np.array_equal(s.aggregates(l).cpu().numpy(), o.aggregates(l))
        g = rng.standard_normal(n)
        lam, il = s.solve_transpose(g, 1e-11, 500)
        lo, ilo = o.solve_transpose(g, 1e-13, 500, 1, 1, 0)
        assert il.status == 0 and rel(lam.cpu().numpy(), lo) <= 1e-6
        assert np.allclose(lam.cpu().numpy(), np.linalg.solve(D.T, g), rtol=1e-7, atol=1e-9)
        for l in range(s.num_levels):
            rows = s.level_info(l)[0]
            x = rng.standard_normal(rows)
            Al = csr_of(*o.level_csr(l))
            assert rel(s.level_op(l, 7, x, None, rows).cpu().numpy(), Al.T @ x) <= 1e-13
    finally:
        s.close()
        o.close()


# ------------------------------------------------------------------------------------------
# GPU twins of the round-2 oracle pins (tests/test_oracle_pins.py holds the matrices and the python
# restatement of O-2; the expected values are numpy's / python's, not the oracle's)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("tail", [2304, 0])
@pytest.mark.parametrize("n", [12, 61, 100])
def test_dense_lu_row_swaps_on_the_device(B, n, tail):
    """k_dense_lu / k_lu_solve* with piv[k] != k (U6, S5): a coarsest operator that needs partial
    pivoting, for A_L and for A_L^T; n = 100 takes the large-matrix solve kernel (> LU_SMALL_MAX)."""
    from test_oracle_pins import _csr_from_dense, _lu_nopivot_solve, _needs_pivoting_matrix

    D = _needs_pivoting_matrix(n, 31 + n)
    rp, cl, vl = _csr_from_dense(D)
    s = B.AmgSolver(rp, cl, vl, coarse_max_rows=n, tail_dense_rows=tail)
    try:
        assert s.num_levels == 1 and s.symmetric == 0
        r = np.random.default_rng(5).standard_normal(n)
        want, want_t = np.linalg.solve(D, r), np.linalg.solve(D.T, r)
        assert rel(s.apply_preconditioner(r).cpu().numpy(), want) <= 1e-9
        assert rel(s.level_op(0, 8, None, r, n).cpu().numpy(), want_t) <= 1e-9
        assert not rel(_lu_nopivot_solve(D, r), want) <= 1e-6  # the swaps matter on this matrix
        x, info = s.solve(r, 1e-8, 5, 1)
        assert info.iterations == 1 and info.status == 0 and rel(x.cpu().numpy(), want) <= 1e-8
        lam, info = s.solve_transpose(r, 1e-8, 5)
        assert info.iterations == 1 and info.status == 0 and rel(lam.cpu().numpy(), want_t) <= 1e-8
    finally:
        s.close()


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_singleton_merge_target_on_the_device(B, seed):
    """k_propose / k_handshake / k_roots against the python-integer restatement of O-2 (A5: a leftover
    vertex joins the matched neighbour with the LARGEST key)."""
    from test_oracle_pins import _csr_from_dense, _random_mesh_matrix, py_aggregate

    D = _random_mesh_matrix(56, seed)
    rp, cl, vl = _csr_from_dense(D)
    salt = 777 + seed
    s = B.AmgSolver(rp, cl, vl, coarse_max_rows=8, hash_seed=salt)
    try:
        _, pa, pnc, choices = py_aggregate(D, 0.25, salt)
        _, wa, _, _ = py_aggregate(D, 0.25, salt, merge="min")
        got = s.aggregates(0).cpu().numpy()
        assert choices >= 1 and not np.array_equal(wa, pa)
        assert np.array_equal(got, pa) and s.level_info(1)[0] == pnc
    finally:
        s.close()


def test_stall_rule_on_the_device(B):
    """A6 on the device: n_{l+1} > 0.8 n_l (strict) ends the coarsening; above 4096 rows it is an error."""
    from test_oracle_pins import _csr_from_dense

    def matrix(npairs, nlone):
        n = 2 * npairs + nlone
        D = np.diag(np.full(n, 4.0))
        for p in range(npairs):
            D[2 * p, 2 * p + 1] = D[2 * p + 1, 2 * p] = -1.0
        for i in range(2 * npairs, n - 1):
            D[i, i + 1] = D[i + 1, i] = 0.5
        return D

    s = B.AmgSolver(*_csr_from_dense(matrix(20, 60)))
    assert s.num_levels == 2 and s.level_info(1)[0] == 80  # 80 = 0.8 * 100 is not a stall; level 1 stalls
    s.close()
    D = matrix(19, 62)
    s = B.AmgSolver(*_csr_from_dense(D))
    assert s.num_levels == 1  # 81 > 80
    r = np.random.default_rng(3).standard_normal(100)
    assert rel(s.apply_preconditioner(r).cpu().numpy(), np.linalg.solve(D, r)) <= 1e-12
    s.close()
    n = 4097
    with pytest.raises(B.AmgError) as e:
        B.AmgSolver(np.arange(n + 1, dtype=np.int32), np.arange(n, dtype=np.int32), np.full(n, 2.0))
    assert e.value.status == 6
    n = 300
    s = B.AmgSolver(np.arange(n + 1, dtype=np.int32), np.arange(n, dtype=np.int32), np.full(n, 2.0))
    assert s.num_levels == 1 and np.allclose(s.apply_preconditioner(np.ones(n)).cpu().numpy(), 0.5)
    s.close()
