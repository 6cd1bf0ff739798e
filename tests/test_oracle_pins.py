"""Pins for the CPU oracle (SURVEY.md §8(c) P1 … P12): the oracle is checked against what the
mathematics and the paper fix — closed forms, invariants, numpy's dense LU, brute force on tiny
inputs, finite differences, the paper's worked examples — never against itself or the CUDA path.
"""
import os

import numpy as np
import pytest

from paper_2606_09001_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_worked_examples.txt")


def golden():
    out = {}
    with open(GOLDEN) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if "=" in line:
                k, v = [s.strip() for s in line.split("=")]
                out[k] = float(v)
    return out


def lap_eig(n, k):
    """Closed form for T_n = tridiag(-1,2,-1): lambda_k, v_k (k = 1..n)."""
    i = np.arange(1, n + 1)
    return 2.0 - 2.0 * np.cos(k * np.pi / (n + 1)), np.sin(i * k * np.pi / (n + 1))


def kron_eig(shape, ks):
    lam, v = 0.0, np.ones(1)
    for n, k in zip(shape, ks):  # shape = (slowest … fastest)
        l1, v1 = lap_eig(n, k)
        lam += l1
        v = np.kron(v, v1)
    return lam, v


def dense(A):
    return A.to_dense()


# ------------------------------------------------------------------------------------------
# P1: generators + SpMV against closed-form eigenpairs, row sums, nnz formula
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape,ks", [((64, 64), (1, 1)), ((64, 64), (64, 3)), ((17, 9), (5, 9)),
                                      ((8, 8, 8), (2, 7, 1)), ((5, 6, 7), (5, 1, 4)), ((33,), (12,))])
def test_p1_spmv_eigenpairs(oracle_mod, shape, ks):
    A = inputs.poisson_csr(shape)
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, aggregates=[])
    lam, v = kron_eig(shape, ks)
    lam_max = 4.0 * len(shape)
    assert np.max(np.abs(o.spmv(0, v) - lam * v)) <= 1e-13 * lam_max


def test_p1_structure():
    for shape in [(64, 64), (17, 9), (8, 8, 8), (5, 6, 7)]:
        A = inputs.poisson_csr(shape)
        d = len(shape)
        n = int(np.prod(shape))
        faces = sum(n // s * (s - 1) for s in shape)
        assert A.nnz == n + 2 * faces
        if len(set(shape)) == 1:
            e = shape[0]
            assert A.nnz == n + 2 * d * e ** (d - 1) * (e - 1)  # SURVEY.md §8 size formula
        rs = np.add.reduceat(A.val, A.rowptr[:-1])
        grid = np.indices(shape)
        interior = np.all([(g > 0) & (g < s - 1) for g, s in zip(grid, shape)], axis=0).reshape(-1)
        assert np.all(rs[interior] == 0.0) and np.all(rs[~interior] > 0.0)
        # ascending unique columns
        for i in range(0, n, max(1, n // 50)):
            c = A.col[A.rowptr[i]:A.rowptr[i + 1]]
            assert np.all(np.diff(c) > 0)
    assert inputs.poisson_csr((128, 128, 128)).nnz == 14581760  # cfg 3


def test_p1_variable_coefficient_generator():
    shape = (6, 5, 7)
    A = inputs.variable_diffusion_csr(shape, seed=7, sigma=2.0, ell=2.0)
    D = dense(A)
    assert np.array_equal(D, D.T)  # same bits for (i,j) and (j,i)
    assert np.all(np.diag(D) > 0) and np.all(D - np.diag(np.diag(D)) <= 0)
    assert np.all(np.linalg.eigvalsh(D) > 0)
    # k == 1 reduces to the Laplacian
    B = inputs._stencil_csr(shape, np.ones(shape))
    P = inputs.poisson_csr(shape)
    assert np.array_equal(B.col, P.col) and np.array_equal(B.val, P.val)
    # symmetric permutation keeps the spectrum and sorted rows
    perm = np.random.default_rng(3).permutation(A.n)
    Ap = inputs.permute_symmetric(A, perm)
    Dp = dense(Ap)
    assert np.array_equal(Dp[np.ix_(perm, perm)], D)
    for i in range(Ap.n):
        assert np.all(np.diff(Ap.col[Ap.rowptr[i]:Ap.rowptr[i + 1]]) > 0)


# ------------------------------------------------------------------------------------------
# P2 / P3: CG recurrences — finite termination, Chebyshev bound
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("m", [1, 2, 3, 4, 5, 6])
def test_p2_cg_finite_termination(oracle_mod, m):
    shape = (12, 10)
    A = inputs.poisson_csr(shape)
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, aggregates=[])
    ks = [(1, 1), (2, 5), (7, 3), (12, 10), (4, 9), (9, 2)][:m]
    lams = [kron_eig(shape, k)[0] for k in ks]
    assert len(set(np.round(lams, 12))) == m
    b = sum((1.0 + 0.3 * t) * kron_eig(shape, k)[1] for t, k in enumerate(ks))
    x, info = o.solve(b, rtol=1e-12, maxit=50, krylov=0, precond=0)
    assert info.status == 0 and info.iterations == m
    if m == 1:
        assert np.allclose(x, b / lams[0], rtol=1e-13, atol=0)
    # one fewer iteration is not enough
    if m > 1:
        _, info2 = o.solve(b, rtol=1e-12, maxit=m - 1, krylov=0, precond=0)
        assert info2.status == 1 and info2.rel_residual > 1e-12


def test_p3_cg_chebyshev_bound(oracle_mod):
    n = 16
    A = inputs.poisson_csr((n, n))
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, aggregates=[])
    D = dense(A)
    kappa = 1.0 / np.tan(np.pi / (2 * (n + 1))) ** 2  # kappa(T_n (+) T_n) = cot^2(pi / (2(n+1)))
    assert np.isclose(np.linalg.cond(D), kappa, rtol=1e-10)
    b = inputs.rhs_uniform(A.n, 11)
    xs = np.linalg.solve(D, b)
    e0 = np.sqrt(xs @ D @ xs)
    q = (np.sqrt(kappa) - 1) / (np.sqrt(kappa) + 1)
    prev = e0
    for k in [1, 2, 5, 10, 20, 40]:
        x, _ = o.solve(b, rtol=1e-300, maxit=k, krylov=0, precond=0)
        ek = np.sqrt((x - xs) @ D @ (x - xs))
        assert ek <= 2 * q**k * e0 * (1 + 1e-10)
        assert ek <= prev * (1 + 1e-12)  # CG minimises the A-norm error: monotone
        prev = ek


# ------------------------------------------------------------------------------------------
# P4: whole solve against numpy's dense LU; exact preconditioner => 1 iteration
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("krylov", [0, 1])
@pytest.mark.parametrize("which", ["poisson2d", "poisson3d", "variable"])
def test_p4_dense_solve(oracle_mod, krylov, which):
    if which == "poisson2d":
        A = inputs.poisson_csr((16, 15))
    elif which == "poisson3d":
        A = inputs.poisson_csr((6, 6, 7))
    else:
        A = inputs.variable_diffusion_csr((6, 6, 6), seed=5, sigma=2.0, ell=2.0)
        A = inputs.permute_symmetric(A, np.random.default_rng(6).permutation(A.n))
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, coarse_max_rows=8)
    assert o.num_levels >= 4
    b = inputs.rhs_uniform(A.n, 21)
    xs = np.linalg.solve(dense(A), b)
    x, info = o.solve(b, rtol=1e-12, maxit=200, krylov=krylov, precond=1)
    assert info.status == 0
    assert np.linalg.norm(x - xs) / np.linalg.norm(xs) <= 1e-9


@pytest.mark.parametrize("krylov", [0, 1])
def test_p4_exact_preconditioner_one_iteration(oracle_mod, krylov):
    A = inputs.poisson_csr((9, 11))
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, coarse_max_rows=A.n)
    assert o.num_levels == 1
    b = inputs.rhs_uniform(A.n, 22)
    x, info = o.solve(b, rtol=1e-10, maxit=10, krylov=krylov, precond=1)
    assert info.iterations == 1 and info.status == 0
    assert np.allclose(x, np.linalg.solve(dense(A), b), rtol=1e-11, atol=1e-13)


# ------------------------------------------------------------------------------------------
# P5: Galerkin RAP
# ------------------------------------------------------------------------------------------
def test_p5_galerkin_1d_closed_form(oracle_mod):
    n = 40
    A = inputs.poisson_csr((n,))
    agg = np.arange(n) // 2
    rp, cl, vl = oracle_mod.galerkin(A.rowptr, A.col, A.val, agg, n // 2)
    T = inputs.poisson_csr((n // 2,))  # pairs {2I, 2I+1} of T_n give exactly T_{n/2}
    assert np.array_equal(rp, T.rowptr) and np.array_equal(cl, T.col) and np.array_equal(vl, T.val)


def test_p5_galerkin_2d_x_pairs(oracle_mod):
    ny, nx = 6, 8
    A = inputs.poisson_csr((ny, nx))
    i = np.arange(ny * nx)
    agg = (i // nx) * (nx // 2) + (i % nx) // 2
    rp, cl, vl = oracle_mod.galerkin(A.rowptr, A.col, A.val, agg, ny * nx // 2)
    C = inputs.Csr(ny * nx // 2, rp, cl, vl).to_dense()
    cx = nx // 2
    for I in range(C.shape[0]):
        y, x = divmod(I, cx)
        assert C[I, I] == 6.0  # 4+4-1-1
        if x > 0:
            assert C[I, I - 1] == -1.0
        if x < cx - 1:
            assert C[I, I + 1] == -1.0
        if y > 0:
            assert C[I, I - cx] == -2.0
        if y < ny - 1:
            assert C[I, I + cx] == -2.0
    assert np.count_nonzero(C) == len(vl)


@pytest.mark.parametrize("which", ["poisson", "variable"])
def test_p5_galerkin_invariants_and_dense(oracle_mod, which):
    if which == "poisson":
        A = inputs.poisson_csr((10, 9))
    else:
        A = inputs.variable_diffusion_csr((5, 5, 6), seed=9, sigma=2.0, ell=2.0)
    rng = np.random.default_rng(31)
    nc = A.n // 3
    agg = rng.integers(0, nc, A.n).astype(np.int32)
    agg[:nc] = np.arange(nc)  # every coarse id used
    rp, cl, vl = oracle_mod.galerkin(A.rowptr, A.col, A.val, agg, nc)
    C = inputs.Csr(nc, rp, cl, vl).to_dense()
    P = np.zeros((A.n, nc))
    P[np.arange(A.n), agg] = 1.0
    D = dense(A)
    ref = P.T @ D @ P
    assert np.allclose(C, ref, rtol=1e-13, atol=1e-13 * np.abs(D).max())
    # pattern is structurally symmetric, values symmetric to rounding, diagonal > 0, sums kept
    assert np.array_equal(C != 0, (C != 0).T) or which == "poisson"
    assert np.allclose(C, C.T, rtol=0, atol=1e-15 * np.abs(D).max() * 50)
    assert np.all(np.diag(C) > 0)
    assert np.allclose(C.sum(axis=1), P.T @ D.sum(axis=1), atol=1e-12 * np.abs(D).max())
    assert np.isclose(C.sum(), D.sum(), atol=1e-11 * np.abs(D).max())
    for I in range(nc):
        assert np.all(np.diff(cl[rp[I]:rp[I + 1]]) > 0)


# ------------------------------------------------------------------------------------------
# P6: the V-cycle operator B is symmetric positive definite, spec(BA) in (0, 1]
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("smoother", [0, 1])
def test_p6_vcycle_operator(oracle_mod, smoother):
    A = inputs.poisson_csr((12, 12))
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, coarse_max_rows=8, smoother=smoother)
    assert o.num_levels >= 4
    B = np.column_stack([o.vcycle(e) for e in np.eye(A.n)])
    assert np.linalg.norm(B - B.T) / np.linalg.norm(B) <= 1e-14
    Bs = 0.5 * (B + B.T)
    assert np.linalg.eigvalsh(Bs).min() > 0
    D = dense(A)
    ev = np.linalg.eigvals(Bs @ D).real
    if smoother == 0:  # L1-Jacobi: D_l1 - A is PSD on every level => I - BA is PSD in the A-inner product
        assert ev.min() > 0 and ev.max() <= 1 + 1e-12
    kappa = ev.max() / ev.min()
    # P3 with kappa(BA): PCG iteration count consistent with the bound
    b = inputs.rhs_uniform(A.n, 41)
    xs = np.linalg.solve(D, b)
    e0 = np.sqrt(xs @ D @ xs)
    q = (np.sqrt(kappa) - 1) / (np.sqrt(kappa) + 1)
    for k in [1, 3, 6, 10]:
        x, _ = o.solve(b, rtol=1e-300, maxit=k, krylov=0, precond=1)
        ek = np.sqrt((x - xs) @ D @ (x - xs))
        assert ek <= 2 * q**k * e0 * (1 + 1e-9)


# ------------------------------------------------------------------------------------------
# P7: smoother
# ------------------------------------------------------------------------------------------
def test_p7_damped_jacobi_eigenvector_factor(oracle_mod):
    shape = (7, 9)
    A = inputs.poisson_csr(shape)
    omega = 2.0 / 3.0
    agg = (np.arange(A.n) // 2).astype(np.int32)
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, aggregates=[agg], smoother=1, omega=omega)
    assert np.allclose(o.dinv(0), omega / 4.0, rtol=1e-15)
    for ks in [(1, 1), (3, 5), (7, 9)]:
        lam, v = kron_eig(shape, ks)
        # b = 0: the error e = x - 0 is multiplied by 1 - omega lam / (2d) exactly
        out = o.smooth(0, np.zeros(A.n), v)
        assert np.allclose(out, (1 - omega * lam / 4.0) * v, rtol=0, atol=1e-14)


def test_p7_l1_jacobi(oracle_mod):
    A = inputs.poisson_csr((6, 6, 6))
    agg = (np.arange(A.n) // 2).astype(np.int32)
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, aggregates=[agg], smoother=0)
    dinv = o.dinv(0)
    grid = np.indices((6, 6, 6))
    interior = np.all([(g > 0) & (g < 5) for g in grid], axis=0).reshape(-1)
    assert np.all(dinv[interior] == 1.0 / 12.0)  # interior 7-point row: d_l1 = 4d = 12
    D = dense(A)
    assert np.linalg.eigvalsh(np.diag(1.0 / dinv) - D).min() >= -1e-12  # D_l1 - A is PSD
    rng = np.random.default_rng(5)
    b = rng.standard_normal(A.n)
    xs = np.linalg.solve(D, b)
    x = rng.standard_normal(A.n)
    en = lambda y: np.sqrt((y - xs) @ D @ (y - xs))
    for _ in range(5):
        xn = o.smooth(0, b, x)
        assert np.allclose(xn, x + dinv * (b - D @ x), rtol=1e-13, atol=1e-13)
        assert en(xn) <= en(x) * (1 + 1e-12)  # A-norm of the error never increases
        x = xn


def test_p7_residual_restrict_and_vcycle_structure(oracle_mod):
    """rc = P^T (b - A x) by dense algebra; a two-level cycle equals its textbook matrix form."""
    A = inputs.variable_diffusion_csr((5, 6, 5), seed=2, sigma=1.0, ell=2.0)
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, coarse_max_rows=100)
    assert o.num_levels == 2
    agg = o.aggregates(0)
    nc = o.level_info(1)[0]
    P = np.zeros((A.n, nc))
    P[np.arange(A.n), agg] = 1.0
    D = dense(A)
    rng = np.random.default_rng(8)
    b, x = rng.standard_normal(A.n), rng.standard_normal(A.n)
    assert np.allclose(o.residual_restrict(0, b, x), P.T @ (b - D @ x), rtol=1e-12, atol=1e-12)
    # V(2,2) two-grid in matrix form: S = I - Dinv A
    Dinv = np.diag(o.dinv(0))
    Ac = P.T @ D @ P
    x1 = Dinv @ b
    x2 = x1 + Dinv @ (b - D @ x1)
    x3 = x2 + P @ np.linalg.solve(Ac, P.T @ (b - D @ x2))
    x4 = x3 + Dinv @ (b - D @ x3)
    x5 = x4 + Dinv @ (b - D @ x4)
    assert np.allclose(o.vcycle(b), x5, rtol=1e-11, atol=1e-12)


# ------------------------------------------------------------------------------------------
# P8: aggregation — structural invariants, handshake == greedy, maximality, ratio
# ------------------------------------------------------------------------------------------
def _candidates(A, beta=0.25):
    """Brute-force candidate edge set from the definition (dense)."""
    D = dense(A)
    W = -(D - np.diag(np.diag(D)))
    m = np.maximum(W, 0).max(axis=1)
    return (W > 0) & (W >= beta * np.minimum.outer(m, m))


@pytest.mark.parametrize("which", ["poisson2d", "poisson3d", "variable", "varperm"])
def test_p8_aggregation(oracle_mod, which):
    if which == "poisson2d":
        A = inputs.poisson_csr((24, 24))
    elif which == "poisson3d":
        A = inputs.poisson_csr((9, 8, 7))
    else:
        A = inputs.variable_diffusion_csr((12, 12, 12) if which == "variable" else (8, 9, 10),
                                          seed=17, sigma=2.0, ell=3.0)
        if which == "varperm":
            A = inputs.permute_symmetric(A, np.random.default_rng(18).permutation(A.n))
    n = A.n
    for salt in (0, 5):
        match, agg, nc, rounds = oracle_mod.aggregate(A.rowptr, A.col, A.val, 0.25, salt, 0, 0)
        match_g, agg_g, nc_g, _ = oracle_mod.aggregate(A.rowptr, A.col, A.val, 0.25, salt, 0, 1)
        assert np.array_equal(match, match_g) and np.array_equal(agg, agg_g) and nc == nc_g
        assert rounds <= 12
        cand = _candidates(A)
        matched = match >= 0
        idx = np.arange(n)
        assert np.array_equal(match[match[matched]], idx[matched])  # involution
        assert np.all(cand[idx[matched], match[matched]])  # matched pairs are candidate edges
        # maximality: no candidate edge joins two unmatched vertices
        um = ~matched
        assert not np.any(cand[np.ix_(um, um)])
        # ids contiguous and increasing with the root index (root = smaller index of the matched
        # pair, or the vertex itself for an aggregate without a pair; merged singletons do not count)
        assert set(agg.tolist()) == set(range(nc))
        root = np.full(nc, n)
        np.minimum.at(root, agg[matched], idx[matched])
        lone = root == n
        first = np.full(nc, n)
        np.minimum.at(first, agg, idx)
        root[lone] = first[lone]
        assert np.all(np.diff(root) > 0)
        # matched pairs share an aggregate; singletons merged only along candidate edges to matched vertices
        assert np.all(agg[matched] == agg[match[matched]])
        sizes = np.bincount(agg)
        for i in idx[um]:
            if cand[i, matched].any():
                assert sizes[agg[i]] >= 3
            else:
                assert sizes[agg[i]] == 1
        assert 1.8 <= n / nc <= 2.6


def test_p8_key_order_bruteforce(oracle_mod):
    """First handshake round on a tiny graph, re-derived with python integers from the
    definition of key(i,j) (A3, A4): every vertex points to its arg-max key neighbour."""
    A = inputs.variable_diffusion_csr((4, 4, 3), seed=4, sigma=2.0, ell=2.0)
    D = dense(A)
    n = A.n
    W = -(D - np.diag(np.diag(D)))
    m = np.maximum(W, 0).max(axis=1)
    cand = _candidates(A)
    M64 = (1 << 64) - 1

    def mix64(z):
        z ^= z >> 30
        z = (z * 0xBF58476D1CE4E5B9) & M64
        z ^= z >> 27
        z = (z * 0x94D049BB133111EB) & M64
        z ^= z >> 31
        return z

    salt = 12345
    def key(i, j):
        lo, hi = min(i, j), max(i, j)
        M = max(m[i], m[j])
        q = 0 if 2 * W[i, j] > M else (1 if 4 * W[i, j] > M else 2)
        h = mix64((lo * 0x9E3779B97F4A7C15 + hi * 0xBF58476D1CE4E5B9 + salt) & M64)
        return (-q, h, -lo, -hi)

    ptr = [max((j for j in range(n) if cand[i, j]), key=lambda j: key(i, j), default=-1) for i in range(n)]
    expect = np.array([ptr[i] if ptr[i] >= 0 and ptr[ptr[i]] == i else -1 for i in range(n)])
    match, _, _, rounds = oracle_mod.aggregate(A.rowptr, A.col, A.val, 0.25, salt, 1, 0)
    assert rounds == 1 and np.array_equal(match, expect)
    assert (expect >= 0).sum() >= 4


# ------------------------------------------------------------------------------------------
# P9: manufactured solution (cfg 2 recipe at reduced size); A12: 1e-8 is not enough for 1e-6
# ------------------------------------------------------------------------------------------
def test_p9_manufactured_solution(oracle_mod):
    A = inputs.config_matrix(2, edge=96)
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val)
    xt = inputs.config_rhs(2, A.n, 0)
    b = A.to_scipy() @ xt
    x, info = o.solve(b, rtol=1e-11, maxit=500)
    assert info.status == 0
    assert np.linalg.norm(x - xt) / np.linalg.norm(xt) <= 1e-6
    r = b - A.to_scipy() @ x
    assert np.linalg.norm(r) / np.linalg.norm(b) <= 1.05e-11


# ------------------------------------------------------------------------------------------
# P10: adjoint + gradient
# ------------------------------------------------------------------------------------------
def test_p10_gradient_finite_differences(oracle_mod):
    A = inputs.variable_diffusion_csr((4, 4, 4), seed=3, sigma=1.0, ell=2.0)
    n = A.n
    D = dense(A)
    rng = np.random.default_rng(77)
    b = rng.standard_normal(n)
    xt = rng.standard_normal(n)
    loss = lambda Dm, bv: 0.5 * np.sum((np.linalg.solve(Dm, bv) - xt) ** 2)
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, coarse_max_rows=8)
    x, i1 = o.solve(b, rtol=1e-13, maxit=300)
    lam, i2 = o.solve_transpose(x - xt, rtol=1e-13, maxit=300)
    assert i1.status == 0 and i2.status == 0
    gA = o.grad_values(lam, x)
    rows = np.repeat(np.arange(n), np.diff(A.rowptr))
    h = 1e-5
    ks = rng.choice(A.nnz, 60, replace=False)
    fd = np.empty(len(ks))
    for t, k in enumerate(ks):
        i, j = rows[k], A.col[k]
        Dp, Dm = D.copy(), D.copy()
        Dp[i, j] += h  # each stored entry is an independent parameter (no symmetrisation)
        Dm[i, j] -= h
        fd[t] = (loss(Dp, b) - loss(Dm, b)) / (2 * h)
    # FD noise is ~eps*loss/h ~ 4e-10 absolute here; a wrong sign / index / transposed operand is O(|gA|)
    assert np.linalg.norm(gA[ks] - fd) / np.linalg.norm(fd) <= 1e-7
    assert np.max(np.abs(gA[ks] - fd)) <= 1e-8 * np.abs(gA).max()
    ii = rng.choice(n, 12, replace=False)
    fdb = np.empty(len(ii))
    for t, i in enumerate(ii):
        bp, bm = b.copy(), b.copy()
        bp[i] += h
        bm[i] -= h
        fdb[t] = (loss(D, bp) - loss(D, bm)) / (2 * h)
    assert np.linalg.norm(lam[ii] - fdb) / np.linalg.norm(fdb) <= 1e-7
    # asymmetric pattern entries differ: gA[(i,j)] != gA[(j,i)] in general (not symmetrised)
    assert not np.allclose(gA, inputs.Csr(n, A.rowptr, A.col, gA).to_dense().T[rows, A.col])
    # identity g^T x = lam^T b for A x = b, A^T lam = g
    g = x - xt
    assert abs(g @ x - lam @ b) <= 1e-8 * np.linalg.norm(g) * np.linalg.norm(x)
    # batch of right-hand sides: cotangents add (A17); accumulate flag
    x2, _ = o.solve(2 * b, rtol=1e-13, maxit=300)
    lam2, _ = o.solve_transpose(x2 - xt, rtol=1e-13, maxit=300)
    gb = o.grad_values(np.stack([lam, lam2]), np.stack([x, x2]))
    assert np.allclose(gb, gA + o.grad_values(lam2, x2), rtol=1e-13, atol=1e-15)
    acc = o.grad_values(lam2, x2, accumulate_into=gA.copy())
    assert np.allclose(acc, gb, rtol=1e-13, atol=1e-15)


def test_p10_symmetric_transpose_is_solve_bitwise(oracle_mod):
    A = inputs.poisson_csr((20, 20))
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val)
    g = inputs.rhs_uniform(A.n, 5)
    for krylov in (0, 1):
        x, i1 = o.solve(g, krylov=krylov)
        lam, i2 = o.solve_transpose(g, krylov=krylov, symmetric=1)
        assert np.array_equal(x, lam) and i1.iterations == i2.iterations


def test_p10_nonsymmetric_adjoint(oracle_mod):
    """A = D^-1 S (row-scaled SPD: nonsymmetric values, symmetric pattern): transposed
    hierarchy solves A^T lam = g; (P^T A P)^T = P^T A^T P."""
    S = inputs.variable_diffusion_csr((5, 5, 5), seed=12, sigma=1.0, ell=2.0)
    n = S.n
    rng = np.random.default_rng(13)
    scale = rng.uniform(0.5, 2.0, n)
    rows = np.repeat(np.arange(n), np.diff(S.rowptr))
    val = S.val * scale[rows]
    o = oracle_mod.Oracle(S.rowptr, S.col, val, coarse_max_rows=8)
    D = inputs.Csr(n, S.rowptr, S.col, val).to_dense()
    assert not np.allclose(D, D.T)
    g = rng.standard_normal(n)
    lam, info = o.solve_transpose(g, rtol=1e-12, maxit=300, krylov=1, symmetric=0)
    assert info.status == 0
    assert np.allclose(lam, np.linalg.solve(D.T, g), rtol=1e-8, atol=1e-10)
    b = rng.standard_normal(n)
    x, info = o.solve(b, rtol=1e-12, maxit=300, krylov=1)
    assert np.allclose(x, np.linalg.solve(D, b), rtol=1e-8, atol=1e-10)
    assert abs(g @ x - lam @ b) <= 1e-8 * np.linalg.norm(g) * np.linalg.norm(x)


def test_p10_paper_inverse_problem(oracle_mod):
    """PAPER.md:154-186 §3.2: recover d = 4 from d = 10 by gradient descent through the solve.
    dL/dd = sum_i gA[diag_i];  loss = sum((x - x_target)^2) WITHOUT 1/2 (A20)."""
    G = golden()
    n, d_true, d, lr = int(G["s3_2.n"]), G["s3_2.true_diag"], G["s3_2.init_diag"], G["s3_2.lr"]
    b = inputs.rhs_ones(n)
    At = inputs.tridiagonal_csr(n, d_true)
    x_target = np.linalg.solve(dense(At), b)
    rows = np.repeat(np.arange(n), np.diff(At.rowptr))
    is_diag = At.col == rows
    steps, first_grad = None, None
    for step in range(int(G["s3_2.max_iters"])):
        A = inputs.tridiagonal_csr(n, d)
        o = oracle_mod.Oracle(A.rowptr, A.col, A.val, coarse_max_rows=8)
        x, i1 = o.solve(b, rtol=1e-13, maxit=200, krylov=1)
        lam, i2 = o.solve_transpose(2.0 * (x - x_target), rtol=1e-13, maxit=200, krylov=1)
        assert i1.status == 0 and i2.status == 0
        grad = o.grad_values(lam, x)[is_diag].sum()
        if first_grad is None:
            first_grad = grad
            f = lambda dd: np.sum((np.linalg.solve(dense(inputs.tridiagonal_csr(n, dd)), b) - x_target) ** 2)
            fd = (f(d + 1e-5) - f(d - 1e-5)) / 2e-5
            assert abs(grad - fd) <= 1e-8 * abs(fd)
        d -= lr * grad
        if abs(grad) < G["s3_2.tol"]:
            steps = step + 1
            break
    assert steps is not None and abs(d - d_true) < 1e-3  # hard pin: converges to 4.0 within 200
    assert abs(first_grad - 0.36086585929) < 1e-9        # SURVEY.md P10(ii), equal to central FD
    assert steps <= int(G["s3_2.steps_upper_soft"]) + 10  # soft: paper "fewer than 100"; exact solves 107


# ------------------------------------------------------------------------------------------
# P11: BiCGSTAB — the paper's §3.1 example, B = I PCG == CG
# ------------------------------------------------------------------------------------------
def test_p11_paper_poisson32_bicgstab(oracle_mod):
    G = golden()
    n = int(G["s3_1.grid"])
    A = inputs.poisson_csr((n, n))
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val)
    b = inputs.rhs_ones(A.n)
    x, info = o.solve(b, rtol=G["s3_1.tolerance"], maxit=500, krylov=1, precond=0)
    paper = int(G["s3_1.iterations_unpreconditioned"])
    assert info.status == 0 and paper - 3 <= info.iterations <= paper + 5  # soft pin 34..42
    xs = np.linalg.solve(dense(A), b)
    assert np.linalg.norm(x - xs) / np.linalg.norm(xs) <= 1e-5
    # with the AMG preconditioner far fewer iterations (paper: 6 with AmgX's AMG — context only)
    x, info_p = o.solve(b, rtol=G["s3_1.tolerance"], maxit=500, krylov=1, precond=1)
    assert info_p.status == 0 and info_p.iterations <= 15 < info.iterations
    assert np.linalg.norm(x - xs) / np.linalg.norm(xs) <= 1e-5


def test_p11_half_step_and_breakdown(oracle_mod):
    A = inputs.poisson_csr((7, 7))
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, coarse_max_rows=A.n)
    b = inputs.rhs_uniform(A.n, 2)
    x, info = o.solve(b, rtol=1e-10, maxit=5, krylov=1)  # exact B => s = 0 at the half step
    assert info.iterations == 1 and info.status == 0
    x, info = o.solve(np.zeros(A.n), krylov=1)
    assert info.iterations == 0 and info.status == 0 and np.all(x == 0)
    x, info = o.solve(np.zeros(A.n), krylov=0)
    assert info.iterations == 0 and info.status == 0 and np.all(x == 0)
    _, info = o.solve(b, rtol=1e-30, maxit=3, krylov=0, precond=0)
    assert info.status == 1 and info.iterations == 3


# ------------------------------------------------------------------------------------------
# P12: determinism; thread count does not change results
# ------------------------------------------------------------------------------------------
def test_p12_determinism(oracle_mod):
    A = inputs.config_matrix(3, edge=30)
    b = inputs.config_rhs(3, A.n)
    res = []
    for threads in (1, 1, 4):
        oracle_mod.set_threads(threads)
        o = oracle_mod.Oracle(A.rowptr, A.col, A.val)
        x, info = o.solve(b)
        res.append((x, info.iterations, [o.aggregates(l) for l in range(o.num_levels - 1)]))
    oracle_mod.set_threads(1)
    for r in res[1:]:
        assert np.array_equal(r[0], res[0][0]) and r[1] == res[0][1]
        assert all(np.array_equal(a, b_) for a, b_ in zip(r[2], res[0][2]))


def test_setup_rules(oracle_mod):
    """O-1: coarsest <= coarse_max_rows, max_levels, imported aggregates, bad CSR rejected."""
    A = inputs.config_matrix(1)
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val)
    L = o.num_levels
    assert o.level_info(L - 1)[0] <= 64 < o.level_info(L - 2)[0]
    o3 = oracle_mod.Oracle(A.rowptr, A.col, A.val, max_levels=3)
    assert o3.num_levels == 3
    aggs = [o.aggregates(l) for l in range(2)]
    oi = oracle_mod.Oracle(A.rowptr, A.col, A.val, aggregates=aggs)
    assert oi.num_levels == 3
    for l in range(3):
        for a, b_ in zip(oi.level_csr(l), o.level_csr(l)):
            assert np.array_equal(a, b_)
    bad = A.val.copy()
    bad[A.col == np.repeat(np.arange(A.n), np.diff(A.rowptr))] = -1.0
    with pytest.raises(RuntimeError):
        oracle_mod.Oracle(A.rowptr, A.col, bad)
    # salt changes the matching (A4) but not its quality
    o5 = oracle_mod.Oracle(A.rowptr, A.col, A.val, hash_seed=99)
    assert not np.array_equal(o5.aggregates(0), o.aggregates(0))
    assert abs(o5.level_info(1)[0] - o.level_info(1)[0]) < 0.05 * o.level_info(1)[0]


# ------------------------------------------------------------------------------------------
# Round-2 pins of branches no earlier pin exercised: LU row swaps, the singleton-merge target (A5),
# the stall rule (A6); then the readings added in round 2 (nonsymmetric strength A1, agg_passes,
# residual history)
# ------------------------------------------------------------------------------------------
def _csr_from_dense(D):
    import scipy.sparse as sp

    S = sp.csr_matrix(D)
    S.sort_indices()
    return S.indptr.astype(np.int32), S.indices.astype(np.int32), S.data.astype(np.float64)


def _needs_pivoting_matrix(n, seed):
    """Dense nonsymmetric matrix with a tiny positive diagonal and O(1) off-diagonals: LU without row
    exchanges loses every digit (pivots ~1e-13), partial pivoting swaps in almost every column."""
    rng = np.random.default_rng(seed)
    D = rng.uniform(-1.0, 1.0, (n, n))
    D[np.abs(D) < 0.05] = 0.05
    np.fill_diagonal(D, 1e-13 * rng.uniform(1.0, 2.0, n))
    return D


def _lu_nopivot_solve(D, b):
    a = D.copy()
    n = len(b)
    x = b.copy()
    for k in range(n):
        for i in range(k + 1, n):
            l = a[i, k] / a[k, k]
            a[i, k:] -= l * a[k, k:]
            x[i] -= l * x[k]
    for i in range(n - 1, -1, -1):
        x[i] = (x[i] - a[i, i + 1:] @ x[i + 1:]) / a[i, i]
    return x


@pytest.mark.parametrize("n", [12, 61])
def test_dense_lu_row_swaps(oracle_mod, n):
    """S5/U6 with piv[k] != k: a coarsest operator that NEEDS partial pivoting (every earlier case was
    SPD and diagonally dominant, so the row-swap branch of dense_lu / dense_lu_solve never ran).
    coarse_max_rows >= n makes the V-cycle the LU solve alone: compare with numpy.linalg.solve."""
    D = _needs_pivoting_matrix(n, 31 + n)
    rp, cl, vl = _csr_from_dense(D)
    o = oracle_mod.Oracle(rp, cl, vl, coarse_max_rows=n)
    assert o.num_levels == 1
    rng = np.random.default_rng(5)
    r = rng.standard_normal(n)
    want = np.linalg.solve(D, r)
    z = o.vcycle(r)
    assert np.linalg.norm(z - want) <= 1e-10 * np.linalg.norm(want)
    # the case really exercises the swaps: the same elimination without them is useless here
    bad = _lu_nopivot_solve(D, r)
    assert not np.linalg.norm(bad - want) <= 1e-6 * np.linalg.norm(want)
    # the exact preconditioner gives one Krylov iteration, also for the transposed factors (O-7)
    x, info = o.solve(r, rtol=1e-9, maxit=5, krylov=1)
    assert info.iterations == 1 and info.status == 0 and np.linalg.norm(x - want) <= 1e-9 * np.linalg.norm(want)
    lam, info = o.solve_transpose(r, rtol=1e-9, maxit=5, krylov=1, symmetric=0)
    want_t = np.linalg.solve(D.T, r)
    assert info.iterations == 1 and np.linalg.norm(lam - want_t) <= 1e-9 * np.linalg.norm(want_t)


_M64 = (1 << 64) - 1


def _py_mix64(z):
    z ^= z >> 30
    z = (z * 0xBF58476D1CE4E5B9) & _M64
    z ^= z >> 27
    z = (z * 0x94D049BB133111EB) & _M64
    z ^= z >> 31
    return z


def py_aggregate(D, beta, salt, merge="max"):
    """O-2 from its definition with python integers / floats on a dense matrix: handshake rounds to the
    fix-point, singleton merge into the matched neighbour with the LARGEST key (A5), numbering by
    ascending root.  merge="min" is the plausible mistake the pin has to catch."""
    n = D.shape[0]
    W = -(D - np.diag(np.diag(D)))
    m = np.maximum(W, 0).max(axis=1)
    cand = (W > 0) & (W >= beta * np.minimum.outer(m, m))

    def key(i, j):
        lo, hi = min(i, j), max(i, j)
        M = max(m[i], m[j])
        q = 0 if 2 * W[i, j] > M else (1 if 4 * W[i, j] > M else 2)
        return (-q, _py_mix64((lo * 0x9E3779B97F4A7C15 + hi * 0xBF58476D1CE4E5B9 + salt) & _M64), -lo, -hi)

    match = [-1] * n
    while True:
        ptr = [-1] * n
        for i in range(n):
            if match[i] < 0:
                nb = [j for j in range(n) if cand[i, j] and match[j] < 0]
                if nb:
                    ptr[i] = max(nb, key=lambda j: key(i, j))
        added = 0
        for i in range(n):
            if ptr[i] >= 0 and ptr[ptr[i]] == i:
                match[i] = ptr[i]
                added += 1
        if not added:
            break
    root = [min(i, match[i]) if match[i] >= 0 else i for i in range(n)]
    root2 = list(root)
    choices = 0  # singletons whose matched candidate neighbours sit in more than one aggregate
    for i in range(n):
        if match[i] < 0:
            nb = [j for j in range(n) if cand[i, j] and match[j] >= 0]
            if nb:
                pick = max if merge == "max" else min
                root2[i] = root[pick(nb, key=lambda j: key(i, j))]
                choices += len({root[j] for j in nb}) > 1
    ids = {r: t for t, r in enumerate(sorted(set(root2)))}
    return np.array(match), np.array([ids[r] for r in root2]), len(ids), choices


def _random_mesh_matrix(n, seed, k=4):
    """SPD M-matrix of a random planar-ish point cloud (k nearest neighbours, weights over two decades)."""
    rng = np.random.default_rng(seed)
    pts = rng.uniform(0, 1, (n, 2))
    d2 = ((pts[:, None, :] - pts[None, :, :]) ** 2).sum(-1)
    W = np.zeros((n, n))
    for i in range(n):
        for j in np.argsort(d2[i])[1:k + 1]:
            w = 10.0 ** rng.uniform(-1.0, 1.0)
            W[i, j] = W[j, i] = max(W[i, j], w)
    return np.diag(W.sum(axis=1) + 0.1) - W


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_p8_whole_aggregation_bruteforce(oracle_mod, seed):
    """The WHOLE of O-2 on a 56-vertex graph against python integers: matching to the fix-point, and
    which matched neighbour a leftover vertex joins (A5: the one with the largest key)."""
    D = _random_mesh_matrix(56, seed)
    rp, cl, vl = _csr_from_dense(D)
    salt = 777 + seed
    match, agg, nc, _ = oracle_mod.aggregate(rp, cl, vl, 0.25, salt, 0, 0)
    pm, pa, pnc, choices = py_aggregate(D, 0.25, salt)
    assert np.array_equal(match, pm) and np.array_equal(agg, pa) and nc == pnc
    wm, wa, _, _ = py_aggregate(D, 0.25, salt, merge="min")
    assert choices >= 1 and not np.array_equal(wa, pa)  # the case can tell "largest" from "smallest"


def test_stall_rule_and_coarsen_stall(oracle_mod):
    """A6: n_{l+1} > 0.8 n_l  =>  level l is the coarsest (strict, factor 0.8); n_L > 4096 => error."""
    def matrix(npairs, nlone):
        # npairs strongly coupled pairs + nlone rows without any negative off-diagonal (never candidates)
        n = 2 * npairs + nlone
        D = np.diag(np.full(n, 4.0))
        for p in range(npairs):
            D[2 * p, 2 * p + 1] = D[2 * p + 1, 2 * p] = -1.0
        for i in range(2 * npairs, n - 1):  # positive couplings keep the lone rows connected but weak (A1)
            D[i, i + 1] = D[i + 1, i] = 0.5
        return D

    # 100 rows: 20 pairs + 60 lone -> n_c = 80 = 0.8 n: NOT a stall (strict inequality): one coarse level
    rp, cl, vl = _csr_from_dense(matrix(20, 60))
    o = oracle_mod.Oracle(rp, cl, vl)
    assert o.level_info(0)[0] == 100 and o.num_levels >= 2 and o.level_info(1)[0] == 80
    # 19 pairs + 62 lone -> n_c = 81 > 80: stall, level 0 is the coarsest and is solved densely
    D = matrix(19, 62)
    rp, cl, vl = _csr_from_dense(D)
    o = oracle_mod.Oracle(rp, cl, vl)
    assert o.num_levels == 1
    r = np.random.default_rng(3).standard_normal(100)
    assert np.allclose(o.vcycle(r), np.linalg.solve(D, r), rtol=1e-12, atol=1e-14)
    x, info = o.solve(r, rtol=1e-10, maxit=5)
    assert info.iterations == 1 and info.status == 0
    # the second level of the first matrix stalls (80 rows > 64, no candidates left but the lone chain)
    o = oracle_mod.Oracle(*_csr_from_dense(matrix(20, 60)))
    assert o.num_levels == 2
    # a stalled coarsest level above 4096 rows is an error (O-1), at 4096 + 1 exactly
    n = 4097
    rp = np.arange(n + 1, dtype=np.int32)
    with pytest.raises(RuntimeError, match="-4"):
        oracle_mod.Oracle(rp, np.arange(n, dtype=np.int32), np.full(n, 2.0))
    n = 300  # ... and fine below
    o = oracle_mod.Oracle(np.arange(n + 1, dtype=np.int32), np.arange(n, dtype=np.int32), np.full(n, 2.0))
    assert o.num_levels == 1 and np.allclose(o.vcycle(np.ones(n)), 0.5)


def _row_scaled(S, seed):
    """A = diag(s) S: nonsymmetric values on a symmetric pattern (the pressure-Poisson-like D^-1 S form)."""
    n = S.n
    scale = np.random.default_rng(seed).uniform(0.5, 2.0, n)
    rows = np.repeat(np.arange(n), np.diff(S.rowptr))
    return inputs.Csr(n, S.rowptr, S.col, S.val * scale[rows])


def _transpose_csr(A):
    T = A.to_scipy().T.tocsr()
    T.sort_indices()
    return inputs.Csr(A.n, T.indptr.astype(np.int32), T.indices.astype(np.int32), T.data.astype(np.float64))


def test_nonsymmetric_strength(oracle_mod):
    """A1, nonsymmetric case: the matching runs on (A + A^T)/2.  Pins: bitwise no-op on a bitwise
    symmetric matrix; A and A^T get the SAME aggregates; handshake == greedy still holds (the key is
    symmetric again); structurally nonsymmetric patterns (union pattern) work."""
    S = inputs.variable_diffusion_csr((7, 6, 5), seed=21, sigma=1.5, ell=2.0)
    a1 = oracle_mod.aggregate(S.rowptr, S.col, S.val, 0.25, 3, 0, 0, symmetric=1)
    a0 = oracle_mod.aggregate(S.rowptr, S.col, S.val, 0.25, 3, 0, 0, symmetric=0)
    assert np.array_equal(a1[0], a0[0]) and np.array_equal(a1[1], a0[1])
    A = _row_scaled(S, 22)
    At = _transpose_csr(A)
    m, agg, nc, _ = oracle_mod.aggregate(A.rowptr, A.col, A.val, 0.25, 3, 0, 0, symmetric=0)
    mt, aggt, nct, _ = oracle_mod.aggregate(At.rowptr, At.col, At.val, 0.25, 3, 0, 0, symmetric=0)
    assert np.array_equal(m, mt) and np.array_equal(agg, aggt) and nc == nct
    mg, aggg, _, _ = oracle_mod.aggregate(A.rowptr, A.col, A.val, 0.25, 3, 0, 1, symmetric=0)
    assert np.array_equal(m, mg) and np.array_equal(agg, aggg)
    # the same from the definition: python-integer O-2 on the dense (A + A^T)/2
    D = A.to_dense()
    pm, pa, pnc, _ = py_aggregate((D + D.T) / 2, 0.25, 3)
    assert np.array_equal(m, pm) and np.array_equal(agg, pa) and nc == pnc
    assert 1.8 <= A.n / nc <= 2.6
    # structurally nonsymmetric: drop some (i, j) entries but keep (j, i)
    rng = np.random.default_rng(23)
    Dn = D.copy()
    iu = np.argwhere(np.triu(D, 1) != 0)
    for i, j in iu[rng.choice(len(iu), len(iu) // 4, replace=False)]:
        Dn[i, j] = 0.0
    rp, cl, vl = _csr_from_dense(Dn)
    m2, agg2, nc2, _ = oracle_mod.aggregate(rp, cl, vl, 0.25, 3, 0, 0, symmetric=0)
    pm2, pa2, pnc2, _ = py_aggregate((Dn + Dn.T) / 2, 0.25, 3)
    assert np.array_equal(m2, pm2) and np.array_equal(agg2, pa2) and nc2 == pnc2


def test_nonsymmetric_hierarchy_and_adjoint(oracle_mod):
    """O-7 with symmetric = 0 in the options: (P^T A P)^T = P^T A^T P level by level (the transposed
    hierarchy is the Galerkin hierarchy of A^T on the same aggregates), lambda = A^-T g against numpy,
    g.x = lambda.b, and the gradient against central finite differences."""
    S = inputs.variable_diffusion_csr((5, 5, 4), seed=31, sigma=1.0, ell=2.0)
    A = _row_scaled(S, 32)
    At = _transpose_csr(A)
    n = A.n
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, coarse_max_rows=8, symmetric=0)
    ot = oracle_mod.Oracle(At.rowptr, At.col, At.val, coarse_max_rows=8, symmetric=0)
    assert o.num_levels == ot.num_levels >= 3
    for l in range(o.num_levels):
        if l < o.num_levels - 1:
            assert np.array_equal(o.aggregates(l), ot.aggregates(l))
        rp, cl, vl = o.level_csr(l)
        Tl = _transpose_csr(inputs.Csr(len(rp) - 1, rp, cl, vl))
        rpt, clt, vlt = ot.level_csr(l)
        assert np.array_equal(Tl.rowptr, rpt) and np.array_equal(Tl.col, clt)  # pattern: bitwise
        assert np.max(np.abs(Tl.val - vlt)) <= 1e-14 * np.max(np.abs(vlt))     # values: summation order only
    D = A.to_dense()
    rng = np.random.default_rng(33)
    b, xt = rng.standard_normal(n), rng.standard_normal(n)
    x, i1 = o.solve(b, rtol=1e-13, maxit=300, krylov=1)
    lam, i2 = o.solve_transpose(x - xt, rtol=1e-13, maxit=300, krylov=1, symmetric=0)
    assert i1.status == 0 and i2.status == 0
    assert np.allclose(x, np.linalg.solve(D, b), rtol=1e-9, atol=1e-11)
    assert np.allclose(lam, np.linalg.solve(D.T, x - xt), rtol=1e-9, atol=1e-11)
    g = x - xt
    assert abs(g @ x - lam @ b) <= 1e-9 * np.linalg.norm(g) * np.linalg.norm(x)
    # the transposed V-cycle is the transpose of the V-cycle operator (nu1 = nu2): <B^T u, v> = <u, B v>
    u, v = rng.standard_normal(n), rng.standard_normal(n)
    Bv = o.vcycle(v)
    Btu = o.vcycle_transpose(u)  # A_l^T, same aggregates, same dinv (A16)
    assert abs(Btu @ v - u @ Bv) <= 1e-12 * np.linalg.norm(u) * np.linalg.norm(Bv)
    assert not abs(o.vcycle(u) @ v - u @ Bv) <= 1e-6 * np.linalg.norm(u) * np.linalg.norm(Bv)  # B itself is not symmetric
    gA = o.grad_values(lam, x)
    rows = np.repeat(np.arange(n), np.diff(A.rowptr))
    loss = lambda Dm: 0.5 * np.sum((np.linalg.solve(Dm, b) - xt) ** 2)
    ks = rng.choice(A.nnz, 40, replace=False)
    fd = np.empty(len(ks))
    for t, k in enumerate(ks):
        Dp, Dm = D.copy(), D.copy()
        Dp[rows[k], A.col[k]] += 1e-5
        Dm[rows[k], A.col[k]] -= 1e-5
        fd[t] = (loss(Dp) - loss(Dm)) / 2e-5
    assert np.linalg.norm(gA[ks] - fd) <= 1e-7 * np.linalg.norm(fd)


def test_agg_passes_two(oracle_mod):
    """agg_passes = 2 (O-1; north_star "pairwise or size-4"): the aggregates are the composition of two
    pairwise matchings, the second one on the intermediate Galerkin matrix with salt hash_seed + l + 1000."""
    A = inputs.config_matrix(3, 14)
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, agg_passes=2, hash_seed=4)
    _, agg1, nc1, _ = oracle_mod.aggregate(A.rowptr, A.col, A.val, 0.25, 4, 0, 0)
    mid = oracle_mod.galerkin(A.rowptr, A.col, A.val, agg1, nc1)
    _, agg2, nc2, _ = oracle_mod.aggregate(mid[0], mid[1], mid[2], 0.25, 4 + 1000, 0, 0)
    assert np.array_equal(o.aggregates(0), agg2[agg1]) and o.level_info(1)[0] == nc2
    sizes = np.bincount(o.aggregates(0))
    assert 3.5 <= A.n / nc2 <= 5.5 and sizes.max() <= 12 and np.median(sizes) == 4
    # the coarse operator is the Galerkin product on the composed map (dense P^T A P)
    P = np.zeros((A.n, nc2))
    P[np.arange(A.n), o.aggregates(0)] = 1.0
    rp, cl, vl = o.level_csr(1)
    assert np.allclose(inputs.Csr(nc2, rp, cl, vl).to_dense(), P.T @ dense(A) @ P, rtol=1e-13, atol=1e-13)
    # fewer levels than pairwise, still an SPD preconditioner that PCG converges with
    o1 = oracle_mod.Oracle(A.rowptr, A.col, A.val, hash_seed=4)
    assert o.num_levels < o1.num_levels
    b = inputs.config_rhs(3, A.n)
    x, info = o.solve(b, rtol=1e-10, maxit=200)
    assert info.status == 0 and info.iterations <= 2 * o1.solve(b, rtol=1e-10, maxit=200)[1].iterations
    assert np.linalg.norm(b - A.to_scipy() @ x) <= 1.01e-10 * np.linalg.norm(b)


@pytest.mark.parametrize("krylov", [0, 1])
def test_residual_history(oracle_mod, krylov):
    """PAPER.md:125 diagnostics: ||r_k|| / ||b|| per iteration; the iterates do not depend on rtol, so the
    history of a looser solve is a bitwise prefix of a tighter one (what the full-size goldens rely on)."""
    A = inputs.config_matrix(3, 12)
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val)
    b = inputs.config_rhs(3, A.n)
    _, i12 = o.solve(b, rtol=1e-12, maxit=200, krylov=krylov)
    h12 = o.residual_history()
    _, i8 = o.solve(b, rtol=1e-8, maxit=200, krylov=krylov)
    h8 = o.residual_history()
    assert len(h12) == i12.iterations and len(h8) == i8.iterations < i12.iterations
    assert h8[-1] == i8.rel_residual <= 1e-8 < h8[-2]
    if krylov == 0:
        assert np.array_equal(h8, h12[:len(h8)])
        assert int(np.argmax(h12 <= 1e-8)) + 1 == i8.iterations
    else:  # BiCGSTAB: the last entry of the looser solve may be its half-step exit ||s|| / ||b|| (A11)
        assert np.array_equal(h8[:-1], h12[:len(h8) - 1])


# ------------------------------------------------------------------------------------------
# NEXT-4: mixed-precision hierarchy (hierarchy_fp32): the V-cycle on fp32-rounded level operators
# ------------------------------------------------------------------------------------------
def py_vcycle(o, l, b, round32, nu1=2, nu2=2, gamma=1.0):
    """O-4 written out with scipy matrices taken from the oracle's level CSRs (plain definition, recursion)."""
    import scipy.sparse as sp

    L = o.num_levels - 1
    rp, cl, vl = o.level_csr(l)
    n = len(rp) - 1
    if l == L:
        return np.linalg.solve(sp.csr_matrix((vl, cl, rp), shape=(n, n)).toarray(), b)
    v = vl.astype(np.float32).astype(np.float64) if round32 else vl
    A = sp.csr_matrix((v, cl, rp), shape=(n, n))
    dinv = o.dinv(l)
    agg = o.aggregates(l)
    nc = o.level_info(l + 1)[0]
    x = dinv * b if nu1 > 0 else np.zeros(n)
    for _ in range(1, nu1):
        x = x + dinv * (b - A @ x)
    rc = np.bincount(agg, weights=b - A @ x, minlength=nc)
    x = x + gamma * py_vcycle(o, l + 1, rc, round32, nu1, nu2, gamma)[agg]
    for _ in range(nu2):
        x = x + dinv * (b - A @ x)
    return x


def test_mixed_precision_hierarchy(oracle_mod):
    """hierarchy_fp32 = 1: inside the V-cycle every sparse level operator is the fp64 one rounded to fp32 (used
    in fp64 arithmetic); dinv, the coarsest LU and the Krylov operator stay fp64.  Pinned by the recursion
    written out with scipy on the rounded matrices; the fp64 cycle is pinned by the same recursion unrounded."""
    A = inputs.variable_diffusion_csr((12, 12, 12), seed=9, sigma=1.5, ell=3.0)
    o64 = oracle_mod.Oracle(A.rowptr, A.col, A.val)
    o32 = oracle_mod.Oracle(A.rowptr, A.col, A.val, hierarchy_fp32=1)
    assert o64.num_levels == o32.num_levels >= 4
    for l in range(o64.num_levels):  # the hierarchy itself (aggregates, Galerkin values, dinv) is the fp64 one
        assert all(np.array_equal(a, b) for a, b in zip(o64.level_csr(l), o32.level_csr(l)))
    r = np.random.default_rng(3).standard_normal(A.n)
    z64, z32 = o64.vcycle(r), o32.vcycle(r)
    rel = lambda a, b: np.linalg.norm(a - b) / np.linalg.norm(b)
    assert rel(z64, py_vcycle(o64, 0, r, False)) <= 1e-13
    assert rel(z32, py_vcycle(o32, 0, r, True)) <= 1e-13
    assert 1e-10 < rel(z32, z64) < 1e-6          # a perturbation of fp32 size, not the same operator
    for l in (1, 2):                             # cycles started below level 0
        nl = o32.level_info(l)[0]
        rl = np.random.default_rng(l).standard_normal(nl)
        assert rel(o32.vcycle(rl, l), py_vcycle(o32, l, rl, True)) <= 1e-13
    # rounding a bitwise symmetric matrix keeps it symmetric: B stays symmetric, PCG applies and converges to the
    # fp64 tolerance with the fp64 operator A in the Krylov recurrences
    u, v = np.random.default_rng(5).standard_normal((2, A.n))
    assert abs(o32.vcycle(u) @ v - u @ o32.vcycle(v)) <= 1e-13 * np.linalg.norm(u) * np.linalg.norm(v)
    b = inputs.rhs_uniform(A.n, 4)
    x64, i64 = o64.solve(b, rtol=1e-10, maxit=200)
    x32, i32 = o32.solve(b, rtol=1e-10, maxit=200)
    assert i32.status == 0 and abs(i32.iterations - i64.iterations) <= 1
    assert np.linalg.norm(b - A.to_scipy() @ x32) <= 1.01e-10 * np.linalg.norm(b)
    assert rel(x32, x64) <= 1e-8
    # the solve of a nonsymmetric system and its adjoint with the rounded transposed operators
    N = inputs.stretched_channel_csr((6, 8, 6), 2.0)
    on = oracle_mod.Oracle(N.rowptr, N.col, N.val, symmetric=0, hierarchy_fp32=1, coarse_max_rows=16)
    D = N.to_dense()
    g = np.random.default_rng(6).standard_normal(N.n)
    lam, il = on.solve_transpose(g, rtol=1e-11, maxit=300, krylov=1, symmetric=0)
    assert il.status == 0 and np.allclose(lam, np.linalg.solve(D.T, g), rtol=1e-7, atol=1e-9)


# ------------------------------------------------------------------------------------------
# NEXT-4: Chebyshev-accelerated L1-Jacobi (smoother = 2)
# ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("ratio", [2.0, 6.0, 30.0])
@pytest.mark.parametrize("k", [1, 2, 3, 4])
def test_chebyshev_weights_are_the_minimax_polynomial(oracle_mod, k, ratio):
    """p(mu) = prod_j (1 - tau_j mu) must be THE degree-k polynomial with p(0) = 1 of least maximum on [1/ratio, 1]:
    max |p| = 1 / T_k((1+a)/(1-a)), attained k+1 times with alternating sign (equioscillation); a wrong root
    formula, interval or order of the reciprocal fails one of these."""
    tau = oracle_mod.cheby_weights(k, ratio)
    a = 1.0 / ratio
    assert np.all(np.diff(tau) > 0) and tau[0] > 1.0 and tau[-1] < ratio  # ascending, roots inside (a, 1)
    mu = np.linspace(a, 1.0, 200001)
    p = np.prod(1.0 - tau[:, None] * mu[None, :], axis=0)
    t = (1 + a) / (1 - a)
    Tk = np.cosh(k * np.arccosh(t))
    assert abs(np.max(np.abs(p)) - 1.0 / Tk) <= 1e-9 / Tk * 1e3
    ext = np.cos(np.pi * np.arange(k + 1) / k) * (1 - a) / 2 + (1 + a) / 2  # extrema of T_k mapped to [a, 1]
    pe = np.prod(1.0 - tau[:, None] * ext[None, :], axis=0)
    assert np.allclose(np.abs(pe), 1.0 / Tk, rtol=1e-10) and np.all(pe[:-1] * pe[1:] < 0)
    assert np.all(np.abs(np.prod(1.0 - tau[:, None] * np.linspace(0, a, 1001)[None, :], axis=0)) <= 1.0 + 1e-12)


def py_vcycle_w(o, l, b, wpre, wpost, gamma=1.0):
    """O-4 with per-sweep weights, written out with scipy matrices (post-sweeps take wpost in reverse order)."""
    import scipy.sparse as sp

    L = o.num_levels - 1
    rp, cl, vl = o.level_csr(l)
    n = len(rp) - 1
    A = sp.csr_matrix((vl, cl, rp), shape=(n, n))
    if l == L:
        return np.linalg.solve(A.toarray(), b)
    dinv, agg, nc = o.dinv(l), o.aggregates(l), o.level_info(l + 1)[0]
    x = wpre[0] * dinv * b
    for w in wpre[1:]:
        x = x + w * dinv * (b - A @ x)
    rc = np.bincount(agg, weights=b - A @ x, minlength=nc)
    x = x + gamma * py_vcycle_w(o, l + 1, rc, wpre, wpost, gamma)[agg]
    for w in wpost[::-1]:
        x = x + w * dinv * (b - A @ x)
    return x


def test_chebyshev_smoother(oracle_mod):
    A = inputs.variable_diffusion_csr((10, 10, 10), seed=4, sigma=1.5, ell=3.0)
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, smoother=2, cheby_ratio=6.0)
    o1 = oracle_mod.Oracle(A.rowptr, A.col, A.val)
    for l in range(o.num_levels):  # the hierarchy and the l1 diagonal are those of plain L1-Jacobi
        assert all(np.array_equal(a, b) for a, b in zip(o.level_csr(l), o1.level_csr(l)))
        if l < o.num_levels - 1:
            assert np.array_equal(o.dinv(l), o1.dinv(l))
    # spec(D_l1^-1 A) in (0, 1]: the premise of the fixed interval (Gershgorin), checked densely on level 0
    D = dense(A)
    mu = np.linalg.eigvals(np.diag(o.dinv(0)) @ D).real
    assert mu.min() > 0 and mu.max() <= 1.0 + 1e-12
    rel = lambda a, b: np.linalg.norm(a - b) / np.linalg.norm(b)
    w2 = oracle_mod.cheby_weights(2, 6.0)
    r = np.random.default_rng(2).standard_normal(A.n)
    assert rel(o.vcycle(r), py_vcycle_w(o, 0, r, w2, w2)) <= 1e-13
    assert rel(o1.vcycle(r), py_vcycle_w(o1, 0, r, np.ones(2), np.ones(2))) <= 1e-13  # weights 1: the plain cycle
    # B symmetric positive definite, spec(BA) in (0, 1 + eps]; fewer PCG iterations than plain L1-Jacobi
    n = A.n
    Bm = np.column_stack([o.vcycle(e) for e in np.eye(n)[:, :n]])
    assert np.linalg.norm(Bm - Bm.T) <= 1e-13 * np.linalg.norm(Bm)
    ev = np.linalg.eigvals(Bm @ D).real
    assert ev.min() > 0 and ev.max() <= 1.0 + 1e-10
    b = inputs.rhs_uniform(n, 3)
    x, ic = o.solve(b, rtol=1e-10, maxit=200)
    x1, i1 = o1.solve(b, rtol=1e-10, maxit=200)
    assert ic.status == 0 and ic.iterations < i1.iterations
    assert np.linalg.norm(b - A.to_scipy() @ x) <= 1.01e-10 * np.linalg.norm(b)
    # unequal sweep counts: weights of degree nu1 before, degree nu2 (reversed) after
    o32 = oracle_mod.Oracle(A.rowptr, A.col, A.val, smoother=2, pre_sweeps=3, post_sweeps=1)
    assert rel(o32.vcycle(r), py_vcycle_w(o32, 0, r, oracle_mod.cheby_weights(3, 6.0), oracle_mod.cheby_weights(1, 6.0))) <= 1e-13
