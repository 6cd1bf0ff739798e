"""GPU parity of the NEXT-4 variants: size-4 aggregation (agg_passes = 2; north_star
"pairwise or size-4"), the residual-history diagnostics, the keyed LRU cache of
hierarchies -- each against the oracle option of the same name, through the C ABI.
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


@pytest.mark.parametrize("case", [(3, 40), (4, 28), (2, 96)])
def test_size4_aggregation_matches_the_oracle(oracle_mod, B, case):
    cfg, edge = case
    A = inputs.config_matrix(cfg, edge)
    v = inputs.config_rhs(cfg, A.n)
    b = A.to_scipy() @ v if cfg == 2 else v
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, agg_passes=2, hash_seed=4)
    s = B.AmgSolver(A.rowptr, A.col, A.val, agg_passes=2, hash_seed=4)
    o1 = oracle_mod.Oracle(A.rowptr, A.col, A.val, hash_seed=4)
    try:
        assert s.num_levels == o.num_levels < o1.num_levels
        for l in range(s.num_levels - 1):  # composed map of two matchings: the same integers
            assert np.array_equal(s.aggregates(l).cpu().numpy(), o.aggregates(l)), l
            sizes = np.bincount(o.aggregates(l))
            assert np.median(sizes) == 4 or l >= s.num_levels - 3
        for l in range(s.num_levels):
            rp, cl, vl = (t.cpu().numpy() for t in s.level_csr(l))
            orp, ocl, ovl = o.level_csr(l)
            assert np.array_equal(rp, orp) and np.array_equal(cl, ocl)
            assert np.max(np.abs(vl - ovl)) <= 1e-13 * np.max(np.abs(ovl))
        r = np.random.default_rng(3).standard_normal(A.n)
        assert rel(s.apply_preconditioner(r).cpu().numpy(), o.vcycle(r, 0)) <= 1e-12
        xg, ig = s.solve(b, 1e-8, 500, 0)
        xo, io = o.solve(b, 1e-8, 500, 0, 1)
        assert ig.status == io.status == 0 and abs(ig.iterations - io.iterations) <= 2
        assert np.linalg.norm(b - A.to_scipy() @ xg.cpu().numpy()) <= 1e-8 * np.linalg.norm(b)
        xg, _ = s.solve(b, 1e-11, 500, 0)
        xo, _ = o.solve(b, 1e-13, 500, 0, 1)
        assert rel(xg.cpu().numpy(), xo) <= 1e-6
    finally:
        s.close()
        o.close()
        o1.close()


@pytest.mark.parametrize("krylov", [0, 1])
def test_residual_history_matches_the_oracle(oracle_mod, B, krylov):
    A = inputs.config_matrix(3, 24)
    b = inputs.config_rhs(3, A.n)
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val)
    s = B.AmgSolver(A.rowptr, A.col, A.val)
    try:
        _, ig = s.solve(b, 1e-10, 200, krylov)
        hg = s.residual_history()
        _, io = o.solve(b, 1e-10, 200, krylov, 1)
        ho = o.residual_history()
        assert len(hg) == ig.iterations and hg[-1] == ig.rel_residual <= 1e-10
        m = min(len(hg), len(ho))
        assert abs(len(hg) - len(ho)) <= 2
        # the same residual curve, iteration by iteration (rounding order differs: relative 1e-6 on values
        # that fall by ten orders of magnitude)
        assert np.max(np.abs(hg[:m] - ho[:m]) / ho[:m]) <= 1e-6
        # the iterates do not depend on rtol: the history of a looser solve is a bitwise prefix
        _, i6 = s.solve(b, 1e-6, 200, krylov)
        h6 = s.residual_history()
        assert len(h6) == i6.iterations < len(hg)
        if krylov == 0:
            assert np.array_equal(h6, hg[:len(h6)])
        else:
            assert np.array_equal(h6[:-1], hg[:len(h6) - 1])
        # maxit stop
        _, i3 = s.solve(b, 1e-30, 3, krylov)
        assert i3.status == 1 and len(s.residual_history()) == 3
    finally:
        s.close()
        o.close()


def test_lru_cache_of_hierarchies(oracle_mod, B):
    dev = torch.device("cuda:0")
    to = lambda a, dt: torch.as_tensor(a).to(dtype=dt, device=dev).contiguous()
    mats = [inputs.config_matrix(3, 20), inputs.config_matrix(1, 48), inputs.config_matrix(3, 24)]
    dm = [(A.n, A.nnz, to(A.rowptr, torch.int32), to(A.col, torch.int32), to(A.val, torch.float64)) for A in mats]
    c = B.amg_cache_create(2)
    try:
        h0, hit = B.amg_cache_get(c, *dm[0])
        assert hit == 0
        h0b, hit = B.amg_cache_get(c, *dm[0], on_hit=0)           # same pattern: the same handle, untouched
        assert hit == 1 and h0b.value == h0.value
        h1, hit = B.amg_cache_get(c, *dm[1])
        assert hit == 0 and h1.value != h0.value
        assert B.amg_cache_stats(c) == {"entries": 2, "hits": 1, "misses": 2, "evictions": 0}
        # new values on the pattern of matrix 0 (variable coefficients on the same 20^3 stencil): a hit with a
        # warm resetup; the solve equals the oracle built on the new values
        A0 = mats[0]
        Anew = inputs.variable_diffusion_csr((20, 20, 20), seed=77, sigma=1.0, ell=4.0)
        assert np.array_equal(Anew.col, A0.col)
        h0c, hit = B.amg_cache_get(c, A0.n, A0.nnz, dm[0][2], dm[0][3], to(Anew.val, torch.float64), on_hit=1)
        assert hit == 1 and h0c.value == h0.value
        b = torch.as_tensor(inputs.rhs_uniform(A0.n, 1)).to(dev)
        x = torch.empty_like(b)
        info = B.amg_solve(h0c, b, x, 1e-8, 500)
        o = oracle_mod.Oracle(Anew.rowptr, Anew.col, Anew.val)
        xo, io = o.solve(b.cpu().numpy(), 1e-8, 500, 0, 1)
        assert info.status == 0 and abs(info.iterations - io.iterations) <= 2
        assert np.linalg.norm(b.cpu().numpy() - Anew.to_scipy() @ x.cpu().numpy()) <= 1e-8 * torch.linalg.norm(b).item()
        o.close()
        # a third pattern evicts the least recently used entry (matrix 1), not matrix 0
        h2, hit = B.amg_cache_get(c, *dm[2])
        assert hit == 0 and B.amg_cache_stats(c)["evictions"] == 1
        _, hit = B.amg_cache_get(c, *dm[0], on_hit=0)
        assert hit == 1
        _, hit = B.amg_cache_get(c, *dm[1])
        assert hit == 0                                           # it was evicted: set up again
        # different options on the same pattern are a different key
        _, hit = B.amg_cache_get(c, *dm[1], opt=B.amg_options_default(pre_sweeps=1, post_sweeps=1))
        assert hit == 0
    finally:
        B.amg_cache_destroy(c)


def test_warm_resetup_keeps_graphs_batches_and_the_transposed_hierarchy(oracle_mod, B):
    """NEXT-1 warm path: amg_resetup_values(keep_aggregates = 1) rewrites values only.  Repeated resetups on one
    handle (A0 -> A1 -> A2 -> A0), each followed by single solves (cached CUDA graphs), a batched solve (cached
    work vectors / ring geometry) -- against the oracle built on the same values with the kept aggregates."""
    shape = (24, 24, 24)
    mats = [inputs.variable_diffusion_csr(shape, seed=s, sigma=1.5, ell=4.0) for s in (81, 82, 83)]
    A0 = mats[0]
    n = A0.n
    s = B.AmgSolver(A0.rowptr, A0.col, A0.val)
    o0 = oracle_mod.Oracle(A0.rowptr, A0.col, A0.val)
    aggs = [o0.aggregates(l) for l in range(o0.num_levels - 1)]
    b = inputs.rhs_uniform(n, 5)
    Bh = np.stack([inputs.rhs_uniform(n, 50 + k) for k in range(8)])
    Bd = torch.as_tensor(Bh).cuda().contiguous()
    X = torch.empty_like(Bd)
    x_first, _ = s.solve(b, 1e-8, 500, 0)
    B.amg_solve_batched(s.h, 0, Bd, X, 8, n, 1e-8, 500)
    try:
        for A in (mats[1], mats[2], mats[0]):
            s.resetup_values(A.val, keep_aggregates=True)
            o = oracle_mod.Oracle(A.rowptr, A.col, A.val, aggregates=aggs)
            for l in range(s.num_levels):
                _, _, vg = s.level_csr(l)
                _, _, vo = o.level_csr(l)
                assert np.max(np.abs(vg.cpu().numpy() - vo)) <= 1e-13 * np.max(np.abs(vo)), l
            r = np.random.default_rng(9).standard_normal(n)
            assert rel(s.apply_preconditioner(r).cpu().numpy(), o.vcycle(r, 0)) <= 1e-12
            for krylov in (0, 1):
                xg, ig = s.solve(b, 1e-8, 500, krylov)
                xo, io = o.solve(b, 1e-8, 500, krylov, 1)
                assert ig.status == io.status == 0 and abs(ig.iterations - io.iterations) <= 2
                assert np.linalg.norm(b - A.to_scipy() @ xg.cpu().numpy()) <= 1e-8 * np.linalg.norm(b)
            infos = B.amg_solve_batched(s.h, 0, Bd, X, 8, n, 1e-8, 500)
            for k in (0, 5):
                xo, io = o.solve(Bh[k], 1e-8, 500, 0, 1)
                assert infos[k].status == 0 and abs(infos[k].iterations - io.iterations) <= 2
                assert np.linalg.norm(Bh[k] - A.to_scipy() @ X[k].cpu().numpy()) <= 1e-8 * np.linalg.norm(Bh[k])
            o.close()
        # back on the first values: the first solution again, bitwise (nothing structural moved)
        x_again, _ = s.solve(b, 1e-8, 500, 0)
        assert rel(x_again.cpu().numpy(), x_first.cpu().numpy()) <= 1e-12
    finally:
        s.close()
        o0.close()


def test_warm_resetup_of_a_nonsymmetric_handle(oracle_mod, B):
    A0 = inputs.stretched_channel_csr((10, 16, 12), 2.0)
    A1 = inputs.stretched_channel_csr((10, 16, 12), 1.2)  # same pattern, other stretching: new values
    assert np.array_equal(A0.col, A1.col)
    s = B.AmgSolver(A0.rowptr, A0.col, A0.val)
    o0 = oracle_mod.Oracle(A0.rowptr, A0.col, A0.val, symmetric=0)
    aggs = [o0.aggregates(l) for l in range(o0.num_levels - 1)]
    g = inputs.rhs_uniform(A0.n, 3)
    s.solve_transpose(g, 1e-8, 300)
    s.resetup_values(A1.val, keep_aggregates=True)
    o1 = oracle_mod.Oracle(A1.rowptr, A1.col, A1.val, aggregates=aggs, symmetric=0)
    try:
        assert s.symmetric == 0
        rows = s.level_info(1)[0]
        x = np.random.default_rng(2).standard_normal(rows)
        import scipy.sparse as sp

        rp, cl, vl = o1.level_csr(1)
        A1c = sp.csr_matrix((vl, cl, rp), shape=(rows, rows))
        assert rel(s.level_op(1, 7, x, None, rows).cpu().numpy(), A1c.T @ x) <= 1e-13
        r = np.random.default_rng(4).standard_normal(A0.n)
        assert rel(s.level_op(0, 8, None, r, A0.n).cpu().numpy(), o1.vcycle_transpose(r, 0)) <= 1e-12
        lam, il = s.solve_transpose(g, 1e-8, 300)
        lo, ilo = o1.solve_transpose(g, 1e-8, 300, 1, 1, 0)
        assert il.status == ilo.status == 0 and abs(il.iterations - ilo.iterations) <= 2
        assert np.linalg.norm(g - A1.to_scipy().T @ lam.cpu().numpy()) <= 1e-8 * np.linalg.norm(g)
    finally:
        s.close()
        o0.close()
        o1.close()


@pytest.mark.parametrize("opts", [dict(), dict(force_generic=1), dict(tail_dense_rows=0)])
@pytest.mark.parametrize("case", [(3, 40), (4, 28)])
def test_mixed_precision_hierarchy_matches_the_oracle(oracle_mod, B, case, opts):
    """hierarchy_fp32 = 1 (NEXT-4): the V-cycle's sparse level operators stored in fp32 (6 bytes per
    entry), used in fp64 arithmetic; the Krylov operator, dinv, the LU and all vectors fp64.  The oracle rounds the
    same values: the V-cycle agrees to 1e-12 as in fp64 mode, the solves to the usual bars."""
    cfg, edge = case
    A = inputs.config_matrix(cfg, edge)
    Asp = A.to_scipy()
    n = A.n
    b = inputs.config_rhs(cfg, n)
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, hierarchy_fp32=1)
    o64 = oracle_mod.Oracle(A.rowptr, A.col, A.val)
    s = B.AmgSolver(A.rowptr, A.col, A.val, hierarchy_fp32=1, **opts)
    try:
        assert s.num_levels == o.num_levels
        for l in range(s.num_levels - 1):
            assert np.array_equal(s.aggregates(l).cpu().numpy(), o.aggregates(l))
        r = np.random.default_rng(3).standard_normal(n)
        z = s.apply_preconditioner(r).cpu().numpy()
        assert rel(z, o.vcycle(r, 0)) <= 1e-12
        if cfg == 4:  # (the integer stencils of cfg 3 are exact in fp32: the two cycles coincide there)
            assert 1e-10 < rel(z, o64.vcycle(r, 0)) < 1e-6  # it really is the rounded operator
        for l in range(1, s.num_levels):
            nl = s.level_info(l)[0]
            bl = np.random.default_rng(100 + l).standard_normal(nl)
            assert rel(s.level_op(l, 5, None, bl, nl).cpu().numpy(), o.vcycle(bl, l)) <= 1e-12
        for krylov in (0, 1):
            xg, ig = s.solve(b, 1e-8, 500, krylov)
            xo, io = o.solve(b, 1e-8, 500, krylov, 1)
            assert ig.status == io.status == 0 and abs(ig.iterations - io.iterations) <= 2
            assert np.linalg.norm(b - Asp @ xg.cpu().numpy()) <= 1e-8 * np.linalg.norm(b)   # fp64 residual, fp64 A
            xg, _ = s.solve(b, 1e-11, 500, krylov)
            xo, _ = o64.solve(b, 1e-13, 500, krylov, 1)
            assert rel(xg.cpu().numpy(), xo) <= 1e-6
        # batched solve, warm resetup (fp32 value sections refilled), adjoint
        Bh = np.stack([inputs.rhs_uniform(n, 60 + k) for k in range(8)])
        Bd = torch.as_tensor(Bh).cuda().contiguous()
        X = torch.empty_like(Bd)
        infos = B.amg_solve_batched(s.h, 0, Bd, X, 8, n, 1e-8, 500)
        for k in (0, 7):
            xo, io = o.solve(Bh[k], 1e-8, 500, 0, 1)
            assert infos[k].status == 0 and abs(infos[k].iterations - io.iterations) <= 2
            assert np.linalg.norm(Bh[k] - Asp @ X[k].cpu().numpy()) <= 1e-8 * np.linalg.norm(Bh[k])
        s.resetup_values(A.val * 2.0, keep_aggregates=True)
        z2 = s.apply_preconditioner(r).cpu().numpy()
        assert rel(z2, 0.5 * z) <= 1e-12
        x2, i2 = s.solve(b, 1e-8, 500, 0)
        assert i2.status == 0 and np.linalg.norm(b - 2.0 * (Asp @ x2.cpu().numpy())) <= 1e-8 * np.linalg.norm(b)
    finally:
        s.close()
        o.close()
        o64.close()


def test_mixed_precision_hierarchy_nonsymmetric(oracle_mod, B):
    A = inputs.stretched_channel_csr((12, 20, 16), 2.0)
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, symmetric=0, hierarchy_fp32=1)
    s = B.AmgSolver(A.rowptr, A.col, A.val, hierarchy_fp32=1)
    try:
        r = np.random.default_rng(8).standard_normal(A.n)
        assert rel(s.level_op(0, 8, None, r, A.n).cpu().numpy(), o.vcycle_transpose(r, 0)) <= 1e-12
        g = inputs.rhs_uniform(A.n, 9)
        lam, il = s.solve_transpose(g, 1e-8, 500)
        lo, ilo = o.solve_transpose(g, 1e-8, 500, 1, 1, 0)
        assert il.status == ilo.status == 0 and abs(il.iterations - ilo.iterations) <= 2
        assert np.linalg.norm(g - A.to_scipy().T @ lam.cpu().numpy()) <= 1e-8 * np.linalg.norm(g)
    finally:
        s.close()
        o.close()


@pytest.mark.parametrize("opts", [dict(), dict(force_generic=1), dict(tail_dense_rows=0), dict(pre_sweeps=3, post_sweeps=3),
                                  dict(pre_sweeps=1, post_sweeps=1), dict(pre_sweeps=3, post_sweeps=1)])
@pytest.mark.parametrize("case", [(3, 40), (4, 28)])
def test_chebyshev_smoother_matches_the_oracle(oracle_mod, B, case, opts):
    """smoother = 2 (NEXT-4): Chebyshev-accelerated L1-Jacobi, per-sweep diagonals tau_j * dinv.  V-cycle from every
    level against the oracle (1e-12), solves at the usual bars, fewer iterations than plain L1-Jacobi."""
    cfg, edge = case
    A = inputs.config_matrix(cfg, edge)
    Asp = A.to_scipy()
    n = A.n
    b = inputs.config_rhs(cfg, n)
    oo = {k: v for k, v in opts.items() if k in ("pre_sweeps", "post_sweeps")}
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, smoother=2, **oo)
    s = B.AmgSolver(A.rowptr, A.col, A.val, smoother=2, **opts)
    try:
        for l in range(s.num_levels):
            nl = s.level_info(l)[0]
            bl = np.random.default_rng(100 + l).standard_normal(nl)
            assert rel(s.level_op(l, 5, None, bl, nl).cpu().numpy(), o.vcycle(bl, l)) <= 1e-12, l
        r = np.random.default_rng(3).standard_normal(n)
        assert rel(s.apply_preconditioner(r).cpu().numpy(), o.vcycle(r, 0)) <= 1e-12
        sym = opts.get("pre_sweeps", 2) == opts.get("post_sweeps", 2)
        for krylov in ((0, 1) if sym else (1,)):
            xg, ig = s.solve(b, 1e-8, 500, krylov)
            xo, io = o.solve(b, 1e-8, 500, krylov, 1)
            assert ig.status == io.status == 0 and abs(ig.iterations - io.iterations) <= 2
            assert np.linalg.norm(b - Asp @ xg.cpu().numpy()) <= 1e-8 * np.linalg.norm(b)
        if not opts:
            o1 = oracle_mod.Oracle(A.rowptr, A.col, A.val)
            _, i1 = o1.solve(b, 1e-8, 500, 0, 1)
            xg, ig = s.solve(b, 1e-8, 500, 0)
            assert ig.iterations < i1.iterations
            o1.close()
            # batched solve and warm resetup keep the weighted diagonals
            Bh = np.stack([inputs.rhs_uniform(n, 60 + k) for k in range(8)])
            Bd = torch.as_tensor(Bh).cuda().contiguous()
            X = torch.empty_like(Bd)
            infos = B.amg_solve_batched(s.h, 0, Bd, X, 8, n, 1e-8, 500)
            for k in (0, 7):
                xo, io = o.solve(Bh[k], 1e-8, 500, 0, 1)
                assert infos[k].status == 0 and abs(infos[k].iterations - io.iterations) <= 2
                assert np.linalg.norm(Bh[k] - Asp @ X[k].cpu().numpy()) <= 1e-8 * np.linalg.norm(Bh[k])
            z = s.apply_preconditioner(r).cpu().numpy()
            s.resetup_values(A.val * 4.0, keep_aggregates=True)
            assert rel(s.apply_preconditioner(r).cpu().numpy(), 0.25 * z) <= 1e-12
    finally:
        s.close()
        o.close()


def test_full_size_headline_options_against_the_oracle(oracle_mod, B):
    """The options bench.py runs the headline with (cfg 3, 128^3: size-4 aggregation, Chebyshev-weighted L1-Jacobi,
    gamma = 1.6, all fp64), on the GPU against the oracle with the same options at full size: identical hierarchy
    (integers), iterations +-2, host fp64 residual, x against the oracle's converged solution."""
    import os

    opts = dict(smoother=2, agg_passes=2, coarse_scale=1.6)
    A = inputs.config_matrix(3)
    b = inputs.config_rhs(3, A.n)
    oracle_mod.set_threads(os.cpu_count() or 1)
    try:
        o = oracle_mod.Oracle(A.rowptr, A.col, A.val, **opts)
        s = B.AmgSolver(A.rowptr, A.col, A.val, **opts)
        assert s.num_levels == o.num_levels
        for l in range(s.num_levels):
            assert s.level_info(l) == o.level_info(l)
            if l < s.num_levels - 1:
                assert np.array_equal(s.aggregates(l).cpu().numpy(), o.aggregates(l)), l
        xg, ig = s.solve(b, 1e-8, 500, 0)
        xo, io = o.solve(b, 1e-8, 500, 0, 1)
        assert ig.status == io.status == 0 and abs(ig.iterations - io.iterations) <= 2
        assert ig.iterations < 30  # (the library defaults need 42)
        assert np.linalg.norm(b - A.to_scipy() @ xg.cpu().numpy()) <= 1e-8 * np.linalg.norm(b)
        xg, _ = s.solve(b, 1e-11, 500, 0)
        xo, _ = o.solve(b, 1e-13, 500, 0, 1)
        assert rel(xg.cpu().numpy(), xo) <= 1e-6
        r = np.random.default_rng(1).standard_normal(A.n)
        assert rel(s.apply_preconditioner(r).cpu().numpy(), o.vcycle(r, 0)) <= 1e-12
        u, v = np.random.default_rng(2).standard_normal((2, A.n))
        Bu, Bv = s.apply_preconditioner(u).cpu().numpy(), s.apply_preconditioner(v).cpu().numpy()
        assert abs(Bu @ v - u @ Bv) <= 1e-12 * np.linalg.norm(Bu) * np.linalg.norm(v) and Bu @ u > 0  # B stays SPD
        s.close()
        o.close()
    finally:
        oracle_mod.set_threads(1)


@pytest.mark.parametrize("opts", [dict(), dict(smoother=2, agg_passes=2, coarse_scale=1.6), dict(krylov=1)])
def test_value_dictionary_is_bit_faithful_storage(oracle_mod, B, opts):
    """amg_options::value_dict: a level with at most 255 distinct fp64 values stores 8-bit codes into a table of
    those values.  The operator is the same, value for value: against the oracle (V-cycle <= 1e-12, solve, iteration
    count) exactly like the fp64 layout, and against the fp64 layout of the same handle options to rounding (tile
    boundaries differ, so row sums associate differently).  A Poisson hierarchy takes the dictionary on every level
    that runs the row-tile kernels, a variable-coefficient one on none."""
    A = inputs.config_matrix(3, 40)
    b = inputs.config_rhs(3, A.n)
    okw = {k: v for k, v in opts.items() if k != "krylov"}
    o = oracle_mod.Oracle(A.rowptr, A.col, A.val, **okw)
    sd = B.AmgSolver(A.rowptr, A.col, A.val, value_dict=1, **opts)
    s8 = B.AmgSolver(A.rowptr, A.col, A.val, value_dict=0, **opts)
    try:
        nd = int(B.amg_get_algorithmic_bytes(sd.h, 12))
        assert nd >= 2 and int(B.amg_get_algorithmic_bytes(s8.h, 12)) == 0
        # 4 bytes per entry (column | code) instead of 10
        assert B.amg_get_algorithmic_bytes(sd.h, 11) < 0.5 * B.amg_get_algorithmic_bytes(s8.h, 11)
        r = torch.as_tensor(b, device="cuda")
        zo = o.vcycle(b)
        zd, z8 = sd.apply_preconditioner(r).cpu().numpy(), s8.apply_preconditioner(r).cpu().numpy()
        assert rel(zd, zo) <= 1e-12 and rel(z8, zo) <= 1e-12 and rel(zd, z8) <= 1e-12
        kry = opts.get("krylov", 0)
        xo, io = o.solve(b, 1e-13, 500, kry, 1)
        xd, idd = sd.solve(b, 1e-11, 500, kry)
        x8, i8 = s8.solve(b, 1e-11, 500, kry)
        assert idd.status == 0 and idd.iterations == i8.iterations
        assert rel(xd.cpu().numpy(), xo) <= 1e-6 and rel(xd.cpu().numpy(), x8.cpu().numpy()) <= 1e-9
        _, i1 = sd.solve(b, 1e-8, 500, kry)
        _, io1 = o.solve(b, 1e-8, 500, kry, 1)
        assert abs(i1.iterations - io1.iterations) <= 2
        # 8 right-hand sides at once through the batched kernel (symmetric PCG handles)
        if kry == 0:
            Bm = torch.as_tensor(np.stack([inputs.config_rhs(5, A.n, k) for k in range(8)]), device="cuda").contiguous()
            Xd, X8 = torch.empty_like(Bm), torch.empty_like(Bm)
            B.amg_solve_batched(sd.h, 0, Bm, Xd, 8, A.n, 1e-11, 500)
            B.amg_solve_batched(s8.h, 0, Bm, X8, 8, A.n, 1e-11, 500)
            assert rel(Xd.cpu().numpy(), X8.cpu().numpy()) <= 1e-9
    finally:
        sd.close(), s8.close(), o.close()
    A4 = inputs.config_matrix(4, 20)
    s4 = B.AmgSolver(A4.rowptr, A4.col, A4.val)
    assert int(B.amg_get_algorithmic_bytes(s4.h, 12)) == 0  # all values different: fp64 blobs as before
    s4.close()


def test_value_dictionary_warm_resetup(oracle_mod, B):
    """Warm resetup of a hierarchy stored as codes: new values with few distinct entries rebuild the dictionaries
    in place (the handle stays, graphs stay); new values that are all different do not fit a dictionary: the call
    falls back to the rebuild with fp64 blobs.  Both equal a fresh oracle on the new values."""
    A = inputs.config_matrix(3, 32)
    b = inputs.config_rhs(3, A.n)
    s = B.AmgSolver(A.rowptr, A.col, A.val)
    try:
        assert int(B.amg_get_algorithmic_bytes(s.h, 12)) >= 2
        x0, _ = s.solve(b, 1e-11, 300)
        # (i) another constant-coefficient operator on the same pattern: 2.5 A + 0.75 I
        v1 = 2.5 * A.val
        diag = A.col == np.repeat(np.arange(A.n), np.diff(A.rowptr))
        v1[diag] += 0.75
        s.resetup_values(v1, keep_aggregates=True)
        assert int(B.amg_get_algorithmic_bytes(s.h, 12)) >= 2
        o1 = oracle_mod.Oracle(A.rowptr, A.col, v1)
        x1, i1 = s.solve(b, 1e-11, 300)
        xo1, _ = o1.solve(b, 1e-13, 300, 0, 1)
        assert i1.status == 0 and rel(x1.cpu().numpy(), xo1) <= 1e-6
        z1 = s.apply_preconditioner(torch.as_tensor(b, device="cuda")).cpu().numpy()
        assert rel(z1, o1.vcycle(b)) <= 1e-12
        o1.close()
        # (ii) symmetric random perturbation of every off-diagonal: ~ nnz / 2 distinct values
        import scipy.sparse as sp

        rng = np.random.default_rng(77)
        M = sp.csr_matrix((A.val.copy(), A.col, A.rowptr), shape=(A.n, A.n)).tocoo()
        lo, hi = np.minimum(M.row, M.col), np.maximum(M.row, M.col)
        pert = 1.0 + 0.2 * np.sin(1.0 + 0.37 * lo + 0.11 * hi) * (lo != hi)  # same factor for (i, j) and (j, i)
        M2 = sp.csr_matrix((M.data * pert, (M.row, M.col)), shape=(A.n, A.n))
        M2.sort_indices()
        assert np.array_equal(M2.indices, A.col)
        v2 = M2.data.copy()
        v2[diag] = 6.5
        s.resetup_values(v2, keep_aggregates=True)
        assert int(B.amg_get_algorithmic_bytes(s.h, 12)) == 0  # fell back to fp64 blobs
        o2 = oracle_mod.Oracle(A.rowptr, A.col, v2, aggregates=[s.aggregates(l).cpu().numpy() for l in range(s.num_levels - 1)])
        x2, i2 = s.solve(b, 1e-11, 300)
        xo2, _ = o2.solve(b, 1e-13, 300, 0, 1)
        assert i2.status == 0 and rel(x2.cpu().numpy(), xo2) <= 1e-6
        o2.close()
        del x0
    finally:
        s.close()


def test_report_file(B, tmp_path):
    """optional file-based output with the hierarchy statistics and the residual history."""
    A = inputs.config_matrix(3, 24)
    s = B.AmgSolver(A.rowptr, A.col, A.val)
    try:
        x, info = s.solve(inputs.config_rhs(3, A.n), 1e-8, 200)
        p = tmp_path / "amg_report.txt"
        B.amg_write_report(s.h, p)
        txt = p.read_text().splitlines()
        assert txt[0].startswith("amg_b200 hierarchy report") and f"levels {s.num_levels}" in txt[1]
        rows = [l.split() for l in txt if l.split() and l.split()[0].isdigit() and len(l.split()) == 9]
        # last column: size of the level's value dictionary (a 24^3 Poisson level 0 holds 2 distinct values: -1, 6)
        assert int(rows[0][8]) == 2 and all(0 <= int(r[8]) <= 255 for r in rows)
        assert [(int(r[1]), int(r[2])) for r in rows] == [s.level_info(l) for l in range(s.num_levels)]
        hist = [float(l.split()[1]) for l in txt[txt.index(next(t for t in txt if t.startswith("residual history"))) + 1:]]
        assert len(hist) == info.iterations and np.array_equal(np.array(hist), s.residual_history())
        oc = float(next(t for t in txt if t.startswith("grid complexity")).split()[5])
        assert abs(oc - sum(s.level_info(l)[1] for l in range(s.num_levels)) / A.nnz) < 1e-3
    finally:
        s.close()
