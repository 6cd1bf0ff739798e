"""amg_grad_values_noalloc (include/amg_b200.h): the handle-free, allocation-free variant of the batched
matrix-value gradient (G2, Eq. 2) whose interleaved copy of X lives in a file-scope static
device array.  Compared with the existing path (amg_grad_values on a handle) on two calls in a row that
share the static scratch -- the second with other inputs, another right-hand-side count, a leading dimension
larger than n and accumulation -- at the bar the gradient-kernel tests use (1e-14 * nrhs of the largest
entry); sizes beyond the static maximum are rejected with a message.

The file is named so that pytest collects it last: the run uses `pytest -x`."""
import ctypes as C

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

from paper_2606_09001_b200 import inputs  # noqa: E402

MAX_DOUBLES = 1 << 20  # AMG_NOALLOC_MAX_DOUBLES


@pytest.fixture(scope="module")
def B():
    from paper_2606_09001_b200 import binding

    assert torch.cuda.is_available()
    binding.load_library()
    return binding


def _case(B, cfg, edge):
    A = inputs.config_matrix(cfg, edge)
    s = B.AmgSolver(A.rowptr, A.col, A.val, device="cuda:0")
    d_rowptr = torch.as_tensor(np.ascontiguousarray(A.rowptr, dtype=np.int32), device="cuda:0")
    d_col = torch.as_tensor(np.ascontiguousarray(A.col, dtype=np.int32), device="cuda:0")
    return A, s, d_rowptr, d_col


def _vectors(seed, nrhs, n, ld):
    rng = np.random.default_rng(seed)
    lam = np.zeros((nrhs, ld))
    x = np.zeros((nrhs, ld))
    lam[:, :n] = rng.standard_normal((nrhs, n))
    x[:, :n] = rng.standard_normal((nrhs, n))
    return torch.as_tensor(lam, device="cuda:0").contiguous(), torch.as_tensor(x, device="cuda:0").contiguous()


def test_no_alloc_gradient_matches_the_existing_path_on_two_calls_in_a_row(B):
    # cfg 4 at 24^3: permuted 7-point pattern (short rows -> 8 lanes per row); 13 824 rows x 16 = 221 184 values
    A, s, d_rowptr, d_col = _case(B, 4, 24)
    n, nnz = A.n, A.nnz
    # ---- call 1: 16 right-hand sides, ld = n, overwrite ----
    lam1, x1 = _vectors(11, 16, n, n)
    want1 = torch.empty(nnz, dtype=torch.float64, device="cuda:0")
    B.amg_grad_values(s.h, lam1, x1, 16, n, want1, 0)
    got1 = torch.full((nnz,), float("nan"), dtype=torch.float64, device="cuda:0")
    B.amg_grad_values_noalloc(n, nnz, d_rowptr, d_col, lam1, x1, 16, n, got1, 0)
    torch.cuda.synchronize()
    scale1 = float(want1.abs().max())
    assert scale1 > 0
    assert float((got1 - want1).abs().max()) <= 1e-14 * scale1 * 16
    # ---- call 2, straight after, on the scratch call 1 left behind: other inputs, 5 right-hand sides (generic
    # kernel, odd count), ld > n, accumulate on top of a known vector ----
    ld = n + 37
    lam2, x2 = _vectors(12, 5, n, ld)
    base = torch.as_tensor(np.random.default_rng(13).standard_normal(nnz), device="cuda:0")
    want2 = base.clone()
    B.amg_grad_values(s.h, lam2, x2, 5, ld, want2, 1)
    got2 = base.clone()
    B.amg_grad_values_noalloc(n, nnz, d_rowptr, d_col, lam2, x2, 5, ld, got2, 1)
    torch.cuda.synchronize()
    scale2 = float((want2 - base).abs().max())
    assert scale2 > 0
    assert float((got2 - want2).abs().max()) <= 1e-14 * scale2 * 5
    # and against the definition for a few entries (Eq. 2): gA[k] = base[k] - sum_s lam_s[i] x_s[col[k]]
    lam_h, x_h, got_h, base_h = lam2.cpu().numpy(), x2.cpu().numpy(), got2.cpu().numpy(), base.cpu().numpy()
    rows = np.repeat(np.arange(n), np.diff(A.rowptr))
    for k in np.random.default_rng(14).integers(0, nnz, 200):
        ref = base_h[k] - float(np.dot(lam_h[:, rows[k]], x_h[:, A.col[k]]))
        assert abs(got_h[k] - ref) <= 1e-13 * max(1.0, abs(ref))
    # ---- the first inputs again: the result does not depend on what the scratch held ----
    again = torch.empty(nnz, dtype=torch.float64, device="cuda:0")
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]  # (kernels already loaded: lazy module loading is out of the picture)
    B.amg_grad_values_noalloc(n, nnz, d_rowptr, d_col, lam1, x1, 16, n, again, 0)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before  # the call allocated nothing on the device
    assert torch.equal(again, got1)
    s.close()


def test_no_alloc_gradient_long_rows_and_a_single_right_hand_side(B):
    # rows longer than 12 entries on average take the 32-lanes-per-row kernel: a dense-ish random pattern
    rng = np.random.default_rng(21)
    n = 300
    cols = [np.unique(np.concatenate(([i], rng.integers(0, n, 40)))) for i in range(n)]
    rowptr = np.zeros(n + 1, dtype=np.int32)
    rowptr[1:] = np.cumsum([len(c) for c in cols])
    col = np.concatenate(cols).astype(np.int32)
    nnz = int(rowptr[-1])
    d_rowptr, d_col = torch.as_tensor(rowptr, device="cuda:0"), torch.as_tensor(col, device="cuda:0")
    rows = np.repeat(np.arange(n), np.diff(rowptr))
    for nrhs in (1, 8):
        lam, x = _vectors(30 + nrhs, nrhs, n, n)
        got = torch.empty(nnz, dtype=torch.float64, device="cuda:0")
        B.amg_grad_values_noalloc(n, nnz, d_rowptr, d_col, lam, x, nrhs, n, got, 0)
        want = -np.einsum("sk,sk->k", lam.cpu().numpy()[:, rows], x.cpu().numpy()[:, col])
        assert np.max(np.abs(got.cpu().numpy() - want)) <= 1e-14 * np.max(np.abs(want)) * nrhs


def test_no_alloc_gradient_rejects_sizes_beyond_the_static_scratch(B):
    lib = B.load_library()
    n = MAX_DOUBLES // 16 + 1  # n * 16 is one row over the limit
    d_rowptr = torch.zeros(n + 1, dtype=torch.int32, device="cuda:0")
    d_col = torch.zeros(8, dtype=torch.int32, device="cuda:0")
    v = torch.zeros(16 * n, dtype=torch.float64, device="cuda:0")
    gA = torch.zeros(8, dtype=torch.float64, device="cuda:0")
    with pytest.raises(B.AmgError) as e:
        B.amg_grad_values_noalloc(n, 8, d_rowptr, d_col, v, v, 16, n, gA, 0)
    assert e.value.status == 7 and "AMG_NOALLOC_MAX_DOUBLES" in str(e.value)
    # exactly at the limit the call is accepted (an all-empty pattern: nothing is written)
    n_ok = MAX_DOUBLES // 16
    B.amg_grad_values_noalloc(n_ok, 8, d_rowptr[: n_ok + 1].contiguous(), d_col, v, v, 16, n_ok, gA, 0)
    torch.cuda.synchronize()
    assert float(gA.abs().max()) == 0.0
    with pytest.raises(B.AmgError) as e:  # ld < n, null pointer
        B.amg_grad_values_noalloc(100, 8, d_rowptr, d_col, v, v, 2, 99, gA, 0)
    assert e.value.status == 1
    st = lib.amg_grad_values_noalloc(C.c_int64(4), C.c_int64(4), None, None, None, None, C.c_int32(1), C.c_int64(4), None,
                                     C.c_int32(0), None)
    assert st == 1 and b"null" in lib.amg_last_error(None)
