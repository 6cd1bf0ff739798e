"""Boundary behaviour of the C ABI on the GPU (SURVEY.md §8(b) conventions): the allocator hook routes
library-owned memory through torch's caching allocator ("PyTorch is used only for device memory"),
info == NULL makes a solve return without waiting, distinct handles work concurrently on distinct
streams and threads, every entry point is stream-ordered on the caller's stream.
"""
import ctypes as C
import threading

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

from paper_2606_09001_b200 import inputs  # noqa: E402


@pytest.fixture(scope="module")
def B():
    from paper_2606_09001_b200 import binding

    assert torch.cuda.is_available()
    binding.load_library()
    return binding


def test_allocator_hook_routes_library_memory_through_torch(B):
    lib = B.load_library()
    live, total, freed_unknown = {}, [0], [0]
    ALLOC = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p)
    FREE = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)

    def alloc(nbytes, stream, user):
        p = torch.cuda.caching_allocator_alloc(int(nbytes), device=0, stream=stream or 0)
        live[p] = int(nbytes)
        total[0] += int(nbytes)
        return p

    def free(p, user):
        if p not in live:
            freed_unknown[0] += 1
            return
        del live[p]
        torch.cuda.caching_allocator_delete(p)

    a_cb, f_cb = ALLOC(alloc), FREE(free)
    A = inputs.config_matrix(3, 32)
    b = inputs.config_rhs(3, A.n)
    torch.cuda.synchronize()
    base = torch.cuda.memory_allocated()
    assert lib.amg_set_allocator(a_cb, f_cb, None) == 0
    try:
        s = B.AmgSolver(A.rowptr, A.col, A.val)
        csr_bytes = 12 * A.nnz + 4 * (A.n + 1)
        held = sum(live.values())
        # the whole hierarchy (operator complexity ~2.5, CSR + tile blobs + vectors) lives in torch's allocator
        assert held > 3 * csr_bytes and total[0] > held
        assert torch.cuda.memory_allocated() - base >= held
        x, info = s.solve(b, 1e-8, 200)
        assert info.status == 0
        assert np.linalg.norm(b - A.to_scipy() @ x.cpu().numpy()) <= 1e-8 * np.linalg.norm(b)
        # a handle keeps the allocator it was created with, whatever is installed later
        assert lib.amg_set_allocator(None, None, None) == 0
        lam, _ = s.solve_transpose(x, 1e-8, 200)
        s.grad_values(torch.stack([lam, lam]), torch.stack([x, x]))  # grows the interleave scratch
        assert sum(live.values()) > held
        s.close()
        assert not live and freed_unknown[0] == 0  # everything went back through the hook
    finally:
        lib.amg_set_allocator(None, None, None)
    # a handle created now uses the stream-ordered pool again
    s = B.AmgSolver(A.rowptr, A.col, A.val)
    n_before = total[0]
    s.solve(b, 1e-8, 200)
    s.close()
    assert total[0] == n_before


def test_info_null_returns_without_waiting_and_is_stream_ordered(B):
    A = inputs.config_matrix(3, 40)
    b = torch.as_tensor(inputs.config_rhs(3, A.n)).cuda()
    s = B.AmgSolver(A.rowptr, A.col, A.val)
    try:
        x_ref, info = s.solve(b, 1e-8, 500)
        st = torch.cuda.Stream()
        x = torch.zeros_like(b)
        with torch.cuda.stream(st):
            rc = B.load_library().amg_solve(s.h, C.c_void_p(b.data_ptr()), C.c_void_p(x.data_ptr()), C.c_double(1e-8),
                                            C.c_int32(500), None, C.c_void_p(st.cuda_stream))
            assert rc == 0
            y = x * 2.0  # enqueued behind the solve on the same stream
        st.synchronize()
        assert torch.equal(x, x_ref) and torch.equal(y, x_ref * 2.0)
        # aggregates through the caller's stream
        with torch.cuda.stream(st):
            agg = s.aggregates(0)
        st.synchronize()
        assert torch.equal(agg, s.aggregates(0))
    finally:
        s.close()


def test_distinct_handles_on_distinct_threads_and_streams(B):
    """Header: "distinct handles may be used concurrently from distinct host threads on distinct streams"."""
    mats = [inputs.config_matrix(3, 36), inputs.config_matrix(4, 30), inputs.config_matrix(2, 200)]
    rhs = [inputs.rhs_uniform(A.n, 900 + i) for i, A in enumerate(mats)]
    ref = []
    for A, b in zip(mats, rhs):
        s = B.AmgSolver(A.rowptr, A.col, A.val)
        x, info = s.solve(b, 1e-8, 1000)
        ref.append((x.clone(), info.iterations))
        s.close()
    out, errs = [None] * len(mats), []

    def work(i):
        try:
            torch.cuda.set_device(0)
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                A, b = mats[i], rhs[i]
                for _ in range(3):  # setup, solve, destroy, several times while the others do the same
                    s = B.AmgSolver(A.rowptr, A.col, A.val)
                    x, info = s.solve(b, 1e-8, 1000)
                    out[i] = (x.clone(), info.iterations)
                    s.close()
            st.synchronize()
        except Exception as e:  # noqa: BLE001
            errs.append(repr(e))

    ts = [threading.Thread(target=work, args=(i,)) for i in range(len(mats))]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not errs, errs
    for (x, it), (xr, itr) in zip(out, ref):
        assert it == itr and torch.equal(x, xr)  # bitwise: no cross-talk between handles


@pytest.mark.parametrize("krylov", [0, 1])
def test_device_side_loop_equals_host_controlled_loop(B, krylov):
    """use_while = 1 (default): the Krylov loop is one graph with a conditional WHILE node; use_while = 0: the
    iteration graph replayed under host control with a one-behind poll.  Same kernels in the same order: bitwise
    equal solutions and counts; the device-side loop launches no surplus iteration."""
    A = inputs.config_matrix(3, 40)
    b = inputs.config_rhs(3, A.n)
    res = {}
    for w in (1, 0):
        s = B.AmgSolver(A.rowptr, A.col, A.val, use_while=w)
        x, info = s.solve(b, 1e-8, 500, krylov)
        res[w] = (x.clone(), info.iterations, info.rel_residual, B.amg_get_last_launches(s.h))
        x3, i3 = s.solve(b, 1e-30, 3, krylov)          # maxit stop inside the device-side loop
        assert i3.status == 1 and i3.iterations == 3
        x0, i0 = s.solve(np.zeros(A.n), 1e-8, 500, krylov)  # zero right-hand side: the loop body exits at once
        assert i0.status == 0 and i0.iterations == 0 and not bool(x0.any())
        s.close()
    assert torch.equal(res[1][0], res[0][0]) and res[1][1] == res[0][1] and res[1][2] == res[0][2]
    assert res[1][3] < res[0][3]  # one surplus look-ahead iteration less
