"""Thin ctypes binding of libamg_b200.so (include/amg_b200.h): argument marshalling only.

Every function has the name and argument order of its C entry point; tensors are torch CUDA
tensors (device memory owned by torch), the stream is torch's current stream.  There is no
CPU path: if the library is missing or no GPU is present the calls fail loudly.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libamg_b200.so")

AMG_OK = 0
STATUS_NAMES = ["AMG_OK", "AMG_ERR_INVALID_ARG", "AMG_ERR_BAD_CSR", "AMG_ERR_CUDA", "AMG_ERR_OOM",
                "AMG_ERR_COARSE_SINGULAR", "AMG_ERR_COARSEN_STALL", "AMG_ERR_UNSUPPORTED"]
AMG_CONVERGED, AMG_MAXIT, AMG_BREAKDOWN, AMG_NONFINITE = 0, 1, 2, 3

EXPORTS = ["amg_options_default", "amg_set_allocator", "amg_setup", "amg_setup_with_aggregates", "amg_resetup_values",
           "amg_destroy", "amg_solve", "amg_solve_ex", "amg_solve_transpose", "amg_solve_batched",
           "amg_solve_host", "amg_grad_values", "amg_grad_values_noalloc", "amg_apply_preconditioner", "amg_get_num_levels",
           "amg_get_level_info", "amg_get_aggregates", "amg_get_level_csr", "amg_get_setup_stats",
           "amg_get_level_path", "amg_get_symmetric", "amg_get_residual_history", "amg_write_report", "amg_get_algorithmic_bytes", "amg_get_last_launches", "amg_level_op", "amg_last_error",
           "amg_cache_create", "amg_cache_get", "amg_cache_stats", "amg_cache_destroy"]


class amg_options(C.Structure):
    _fields_ = [("struct_size", C.c_int32), ("krylov", C.c_int32), ("symmetric", C.c_int32),
                ("agg_passes", C.c_int32),
                ("pre_sweeps", C.c_int32), ("post_sweeps", C.c_int32), ("smoother", C.c_int32),
                ("coarse_max_rows", C.c_int32), ("max_levels", C.c_int32),
                ("max_match_rounds", C.c_int32), ("force_generic", C.c_int32),
                ("use_graph", C.c_int32), ("tail_dense_rows", C.c_int32), ("use_pdl", C.c_int32),
                ("split_prolong_rows", C.c_int32), ("use_while", C.c_int32),
                ("omega", C.c_double),
                ("strong_beta", C.c_double), ("coarse_scale", C.c_double), ("hash_seed", C.c_uint64),
                ("hierarchy_fp32", C.c_int32), ("value_dict", C.c_int32), ("cheby_ratio", C.c_double)]


class amg_info(C.Structure):
    _fields_ = [("iterations", C.c_int32), ("status", C.c_int32), ("rel_residual", C.c_double),
                ("b_norm", C.c_double)]


class amg_setup_stats(C.Structure):
    _fields_ = [("total_ms", C.c_double), ("aggregate_ms", C.c_double), ("galerkin_ms", C.c_double),
                ("reorder_ms", C.c_double), ("lu_ms", C.c_double), ("match_rounds_max", C.c_int32),
                ("reserved", C.c_int32)]


class AmgError(RuntimeError):
    def __init__(self, status, msg):
        name = STATUS_NAMES[status] if 0 <= status < len(STATUS_NAMES) else str(status)
        super().__init__(f"{name}: {msg}")
        self.status = status


_lib = None


def load_library(build_if_missing: bool = True):
    """dlopen libamg_b200.so (building it in-tree with nvcc first if it is stale or missing)."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing and _build.needs_build():
        _build.build()
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_09001_b200.build`")
    lib = C.CDLL(LIB_PATH)
    for name in EXPORTS:
        fn = getattr(lib, name)  # AttributeError if an export is missing
        fn.restype = C.c_int
    lib.amg_last_error.restype = C.c_char_p
    lib.amg_last_error.argtypes = [C.c_void_p]
    _lib = lib
    return lib


def _ptr(t, dtype):
    if t is None:
        return C.c_void_p(0)
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("expected a CUDA torch tensor")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"expected a contiguous {dtype} tensor, got {t.dtype}")
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _check(status, handle=None):
    if status != AMG_OK:
        msg = load_library().amg_last_error(handle if handle else C.c_void_p(0))
        raise AmgError(status, msg.decode() if msg else "")


# ---- functions with the names of the C entry points ---------------------------------------
def amg_options_default(**overrides) -> amg_options:
    o = amg_options()
    _check(load_library().amg_options_default(C.byref(o)))
    for k, v in overrides.items():
        if not hasattr(o, k):
            raise AttributeError(k)
        setattr(o, k, v)
    return o


def amg_setup(n, nnz, d_rowptr, d_col, d_val, opt=None):
    h = C.c_void_p()
    st = load_library().amg_setup(C.byref(h), C.c_int64(n), C.c_int64(nnz), _ptr(d_rowptr, torch.int32),
                                  _ptr(d_col, torch.int32), _ptr(d_val, torch.float64),
                                  C.byref(opt) if opt is not None else None, _stream())
    _check(st)
    return h


def amg_setup_with_aggregates(n, nnz, d_rowptr, d_col, d_val, opt, d_aggs):
    h = C.c_void_p()
    arr = (C.c_void_p * max(len(d_aggs), 1))(*[a.data_ptr() for a in d_aggs])
    for a in d_aggs:
        _ptr(a, torch.int32)
    st = load_library().amg_setup_with_aggregates(
        C.byref(h), C.c_int64(n), C.c_int64(nnz), _ptr(d_rowptr, torch.int32), _ptr(d_col, torch.int32),
        _ptr(d_val, torch.float64), C.byref(opt) if opt is not None else None, C.c_int32(len(d_aggs)), arr,
        _stream())
    _check(st)
    return h


def amg_resetup_values(h, d_val, keep_aggregates):
    _check(load_library().amg_resetup_values(h, _ptr(d_val, torch.float64), C.c_int32(int(keep_aggregates)), _stream()), h)


def amg_destroy(h):
    if h:
        load_library().amg_destroy(h)


def amg_solve(h, d_b, d_x, rtol, maxit) -> amg_info:
    info = amg_info()
    _check(load_library().amg_solve(h, _ptr(d_b, torch.float64), _ptr(d_x, torch.float64), C.c_double(rtol),
                                    C.c_int32(maxit), C.byref(info), _stream()), h)
    return info


def amg_solve_ex(h, d_b, d_x, rtol, maxit, krylov, precond) -> amg_info:
    info = amg_info()
    _check(load_library().amg_solve_ex(h, _ptr(d_b, torch.float64), _ptr(d_x, torch.float64), C.c_double(rtol),
                                       C.c_int32(maxit), C.c_int32(krylov), C.c_int32(precond), C.byref(info),
                                       _stream()), h)
    return info


def amg_solve_transpose(h, d_g, d_lambda, rtol, maxit) -> amg_info:
    info = amg_info()
    _check(load_library().amg_solve_transpose(h, _ptr(d_g, torch.float64), _ptr(d_lambda, torch.float64),
                                              C.c_double(rtol), C.c_int32(maxit), C.byref(info), _stream()), h)
    return info


def amg_solve_batched(h, transpose, d_B, d_X, nrhs, ld, rtol, maxit):
    infos = (amg_info * max(nrhs, 1))()
    _check(load_library().amg_solve_batched(h, C.c_int32(transpose), _ptr(d_B, torch.float64),
                                            _ptr(d_X, torch.float64), C.c_int32(nrhs), C.c_int64(ld),
                                            C.c_double(rtol), C.c_int32(maxit), infos, _stream()), h)
    return list(infos)[:nrhs]


def amg_solve_host(h, h_b, h_x, rtol, maxit) -> amg_info:
    """h_b, h_x: CPU float64 tensors (pinned for true async copies)."""
    for t in (h_b, h_x):
        if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
            raise TypeError("amg_solve_host expects contiguous CPU float64 tensors")
    info = amg_info()
    _check(load_library().amg_solve_host(h, C.c_void_p(h_b.data_ptr()), C.c_void_p(h_x.data_ptr()),
                                         C.c_double(rtol), C.c_int32(maxit), C.byref(info), _stream()), h)
    return info


def amg_grad_values(h, d_lambda, d_x, nrhs, ld, d_gA, accumulate):
    _check(load_library().amg_grad_values(h, _ptr(d_lambda, torch.float64), _ptr(d_x, torch.float64),
                                          C.c_int32(nrhs), C.c_int64(ld), _ptr(d_gA, torch.float64),
                                          C.c_int32(accumulate), _stream()), h)


def amg_grad_values_noalloc(n, nnz, d_rowptr, d_col, d_lambda, d_x, nrhs, ld, d_gA, accumulate):
    """Handle-free, allocation-free G2 (static device scratch: n * nrhs <= AMG_NOALLOC_MAX_DOUBLES)."""
    _check(load_library().amg_grad_values_noalloc(C.c_int64(n), C.c_int64(nnz), _ptr(d_rowptr, torch.int32),
                                                  _ptr(d_col, torch.int32), _ptr(d_lambda, torch.float64),
                                                  _ptr(d_x, torch.float64), C.c_int32(nrhs), C.c_int64(ld),
                                                  _ptr(d_gA, torch.float64), C.c_int32(accumulate), _stream()))


def amg_apply_preconditioner(h, d_r, d_z):
    _check(load_library().amg_apply_preconditioner(h, _ptr(d_r, torch.float64), _ptr(d_z, torch.float64),
                                                   _stream()), h)


def amg_get_num_levels(h) -> int:
    v = C.c_int32()
    _check(load_library().amg_get_num_levels(h, C.byref(v)), h)
    return v.value


def amg_get_level_info(h, level):
    r, z = C.c_int64(), C.c_int64()
    _check(load_library().amg_get_level_info(h, C.c_int32(level), C.byref(r), C.byref(z)), h)
    return r.value, z.value


def amg_get_aggregates(h, level, d_agg_out):
    _check(load_library().amg_get_aggregates(h, C.c_int32(level), _ptr(d_agg_out, torch.int32), _stream()), h)


def amg_get_residual_history(h):
    """||r_k|| / ||b||, k = 1 .. iterations, of the last solve on this handle (numpy array)."""
    import numpy as np

    cnt = C.c_int32()
    _check(load_library().amg_get_residual_history(h, None, C.c_int32(0), C.byref(cnt), _stream()), h)
    out = np.empty(max(cnt.value, 0))
    if cnt.value > 0:
        _check(load_library().amg_get_residual_history(h, C.c_void_p(out.ctypes.data), C.c_int32(cnt.value),
                                                       C.byref(cnt), _stream()), h)
    return out


def amg_write_report(h, path):
    _check(load_library().amg_write_report(h, C.c_char_p(str(path).encode()), _stream()), h)


def amg_get_symmetric(h) -> int:
    v = C.c_int32()
    _check(load_library().amg_get_symmetric(h, C.byref(v)), h)
    return v.value


def amg_get_level_csr(h, level, d_rowptr, d_col, d_val):
    _check(load_library().amg_get_level_csr(h, C.c_int32(level), _ptr(d_rowptr, torch.int32),
                                            _ptr(d_col, torch.int32), _ptr(d_val, torch.float64), _stream()), h)


def amg_get_setup_stats(h) -> amg_setup_stats:
    s = amg_setup_stats()
    _check(load_library().amg_get_setup_stats(h, C.byref(s)), h)
    return s


def amg_get_level_path(h, level) -> int:
    v = C.c_int32()
    _check(load_library().amg_get_level_path(h, C.c_int32(level), C.byref(v)), h)
    return v.value


def amg_get_algorithmic_bytes(h, which) -> float:
    v = C.c_double()
    _check(load_library().amg_get_algorithmic_bytes(h, C.c_int32(which), C.byref(v)), h)
    return v.value


def amg_get_last_launches(h) -> int:
    v = C.c_int64()
    _check(load_library().amg_get_last_launches(h, C.byref(v)), h)
    return v.value


def amg_level_op(h, level, op, d_in0, d_in1, d_out, reps=1):
    _check(load_library().amg_level_op(h, C.c_int32(level), C.c_int32(op), _ptr(d_in0, torch.float64),
                                       _ptr(d_in1, torch.float64), _ptr(d_out, torch.float64), C.c_int32(reps),
                                       _stream()), h)


def amg_cache_create(capacity):
    c = C.c_void_p()
    _check(load_library().amg_cache_create(C.byref(c), C.c_int32(capacity)))
    return c


def amg_cache_get(c, n, nnz, d_rowptr, d_col, d_val, opt=None, on_hit=1):
    """Returns (handle, hit).  The handle belongs to the cache."""
    h, hit = C.c_void_p(), C.c_int32()
    _check(load_library().amg_cache_get(c, C.c_int64(n), C.c_int64(nnz), _ptr(d_rowptr, torch.int32),
                                        _ptr(d_col, torch.int32), _ptr(d_val, torch.float64),
                                        C.byref(opt) if opt is not None else None, C.c_int32(on_hit), C.byref(h),
                                        C.byref(hit), _stream()))
    return h, hit.value


def amg_cache_stats(c):
    v = [C.c_int64() for _ in range(4)]
    _check(load_library().amg_cache_stats(c, *[C.byref(x) for x in v]))
    return dict(zip(("entries", "hits", "misses", "evictions"), (x.value for x in v)))


def amg_cache_destroy(c):
    if c:
        load_library().amg_cache_destroy(c)


# ---- small convenience wrapper (owns the handle and the device copy of the matrix) ---------
class AmgSolver:
    """amg_setup on construction, amg_destroy on close.  Inputs: numpy or torch arrays."""

    def __init__(self, rowptr, col, val, aggregates=None, device="cuda:0", **options):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_09001_b200 needs a CUDA device (no CPU path)")
        load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        to = lambda a, dt: torch.as_tensor(a).to(dtype=dt).to(self.device).contiguous()
        self.d_rowptr, self.d_col, self.d_val = to(rowptr, torch.int32), to(col, torch.int32), to(val, torch.float64)
        self.n = self.d_rowptr.numel() - 1
        self.nnz = self.d_col.numel()
        self.opt = amg_options_default(**options)
        if aggregates is None:
            self.h = amg_setup(self.n, self.nnz, self.d_rowptr, self.d_col, self.d_val, self.opt)
        else:
            d_aggs = [to(a, torch.int32) for a in aggregates]
            self.h = amg_setup_with_aggregates(self.n, self.nnz, self.d_rowptr, self.d_col, self.d_val, self.opt,
                                               d_aggs)

    def resetup_values(self, val, keep_aggregates=True):
        """Warm resetup on new values of the same pattern (amg_resetup_values)."""
        self.d_val = torch.as_tensor(val).to(dtype=torch.float64).to(self.device).contiguous()
        assert self.d_val.numel() == self.nnz
        amg_resetup_values(self.h, self.d_val, keep_aggregates)

    def close(self):
        if getattr(self, "h", None):
            amg_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _dev(self, a):
        return torch.as_tensor(a).to(dtype=torch.float64).to(self.device).contiguous()

    def residual_history(self):
        return amg_get_residual_history(self.h)

    @property
    def symmetric(self):
        return amg_get_symmetric(self.h)

    @property
    def num_levels(self):
        return amg_get_num_levels(self.h)

    def level_info(self, level):
        return amg_get_level_info(self.h, level)

    def level_path(self, level):
        return amg_get_level_path(self.h, level)

    def aggregates(self, level):
        out = torch.empty(self.level_info(level)[0], dtype=torch.int32, device=self.device)
        amg_get_aggregates(self.h, level, out)
        return out

    def level_csr(self, level):
        rows, nnz = self.level_info(level)
        rp = torch.empty(rows + 1, dtype=torch.int32, device=self.device)
        cl = torch.empty(nnz, dtype=torch.int32, device=self.device)
        vl = torch.empty(nnz, dtype=torch.float64, device=self.device)
        amg_get_level_csr(self.h, level, rp, cl, vl)
        return rp, cl, vl

    def solve(self, b, rtol=1e-8, maxit=1000, krylov=None, precond=1):
        b = self._dev(b)
        x = torch.empty_like(b)
        if krylov is None:
            krylov = self.opt.krylov
        info = amg_solve_ex(self.h, b, x, rtol, maxit, krylov, precond)
        return x, info

    def solve_transpose(self, g, rtol=1e-8, maxit=1000):
        g = self._dev(g)
        lam = torch.empty_like(g)
        info = amg_solve_transpose(self.h, g, lam, rtol, maxit)
        return lam, info

    def grad_values(self, lam, x, accumulate_into=None):
        lam, x = self._dev(lam), self._dev(x)
        nrhs = 1 if lam.dim() == 1 else lam.shape[0]
        gA = accumulate_into if accumulate_into is not None else torch.empty(self.nnz, dtype=torch.float64,
                                                                               device=self.device)
        amg_grad_values(self.h, lam, x, nrhs, self.n, gA, 0 if accumulate_into is None else 1)
        return gA

    def apply_preconditioner(self, r):
        r = self._dev(r)
        z = torch.empty_like(r)
        amg_apply_preconditioner(self.h, r, z)
        return z

    def level_op(self, level, op, in0, in1, out_rows, reps=1):
        in0 = self._dev(in0) if in0 is not None else None
        in1 = self._dev(in1) if in1 is not None else None
        out = torch.empty(out_rows, dtype=torch.float64, device=self.device)
        amg_level_op(self.h, level, op, in0, in1, out, reps)
        return out
