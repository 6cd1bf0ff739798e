"""ctypes loader for the CPU oracle (TEST INFRASTRUCTURE — see oracle/amg_oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  Nothing under paper_2606_09001_b200/ imports it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "amg_oracle.cpp")
_HDR = os.path.join(_HERE, "amg_oracle.h")
_LIB = os.path.join(_HERE, "libamg_oracle.so")


def build(force: bool = False) -> str:
    """g++ -O2 -fopenmp the oracle into oracle/libamg_oracle.so (rebuilt when sources change)."""
    if not force and os.path.exists(_LIB):
        if os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)):
            return _LIB
    # -ffp-contract=off: no FMA contraction, the arithmetic is exactly what the source says
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-o", _LIB + ".tmp", _SRC]
    subprocess.run(cmd, check=True)
    os.replace(_LIB + ".tmp", _LIB)
    return _LIB


class Options(C.Structure):
    _fields_ = [("pre_sweeps", C.c_int32), ("post_sweeps", C.c_int32), ("smoother", C.c_int32),
                ("coarse_max_rows", C.c_int32), ("max_levels", C.c_int32),
                ("max_match_rounds", C.c_int32), ("omega", C.c_double),
                ("strong_beta", C.c_double), ("coarse_scale", C.c_double),
                ("hash_seed", C.c_uint64), ("agg_passes", C.c_int32), ("symmetric", C.c_int32),
                ("hierarchy_fp32", C.c_int32), ("pad0", C.c_int32), ("cheby_ratio", C.c_double)]


class Info(C.Structure):
    _fields_ = [("iterations", C.c_int32), ("status", C.c_int32), ("rel_residual", C.c_double),
                ("b_norm", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_options_default.restype = None
        _lib.oracle_destroy.restype = None
        _lib.oracle_set_threads.restype = None
    return _lib


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle: {what} failed with code {rc}")


def set_threads(n: int):
    lib().oracle_set_threads(C.c_int(int(n)))


def get_threads() -> int:
    return int(lib().oracle_get_threads())


def default_options(**kw) -> Options:
    o = Options()
    lib().oracle_options_default(C.byref(o))
    for k, v in kw.items():
        if not hasattr(o, k):
            raise AttributeError(k)
        setattr(o, k, v)
    return o


class Oracle:
    """One hierarchy (O-1) and the solves / gradients on it (O-4 … O-8)."""

    def __init__(self, rowptr, col, val, aggregates=None, **opts):
        self.rowptr, self.col, self.val = _i32(rowptr), _i32(col), _f64(val)
        self.n = len(self.rowptr) - 1
        self.opt = default_options(**opts)
        self._h = C.c_void_p()
        L = lib()
        if aggregates is None:
            rc = L.oracle_setup(C.byref(self._h), C.c_int32(self.n), _p(self.rowptr), _p(self.col),
                                _p(self.val), C.byref(self.opt))
        else:
            aggs = [_i32(a) for a in aggregates]
            arr = (C.c_void_p * max(len(aggs), 1))(*[a.ctypes.data for a in aggs])
            rc = L.oracle_setup_with_aggregates(C.byref(self._h), C.c_int32(self.n), _p(self.rowptr),
                                                _p(self.col), _p(self.val), C.byref(self.opt),
                                                C.c_int32(len(aggs)), arr)
        _check(rc, "setup")

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def num_levels(self) -> int:
        return int(lib().oracle_num_levels(self._h))

    def level_info(self, level):
        r, z = C.c_int32(), C.c_int32()
        _check(lib().oracle_level_info(self._h, C.c_int32(level), C.byref(r), C.byref(z)), "level_info")
        return r.value, z.value

    def aggregates(self, level) -> np.ndarray:
        rows, _ = self.level_info(level)
        a = np.empty(rows, dtype=np.int32)
        _check(lib().oracle_get_aggregates(self._h, C.c_int32(level), _p(a)), "get_aggregates")
        return a

    def level_csr(self, level):
        rows, nnz = self.level_info(level)
        rp = np.empty(rows + 1, dtype=np.int32)
        cl = np.empty(nnz, dtype=np.int32)
        vl = np.empty(nnz, dtype=np.float64)
        _check(lib().oracle_get_level_csr(self._h, C.c_int32(level), _p(rp), _p(cl), _p(vl)), "level_csr")
        return rp, cl, vl

    def dinv(self, level) -> np.ndarray:
        rows, _ = self.level_info(level)
        d = np.empty(rows)
        _check(lib().oracle_get_dinv(self._h, C.c_int32(level), _p(d)), "get_dinv")
        return d

    def match_rounds(self, level) -> int:
        return int(lib().oracle_match_rounds(self._h, C.c_int32(level)))

    def spmv(self, level, x) -> np.ndarray:
        x = _f64(x)
        y = np.empty(self.level_info(level)[0])
        _check(lib().oracle_spmv(self._h, C.c_int32(level), _p(x), _p(y)), "spmv")
        return y

    def smooth(self, level, b, x) -> np.ndarray:
        b, x = _f64(b), _f64(x)
        out = np.empty_like(x)
        _check(lib().oracle_smooth(self._h, C.c_int32(level), _p(b), _p(x), _p(out)), "smooth")
        return out

    def residual_restrict(self, level, b, x) -> np.ndarray:
        b, x = _f64(b), _f64(x)
        rc = np.empty(self.level_info(level + 1)[0])
        _check(lib().oracle_residual_restrict(self._h, C.c_int32(level), _p(b), _p(x), _p(rc)),
               "residual_restrict")
        return rc

    def vcycle(self, r, level=0) -> np.ndarray:
        r = _f64(r)
        z = np.empty_like(r)
        _check(lib().oracle_vcycle(self._h, C.c_int32(level), _p(r), _p(z)), "vcycle")
        return z

    def vcycle_transpose(self, r, level=0) -> np.ndarray:
        r = _f64(r)
        z = np.empty_like(r)
        _check(lib().oracle_vcycle_transpose(self._h, C.c_int32(level), _p(r), _p(z)), "vcycle_transpose")
        return z

    def solve(self, b, rtol=1e-8, maxit=1000, krylov=0, precond=1):
        b = _f64(b)
        x = np.empty_like(b)
        info = Info()
        _check(lib().oracle_solve(self._h, _p(b), _p(x), C.c_double(rtol), C.c_int32(maxit),
                                  C.c_int32(krylov), C.c_int32(precond), C.byref(info)), "solve")
        return x, info

    def solve_transpose(self, g, rtol=1e-8, maxit=1000, krylov=0, precond=1, symmetric=1):
        g = _f64(g)
        lam = np.empty_like(g)
        info = Info()
        _check(lib().oracle_solve_transpose(self._h, _p(g), _p(lam), C.c_double(rtol),
                                            C.c_int32(maxit), C.c_int32(krylov), C.c_int32(precond),
                                            C.c_int32(symmetric), C.byref(info)), "solve_transpose")
        return lam, info

    def residual_history(self) -> np.ndarray:
        """||r_k|| / ||b||, k = 1 … iterations, of the last solve / solve_transpose on this handle."""
        m = int(lib().oracle_get_residual_history(self._h, None, C.c_int32(0)))
        out = np.empty(max(m, 0))
        if m > 0:
            lib().oracle_get_residual_history(self._h, _p(out), C.c_int32(m))
        return out

    def grad_values(self, lam, x, accumulate_into=None) -> np.ndarray:
        """lam, x: arrays of shape (nrhs, n) (row b = vector b) or (n,)."""
        lam = _f64(np.atleast_2d(lam))
        x = _f64(np.atleast_2d(x))
        nrhs = lam.shape[0]
        nnz = int(self.rowptr[-1])
        if accumulate_into is None:
            gA = np.empty(nnz)
            acc = 0
        else:
            gA = _f64(accumulate_into)
            acc = 1
        _check(lib().oracle_grad_values(self._h, _p(lam), _p(x), C.c_int32(nrhs),
                                        C.c_int64(self.n), _p(gA), C.c_int32(acc)), "grad_values")
        return gA


def cheby_weights(k: int, ratio: float) -> np.ndarray:
    """Sweep weights of the Chebyshev-accelerated L1-Jacobi smoother (smoother = 2)."""
    w = np.empty(k)
    _check(lib().oracle_cheby_weights(C.c_int32(k), C.c_double(ratio), _p(w)), "cheby_weights")
    return w


def aggregate(rowptr, col, val, beta=0.25, salt=0, max_rounds=0, mode=0, symmetric=1):
    """O-2 on its own.  Returns (match, agg, nc, rounds).  mode 0 handshake, 1 greedy.
    symmetric = 0: the matching runs on (A + A^T)/2 (A1, nonsymmetric case)."""
    rowptr, col, val = _i32(rowptr), _i32(col), _f64(val)
    n = len(rowptr) - 1
    match = np.empty(n, dtype=np.int32)
    agg = np.empty(n, dtype=np.int32)
    nc, rounds = C.c_int32(), C.c_int32()
    _check(lib().oracle_aggregate(C.c_int32(n), _p(rowptr), _p(col), _p(val), C.c_double(beta),
                                  C.c_uint64(salt), C.c_int32(max_rounds), C.c_int32(mode),
                                  C.c_int32(symmetric), _p(match), _p(agg), C.byref(nc), C.byref(rounds)), "aggregate")
    return match, agg, nc.value, rounds.value


def galerkin(rowptr, col, val, agg, nc):
    """O-3 on its own.  Returns the coarse CSR triple."""
    rowptr, col, val, agg = _i32(rowptr), _i32(col), _f64(val), _i32(agg)
    n = len(rowptr) - 1
    cnnz = C.c_int32()
    _check(lib().oracle_galerkin(C.c_int32(n), _p(rowptr), _p(col), _p(val), _p(agg), C.c_int32(nc),
                                 None, None, None, C.byref(cnnz)), "galerkin(size)")
    crp = np.empty(nc + 1, dtype=np.int32)
    ccl = np.empty(cnnz.value, dtype=np.int32)
    cvl = np.empty(cnnz.value, dtype=np.float64)
    _check(lib().oracle_galerkin(C.c_int32(n), _p(rowptr), _p(col), _p(val), _p(agg), C.c_int32(nc),
                                 _p(crp), _p(ccl), _p(cvl), C.byref(cnnz)), "galerkin")
    return crp, ccl, cvl
