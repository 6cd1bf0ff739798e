"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports
every symbol include/amg_b200.h declares; the binding's struct layouts match the header; the
product path fails loudly without a GPU; nothing under the package imports the oracle."""
import ctypes as C
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "amg_b200.h")


def declared_symbols():
    src = open(HEADER).read()
    return sorted(set(re.findall(r"AMG_API\s+(?:const\s+)?[\w\*]+\s+\*?\s*(amg_\w+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    syms = declared_symbols()
    for required in ["amg_setup", "amg_solve", "amg_solve_transpose", "amg_grad_values", "amg_destroy",
                     "amg_solve_batched", "amg_apply_preconditioner", "amg_get_aggregates"]:
        assert required in syms
    assert len(syms) >= 20


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2606_09001_b200 import binding, build

    path = build.build()
    assert os.path.exists(path)
    lib = C.CDLL(path)  # loads without a GPU (cudart is linked statically; no device call at load)
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in amg_b200.h but not exported"
    assert sorted(binding.EXPORTS) == declared_symbols()


def test_struct_layouts_and_defaults():
    from paper_2606_09001_b200 import binding

    o = binding.amg_options_default()
    assert o.struct_size == C.sizeof(binding.amg_options) == 112
    assert (o.krylov, o.symmetric, o.agg_passes, o.pre_sweeps, o.post_sweeps, o.smoother) == (0, -1, 1, 2, 2, 0)
    assert (o.coarse_max_rows, o.max_levels, o.max_match_rounds) == (64, 32, 0)
    assert o.strong_beta == 0.25 and o.coarse_scale == 1.0 and abs(o.omega - 2 / 3) < 1e-16
    assert C.sizeof(binding.amg_info) == 24
    assert C.sizeof(binding.amg_setup_stats) == 48


def test_argument_errors_without_gpu():
    from paper_2606_09001_b200 import binding

    lib = binding.load_library()
    h = C.c_void_p()
    # null pointers are rejected before any CUDA call
    st = lib.amg_setup(C.byref(h), C.c_int64(4), C.c_int64(4), None, None, None, None, None)
    assert st == 1 and not h.value
    assert b"null" in lib.amg_last_error(None)
    st = lib.amg_setup(C.byref(h), C.c_int64(1 << 31), C.c_int64(4), C.c_void_p(8), C.c_void_p(8), C.c_void_p(8),
                       None, None)
    assert st == 7  # AMG_ERR_UNSUPPORTED: int32 indices
    assert lib.amg_solve(None, None, None, C.c_double(1e-8), C.c_int32(1), None, None) == 1
    assert lib.amg_destroy(None) == 0


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_product_path_fails_loudly_without_gpu():
    import numpy as np

    from paper_2606_09001_b200 import binding, inputs

    A = inputs.poisson_csr((4, 4))
    with pytest.raises(RuntimeError):
        binding.AmgSolver(A.rowptr, A.col, A.val)
    with pytest.raises(TypeError):  # CPU tensors are refused: there is no CPU fallback
        binding.amg_setup(A.n, A.nnz, torch.as_tensor(A.rowptr), torch.as_tensor(A.col), torch.as_tensor(A.val))
    assert np.all(np.diff(A.rowptr) > 0)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_09001_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "amg_oracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "amg_oracle.cpp")).read()
    assert "amg_b200.h" not in osrc and "csrc" not in osrc
