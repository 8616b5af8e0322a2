"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/*.h declares, validates
arguments, and fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes as C
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    names = set()
    for h in ("hqmc.h", "hqmc_tuning.h"):
        txt = open(os.path.join(ROOT, "include", h)).read()
        txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
        names |= set(re.findall(r"\b(hqmc_[a-z_A-Z0-9]+)\s*\(", txt))
    return sorted(names)


def test_hot_path_header_has_no_tuning_knobs():
    """include/hqmc.h lists the operations of the method, their batched / estimator / host forms and nothing else."""
    txt = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "hqmc.h")).read(), flags=re.S)
    assert not re.findall(r"\bhqmc_(set_(?!precond|theta)[a-z_]+|reset_stats|get_kernel_stats)\s*\(", txt)


def test_library_loads_and_exports_every_declared_symbol():
    from paper_2508_16298_b200 import hqmc
    names = _declared()
    assert len(names) >= 20
    lib = C.CDLL(hqmc.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(hqmc.SYMBOLS) == names
    assert hqmc.version() >= 100
    lib.hqmc_strerror.restype = C.c_char_p
    assert lib.hqmc_strerror(-3) == b"CG did not converge within max_iter"


def test_argument_validation_and_no_cpu_fallback():
    from paper_2508_16298_b200 import hqmc
    lib = C.CDLL(hqmc.LIB_PATH)
    ctx = C.c_void_p()
    bad = hqmc._Params(5, 8, 0.1, 1.0, 1.0, 1.0, 1, 6, 0)       # odd L
    assert lib.hqmc_create(C.byref(bad), None, C.byref(ctx)) == hqmc.HQMC_EINVAL
    bad = hqmc._Params(4, 8, 0.1, 1.0, 1.0, 1.0, 1, 8, 0)       # W >= Ntau
    assert lib.hqmc_create(C.byref(bad), None, C.byref(ctx)) == hqmc.HQMC_EINVAL
    assert lib.hqmc_apply_M(None, None, None) == hqmc.HQMC_EINVAL
    for fn in (lib.hqmc_slab_dot, lib.hqmc_slab_axpy, lib.hqmc_slab_dupdate, lib.hqmc_slab_scale, lib.hqmc_slab_sum_rows,
               lib.hqmc_slab_field_axpy, lib.hqmc_slab_action_boson, lib.hqmc_set_cg_persistent):
        fn.argtypes = None
    assert lib.hqmc_slab_dot(None, None, None, C.c_longlong(0), None) == hqmc.HQMC_EINVAL
    assert lib.hqmc_slab_action_boson(None, 0, 1, None) == hqmc.HQMC_EINVAL
    assert lib.hqmc_set_cg_persistent(None, 0) == hqmc.HQMC_EINVAL
    if not torch.cuda.is_available():
        ok = hqmc._Params(4, 8, 0.1, 1.0, 1.0, 1.0, 1, 6, 0)
        assert lib.hqmc_create(C.byref(ok), None, C.byref(ctx)) == hqmc.HQMC_ECUDA
        with pytest.raises(hqmc.HqmcError):
            hqmc.HQMC(4, 8, device="cpu")


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2508_16298_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".inl")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU oracle", "").lower() or f == "inputs.py", f
