"""The C-ABI library builds for sm_100a without a GPU, loads, and exports every function that
include/pf.h declares (no compute calls here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "pf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pf_[a-z_0-9]+)\s*\(", text)))


def test_library_builds_and_exports_header_symbols():
    from paper_1711_04060_b200 import build
    lib = ctypes.CDLL(build.build())
    names = declared_functions()
    assert "pf_grid_create" in names and "pf_solve_linear" in names and "pf_solve_pf" in names
    for name in names:
        assert hasattr(lib, name), f"{name} declared in include/pf.h but not exported"


def test_binding_lists_the_same_entry_points():
    from paper_1711_04060_b200 import pf
    assert sorted(pf.EXPORTS) == declared_functions()
    for name in pf.EXPORTS:
        if name not in ("pf_last_error", "pf_grid_linear_iters"):
            assert hasattr(pf, name), name


def test_no_device_is_an_error_not_a_fallback():
    import torch
    if torch.cuda.is_available():
        return
    from paper_1711_04060_b200 import pf
    lib = pf.load()
    handle = ctypes.c_void_p()
    bc = pf.pf_bc()
    eps = (ctypes.c_double * 27)(*([1.0] * 27))
    rc = lib.pf_grid_create(ctypes.byref(handle), 3, 3, 3, 0.5, ctypes.cast(eps, ctypes.c_void_p), None, 0,
                            ctypes.byref(bc), None)
    assert rc == pf.PF_ERR_CUDA and not handle.value
    assert b"no CPU fallback" in lib.pf_last_error(None)
