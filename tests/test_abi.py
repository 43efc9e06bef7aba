"""The C-ABI library builds for sm_100a without a GPU, loads, and exports every function that
include/pf.h declares (no compute calls here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions(headers=None):
    """Functions declared by include/*.h (pf.h: the boundary; pf_debug.h: test and bench introspection)."""
    inc = os.path.join(ROOT, "include")
    names = set()
    for h in headers or sorted(f for f in os.listdir(inc) if f.endswith(".h")):
        text = open(os.path.join(inc, h)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names |= set(re.findall(r"\b(pf_[a-z_0-9]+)\s*\(", text))
    return sorted(names)


def test_library_builds_and_exports_header_symbols():
    from paper_1711_04060_b200 import build
    lib = ctypes.CDLL(build.build())
    names = declared_functions()
    assert "pf_grid_create" in names and "pf_solve_linear" in names and "pf_solve_pf" in names
    for name in names:
        assert hasattr(lib, name), f"{name} declared in include/*.h but not exported"


def test_boundary_header_stays_small():
    """include/pf.h is the boundary of SURVEY.md section 8(b) plus the widened rows (Omega_f nodes, the host-buffer
    solve, the pointwise row alone, histories); everything that only tests and bench need lives in pf_debug.h."""
    boundary = declared_functions(["pf.h"])
    for name in ("pf_grid_create", "pf_grid_workspace_bytes", "pf_grid_set_workspace", "pf_grid_set_option",
                 "pf_solve_linear", "pf_solve_pf", "pf_grid_destroy", "pf_last_error"):
        assert name in boundary
    assert len(boundary) <= 16, boundary
    for name in ("pf_grid_copy_array", "pf_grid_code_layout", "pf_coop_plan", "pf_launch_count", "pf_grid_fault_repeats"):
        assert name not in boundary and name in declared_functions(["pf_debug.h"])


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


def test_product_package_never_touches_the_oracle():
    """The oracle is test infrastructure: nothing under paper_1711_04060_b200/ (Python or CUDA sources) may import,
    include, load or name anything under oracle/ -- and the oracle's sources do not name the product either."""
    pkg = os.path.join(ROOT, "paper_1711_04060_b200")
    # statements that could pull the oracle in: Python imports, C includes, dlopen/CDLL/open/subprocess of its files
    stmt = re.compile(r"^\s*(import|from)\s+\S*oracle|^\s*#\s*include\s*[<\"][^>\"]*oracle|"
                      r"(CDLL|dlopen|open|Popen|run|import_module|__import__)\s*\([^)]*oracle", re.I)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if not f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                continue
            path = os.path.join(dirpath, f)
            for no, line in enumerate(open(path, encoding="utf-8"), 1):
                assert not stmt.search(line), f"{path}:{no} pulls in the oracle: {line.strip()}"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f), encoding="utf-8").read()
            assert "import paper_1711_04060_b200" not in text and "from paper_1711_04060_b200" not in text
            assert "csrc/" not in text.replace("(paper_1711_04060_b200/csrc)", "")


def test_no_alloc_entry_point_source_allocates_nothing():
    """include/pf_noalloc.h promises an entry point without cudaMalloc / cudaFree or allocating library calls, with its
    scratch in a file-scope __device__ array whose device address comes from cudaGetSymbolAddress."""
    src = open(os.path.join(ROOT, "paper_1711_04060_b200", "csrc", "pf_noalloc.cu")).read()
    code = "\n".join(line.split("//")[0] for line in src.splitlines())
    for banned in ("cudaMalloc", "cudaFree", "cudaHostAlloc", "cudaMallocAsync", "new ", "std::vector", "malloc("):
        assert banned not in code, banned
    assert re.search(r"static\s+__device__\s+__align__\(256\)", code) and "cudaGetSymbolAddress" in code
    hdr = open(os.path.join(ROOT, "include", "pf_noalloc.h")).read()
    assert "PF_NOALLOC_MAX_N" in hdr and "race" in hdr
