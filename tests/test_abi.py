"""CPU-only checks of the boundary: libbkr.so builds for sm_100a, loads, and exports every symbol that
include/bkr.h declares (no compute calls without a GPU); the product path has no CPU fallback and never
imports the oracle."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1710_09745_b200 import build
    return build.build()


def header_functions():
    text = open(os.path.join(ROOT, "include", "bkr.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(bkr_[a-zA-Z0-9_]+)\s*\(", text)))


def test_header_declares_the_hot_path_calls():
    names = header_functions()
    for want in ("bkr_load_links", "bkr_dslash", "bkr_apply_M", "bkr_gram", "bkr_block_axpy", "bkr_solve_block",
                 "bkr_solve_cg", "bkr_cholesky_upper", "bkr_hpd_inverse"):
        assert want in names


def test_library_exports_every_declared_symbol(libpath):
    L = ctypes.CDLL(libpath)
    for name in header_functions():
        assert hasattr(L, name), name


def test_binding_lists_every_declared_symbol(libpath):
    from paper_1710_09745_b200 import binding
    assert sorted(binding.SYMBOLS) == header_functions()
    L = binding.lib()
    assert binding.version().startswith("libbkr")
    assert L.bkr_strerror(binding.EBREAKDOWN).decode().lower().startswith("cholesky")


def test_error_codes_without_gpu(libpath):
    """argument errors are detected before any CUDA call."""
    from paper_1710_09745_b200 import binding
    L = binding.lib()
    h = ctypes.c_void_p()
    bad = (ctypes.c_int * 4)(4, 4, 5, 4)  # odd extent
    assert L.bkr_create(ctypes.byref(h), bad, 0, None) == binding.EINVAL
    small = (ctypes.c_int * 4)(2, 4, 4, 4)  # extent < 4
    assert L.bkr_create(ctypes.byref(h), small, 0, None) == binding.EINVAL
    assert L.bkr_destroy(None) == binding.EINVAL
    assert L.bkr_field_bytes(None, 4, 0) == 0


def test_no_cpu_fallback():
    import torch
    from paper_1710_09745_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        binding.Context((4, 4, 4, 4))


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1710_09745_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", src, flags=re.M), f
                assert "liboracle" not in src and "oracle.c" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "oracle.c")).read()
    assert not re.search(r"^\s*(import|from)\s+paper_1710_09745_b200", osrc, flags=re.M)
    assert not re.search(r"#\s*include\s*[\"<][^\">]*(bkr|csrc)", osrc)
