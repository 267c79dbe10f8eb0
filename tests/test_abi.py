"""CPU-side checks of the boundary: libtbsma.so builds/loads and exports every symbol that
include/tbsma.h declares; without a GPU every entry point fails loudly (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_1311_3890_b200 import build
    return build.build()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "tbsma.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tbsma_[a-z_]+)\s*\(", text)))


def test_header_declares_the_boundary_calls():
    syms = declared_symbols()
    for name in ("tbsma_create", "tbsma_destroy", "tbsma_set_system", "tbsma_build_cells",
                 "tbsma_build_neighbors", "tbsma_compute", "tbsma_md_step", "tbsma_md_run",
                 "tbsma_md_run_host", "tbsma_get_neighbors", "tbsma_status", "tbsma_strerror"):
        assert name in syms


def test_library_exports_every_declared_symbol(libpath):
    lib = ctypes.CDLL(libpath)
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in tbsma.h but not exported"


def test_binding_lists_the_same_symbols(libpath):
    from paper_1311_3890_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()
    assert binding.version().startswith("tbsma-b200")
    assert binding.strerror(-1) == "invalid argument"


def test_no_cpu_fallback(libpath):
    import torch
    from paper_1311_3890_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(binding.TbsmaError) as e:
        binding.Context()
    assert e.value.code == binding.ECUDA


def test_invalid_arguments_are_rejected(libpath):
    from paper_1311_3890_b200 import binding
    L = binding.lib()
    h = ctypes.c_void_p()
    p = binding.au_params()
    assert L.tbsma_create(None, 7.0, 0.3, ctypes.byref(h)) == binding.EINVAL
    assert L.tbsma_create(ctypes.byref(p), -1.0, 0.3, ctypes.byref(h)) == binding.EINVAL
    assert L.tbsma_destroy(None) == binding.EINVAL
    assert L.tbsma_launch_count(None) == 0


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1311_3890_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "tbsma_oracle" not in src and "liboracle" not in src, f
    orc = open(os.path.join(ROOT, "oracle", "tbsma_oracle.c")).read()
    assert "tbsma.h" not in re.sub(r"/\*.*?\*/", "", orc, flags=re.S)
