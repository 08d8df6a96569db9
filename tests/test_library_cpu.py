"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/chfsi.h declares,
and validates arguments without touching a GPU.  No compute calls here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2605_30128_b200 import build, binding
    build.build()                                   # nvcc cross-compiles sm_100a without a GPU
    binding.lib()
    return binding


def test_header_symbols_all_exported(B):
    hdr = open(os.path.join(ROOT, "include", "chfsi.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(chfsi_[a-zA-Z0-9_]+)\s*\(", hdr))
    assert {"chfsi_mesh_create", "chfsi_ham_set", "chfsi_apply_H", "chfsi_cheb_filter"} <= declared
    lib = B.lib()
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in chfsi.h but not exported"
    assert declared == set(B.EXPORTS)


def test_version_and_error_strings(B):
    assert "sm_100a" in B.chfsi_version()
    assert isinstance(B.lib().chfsi_last_error(), bytes)


def test_argument_validation_without_gpu(B):
    lib = B.lib()
    h = C.c_void_p()
    assert lib.chfsi_mesh_create(0, 1, 1, 1.0, 1.0, 1.0, 2, None, 0, C.byref(h)) == B.EINVAL
    assert lib.chfsi_mesh_create(1, 1, 1, -1.0, 1.0, 1.0, 2, None, 0, C.byref(h)) == B.EINVAL
    assert lib.chfsi_mesh_create(1, 1, 1, 1.0, 1.0, 1.0, 0, None, 0, C.byref(h)) == B.EINVAL
    assert lib.chfsi_mesh_create(1, 1, 1, 1.0, 1.0, 1.0, 9, None, 0, C.byref(h)) == B.EUNSUPPORTED
    assert lib.chfsi_mesh_create(1, 1, 1, 1.0, 1.0, 1.0, 2, None, 0, None) == B.EINVAL
    assert b"p" in lib.chfsi_last_error() or lib.chfsi_last_error() != b""
    n = C.c_longlong()
    assert lib.chfsi_mesh_num_nodes(None, C.byref(n)) == B.EINVAL
    assert lib.chfsi_apply_H(None, 0, 1, None, 1, None, 1, None, 0, None) == B.EINVAL
    assert lib.chfsi_cheb_filter(None, 0, 1, 4, 0.0, 1.0, -1.0, 1, 0, None, 1, None, None, 1, None, 0, None) == B.EINVAL
    assert lib.chfsi_mesh_destroy(None) == B.OK


def test_no_cpu_fallback_in_product_path():
    """The package never imports the oracle; the binding raises if the shared library is absent."""
    pkg = os.path.join(ROOT, "paper_2605_30128_b200")
    for fn in os.listdir(pkg):
        if fn.endswith(".py"):
            src = open(os.path.join(pkg, fn)).read()
            assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), fn
            assert "fe_oracle" not in src, fn
    from paper_2605_30128_b200 import binding
    old, binding._lib, path = binding._lib, None, binding.LIB_PATH
    try:
        binding.LIB_PATH = path + ".missing"
        with pytest.raises(ImportError):
            binding.lib()
    finally:
        binding.LIB_PATH, binding._lib = path, old
