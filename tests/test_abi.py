"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/lbm.h declares; the binding refuses to run without a GPU (no CPU fallback).  No compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2010_11751_b200 import build
    return build.build()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "lbm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = set(re.findall(r"\b(lbm_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


def test_header_symbols_are_exported(lib_path):
    lib = ctypes.CDLL(lib_path)
    names = _declared_symbols()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), "include/lbm.h declares %s but the library does not export it" % n


def test_binding_lists_every_symbol(lib_path):
    from paper_2010_11751_b200 import binding
    assert sorted(binding.SYMBOLS) == _declared_symbols()
    L = binding.load_library()
    assert b"sm_100a" in L.lbm_version()


def test_enums_match_header():
    from paper_2010_11751_b200 import binding
    text = open(os.path.join(ROOT, "include", "lbm.h")).read()
    models = re.search(r"enum \{ LBM_BGK_W2 = 0,(.*?)LBM_NUM_MODELS", text, re.S).group(0)
    order = re.findall(r"LBM_([A-Z0-9_]+)", models)[:-1]
    assert [binding.MODELS[m] for m in order] == list(range(10))
    schemes = re.search(r"enum \{ LBM_2POP_SOA = 0,(.*?)LBM_NUM_SCHEMES", text, re.S).group(0)
    order = re.findall(r"LBM_([A-Z0-9_]+)", schemes)[:-1]
    assert [binding.SCHEMES[s] for s in order] == list(range(6))


def test_no_cpu_fallback(lib_path):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2010_11751_b200 import Lbm
    from paper_2010_11751_b200.binding import LbmError
    with pytest.raises(LbmError):
        Lbm(8, 8, 8)


def test_create_rejects_bad_arguments_without_gpu(lib_path):
    """argument checks come before any CUDA call, so they can be exercised here"""
    lib = ctypes.CDLL(lib_path)
    lib.lbm_create.restype = ctypes.c_void_p
    lib.lbm_create.argtypes = [ctypes.c_int] * 6 + [ctypes.c_double, ctypes.c_int]
    lib.lbm_last_error.restype = ctypes.c_char_p
    assert lib.lbm_create(2, 8, 8, 19, 0, 0, 1.0, 1) is None and b"extents" in lib.lbm_last_error()
    assert lib.lbm_create(8, 8, 8, 15, 0, 0, 1.0, 1) is None and b"lattice" in lib.lbm_last_error()
    assert lib.lbm_create(8, 8, 8, 19, 10, 0, 1.0, 1) is None
    assert lib.lbm_create(8, 8, 8, 19, 0, 6, 1.0, 1) is None
    assert lib.lbm_create(8, 8, 8, 19, 0, 0, 2.5, 1) is None and b"omega" in lib.lbm_last_error()
    assert lib.lbm_create(8, 8, 8, 19, 7, 0, 1.0, 2) is None and b"dtype" in lib.lbm_last_error()
    # a valid request still fails loudly here: no device, no CPU fallback
    assert lib.lbm_create(8, 8, 8, 19, 7, 0, 1.0, 0) is None and b"no CPU fallback" in lib.lbm_last_error()


def test_product_never_imports_oracle():
    """the product path must not route through the oracle"""
    pkg = os.path.join(ROOT, "paper_2010_11751_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "lbm_oracle" not in src and "from oracle" not in src and "import oracle" not in src, f
