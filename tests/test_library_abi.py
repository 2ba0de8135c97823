"""The C-ABI library builds (nvcc cross-compiles without a GPU), loads, and exports every function that
include/morefit_b200.h declares; the binding's EXPORTS list matches the header; without a CUDA device the
entry points fail loudly instead of falling back to anything."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "morefit_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mf_[a-z0-9_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    from paper_2505_12414_b200 import build
    return ctypes.CDLL(build.build())


def test_header_symbols_are_exported(lib):
    names = declared_functions()
    assert len(names) >= 20
    missing = [n for n in names if not hasattr(lib, n)]
    assert not missing, missing


def test_binding_lists_the_same_symbols():
    import paper_2505_12414_b200 as mf
    assert sorted(mf.EXPORTS) == declared_functions()


def test_no_cpu_fallback():
    import torch

    import paper_2505_12414_b200 as mf
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    lib = mf.load_library()
    h = ctypes.c_void_p()
    st = lib.mf_ctx_create(0, None, ctypes.byref(h))
    assert st == mf.MF_ERR_CUDA and not h.value
    with pytest.raises(mf.MoreFitError):
        mf.Context(0)


def test_oracle_is_not_imported_by_the_product():
    """The product package and bench.py's GPU arm never import oracle/ (only tests, smoke and the CPU legs may)."""
    pkg = os.path.join(ROOT, "paper_2505_12414_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                src = open(os.path.join(dirpath, f), errors="ignore").read()
                assert "import oracle" not in src and "mf_oracle" not in src, f
