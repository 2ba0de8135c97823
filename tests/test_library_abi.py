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


def test_probe_library_is_separate(lib):
    """The measurement / test probes live in their own library: the product ABI exports none of them, the probe
    library exports what csrc/mf_probe.h declares."""
    from paper_2505_12414_b200 import build
    text = open(os.path.join(ROOT, "paper_2505_12414_b200", "csrc", "mf_probe.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    names = sorted(set(re.findall(r"\b(mfp_[a-z0-9_]+)\s*\(", text)))
    assert names == ["mfp_dmma_rate", "mfp_fp64_rate", "mfp_math", "mfp_read_bandwidth"]
    probe = ctypes.CDLL(build.PROBE_LIB_PATH)
    for n in names:
        assert hasattr(probe, n) and not hasattr(lib, n)
    assert not any(n.startswith("mf_probe") for n in declared_functions())


def test_combine_partials_is_rank_ordered_and_compensated():
    """mf_combine_partials (host): exact for cases a plain sum gets wrong, independent of nothing but rank order,
    and non-finite shards propagate."""
    import math

    import numpy as np

    import paper_2505_12414_b200 as mf
    rows = np.array([[1e16, 1.0, 3.0], [1.0, 1e-16, -3.0], [-1e16, 1.0, 0.5], [1.0, 1e-16, 0.25]])
    out = mf.combine_partials(rows)
    assert out[0] == 2.0                               # a plain left-to-right sum gives 1.0 (or 0.0)
    assert out[1] == math.fsum(rows[:, 1]) and out[2] == 0.75
    rng = np.random.default_rng(0)
    big = rng.normal(size=(8, 17)) * 10.0 ** rng.integers(-8, 8, size=(8, 17))
    exact = np.array([math.fsum(big[:, k]) for k in range(17)])
    got = mf.combine_partials(big)
    assert np.all(np.abs(got - exact) <= 2 * np.spacing(np.abs(exact)))
    assert np.array_equal(got, mf.combine_partials(big.copy()))
    bad = big.copy()
    bad[3, 0] = np.inf
    bad[5, 1] = np.nan
    o = mf.combine_partials(bad)
    assert o[0] == np.inf and np.isnan(o[1]) and np.array_equal(o[2:], got[2:])
    with pytest.raises(ValueError):
        mf.combine_partials(np.zeros(3))
