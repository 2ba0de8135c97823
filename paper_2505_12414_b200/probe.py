"""Binding of ``lib/libmorefit_b200_probe.so`` (csrc/mf_probe.h): measurement and test probes.

Not part of the product's C-ABI: ``bench.py`` uses the fp64-rate / read-bandwidth probes for its roofline
denominators and the GPU tests use ``math`` to check the kernels' own exp / log / reciprocal element by element.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

_lib = None


def _load() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        if not os.path.exists(_build.PROBE_LIB_PATH):
            raise ImportError(f"{_build.PROBE_LIB_PATH} is missing: run `python -m paper_2505_12414_b200.build`")
        lib = ctypes.CDLL(_build.PROBE_LIB_PATH)
        dp, vp = ctypes.POINTER(ctypes.c_double), ctypes.c_void_p
        lib.mfp_fp64_rate.restype = ctypes.c_int
        lib.mfp_fp64_rate.argtypes = [ctypes.c_int, vp, dp]
        lib.mfp_dmma_rate.restype = ctypes.c_int
        lib.mfp_dmma_rate.argtypes = [ctypes.c_int, vp, dp]
        lib.mfp_read_bandwidth.restype = ctypes.c_int
        lib.mfp_read_bandwidth.argtypes = [ctypes.c_int, vp, ctypes.c_size_t, ctypes.c_int, dp]
        lib.mfp_math.restype = ctypes.c_int
        lib.mfp_math.argtypes = [ctypes.c_int, vp, ctypes.c_int, ctypes.c_int64, dp, dp]
        _lib = lib
    return _lib


def _check(rc: int, what: str) -> None:
    if rc != 0:
        raise RuntimeError(f"{what}: cudaError {rc}")


def fp64_rate(device: int = 0, stream: int = 0) -> float:
    """Measured fp64-pipe rate (DFMA thread-instructions per second)."""
    v = ctypes.c_double()
    _check(_load().mfp_fp64_rate(int(device), ctypes.c_void_p(stream), ctypes.byref(v)), "mfp_fp64_rate")
    return float(v.value)


def dmma_rate(device: int = 0, stream: int = 0) -> dict:
    """fp64 tensor-core rate against the vector fp64 pipe (see mf_probe.h)."""
    out = (ctypes.c_double * 4)()
    _check(_load().mfp_dmma_rate(int(device), ctypes.c_void_p(stream), out), "mfp_dmma_rate")
    return {"dmma_fma_per_s": out[0], "dfma_fma_per_s": out[1], "mix_4dmma_8dfma_vs_sum": out[2], "mix_1dmma_8dfma_vs_sum": out[3]}


def read_bandwidth(nbytes: int, repeats: int = 1, device: int = 0, stream: int = 0) -> float:
    """Measured read bandwidth (bytes/s) of an nbytes working set read `repeats` times."""
    v = ctypes.c_double()
    _check(_load().mfp_read_bandwidth(int(device), ctypes.c_void_p(stream), int(nbytes), int(repeats), ctypes.byref(v)),
           "mfp_read_bandwidth")
    return float(v.value)


def math(op: str, x, device: int = 0, stream: int = 0) -> np.ndarray:
    """The kernels' device exp / log / rcp / exp32 evaluated element-wise."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    y = np.empty_like(x)
    dp = ctypes.POINTER(ctypes.c_double)
    _check(_load().mfp_math(int(device), ctypes.c_void_p(stream), {"exp": 0, "log": 1, "rcp": 2, "exp32": 3}[op], x.size,
                            x.ctypes.data_as(dp), y.ctypes.data_as(dp)), "mfp_math")
    return y
