"""Builds the C-ABI library ``lib/libmorefit_b200.so`` (and the separate probe library
``lib/libmorefit_b200_probe.so``: measurement / test probes, not part of the product ABI) in-tree with nvcc for sm_100a.

``python -m paper_2505_12414_b200.build`` (or ``__graft_entry__.build()``).  nvcc
cross-compiles without a GPU.  The library is rebuilt only when a source is newer.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB_DIR = os.path.join(HERE, "lib")
LIB_PATH = os.path.join(LIB_DIR, "libmorefit_b200.so")
SOURCES = ["mf_api.cu", "mf_fit.cpp", "mf_dist.cpp", "mf_generate.cu", "mf_noalloc.cu"]
PROBE_LIB_PATH = os.path.join(LIB_DIR, "libmorefit_b200_probe.so")
PROBE_SOURCES = ["mf_probe.cu"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-fopenmp", "-shared"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale() -> bool:
    if not (os.path.exists(LIB_PATH) and os.path.exists(PROBE_LIB_PATH)):
        return True
    t = min(os.path.getmtime(LIB_PATH), os.path.getmtime(PROBE_LIB_PATH))
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(INCLUDE, "morefit_b200.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB_PATH
    os.makedirs(LIB_DIR, exist_ok=True)
    for path, sources in ((LIB_PATH, SOURCES), (PROBE_LIB_PATH, PROBE_SOURCES)):
        tmp = path + f".{os.getpid()}.tmp"
        cmd = [_nvcc(), *NVCC_FLAGS, "-I", INCLUDE, "-o", tmp] + [os.path.join(CSRC, s) for s in sources]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
            print(" ".join(cmd), file=sys.stderr)
        subprocess.check_call(cmd)
        os.replace(tmp, path)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
