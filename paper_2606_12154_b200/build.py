"""Builds libhq.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a, and libhq_host.so (host runtime path) with g++.

    python -m paper_2606_12154_b200.build          # rebuild if sources are newer
    python -m paper_2606_12154_b200.build --force
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libhq.so")
HOST_SRC = os.path.join(HERE, "host", "hq_host.cpp")
HOST_LIB = os.path.join(HERE, "libhq_host.so")

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "static",
]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return sources() + glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        glob.glob(os.path.join(INCLUDE, "*.h"))


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in _deps())


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-I", INCLUDE, "-o", LIB] + sources()
        subprocess.check_call(cmd)
    return LIB


def build_host(force: bool = False) -> str:
    """libhq_host.so: the host-side runtime path (include/hq_host.h), plain g++."""
    deps = [HOST_SRC, os.path.join(INCLUDE, "hq_host.h")]
    if force or not os.path.exists(HOST_LIB) or any(os.path.getmtime(p) > os.path.getmtime(HOST_LIB) for p in deps):
        extra = os.environ.get("HQ_HOST_EXTRA_CXXFLAGS", "").split()   # e.g. -fsanitize=address,undefined (profiles/r02_sanitizers.md)
        subprocess.check_call([os.environ.get("CXX", "g++"), "-O2", "-std=c++17", "-shared", "-fPIC", "-Wall"] + extra + ["-o", HOST_LIB, HOST_SRC])
    return HOST_LIB


if __name__ == "__main__":
    print(build_host(force="--force" in sys.argv))
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
