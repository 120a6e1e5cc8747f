"""Build libcolatus.so (the product) and libcolatus_probe.so (device microbenchmarks, include/colatus_probe.h)
in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcolatus.so")
SOURCES = ["colatus_api.cu", "cosmo_host.cpp"]
HEADERS = ["force_kernels.cuh", "force_sym_kernels.cuh", "integrate_kernels.cuh", "analysis_kernels.cuh", os.path.join("..", "..", "include", "colatus.h")]
PROBE_LIB = os.path.join(HERE, "libcolatus_probe.so")
PROBE_SOURCES = ["colatus_probe.cu"]
PROBE_HEADERS = ["probe_kernels.cuh", "force_kernels.cuh", os.path.join("..", "..", "include", "colatus_probe.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "--cudart", "static"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale(lib, sources, headers) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in sources + headers] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def needs_build() -> bool:
    return _stale(LIB, SOURCES, HEADERS)


def _compile(lib, sources, verbose):
    tmp = lib + f".tmp{os.getpid()}"
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", tmp] + [os.path.join(CSRC, s) for s in sources]
    subprocess.check_call(cmd)
    os.replace(tmp, lib)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        _compile(LIB, SOURCES, verbose)
    if force or _stale(PROBE_LIB, PROBE_SOURCES, PROBE_HEADERS):
        _compile(PROBE_LIB, PROBE_SOURCES, verbose)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
