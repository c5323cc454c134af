"""Build libkcs.so (the product) and libkcs_probe.so (bench-only peak probes) in-tree with nvcc for sm_100a
(cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INC = os.path.join(HERE, "..", "include")
LIB = os.path.join(HERE, "libkcs.so")
SOURCES = ["kcs_api.cu", "kcs_projector.cu", "kcs_kinetic.cu", "kcs_static.cu"]
HEADERS = [os.path.join(CSRC, "kcs_internal.cuh"), os.path.join(INC, "kcs.h")]
PROBE_LIB = os.path.join(HERE, "libkcs_probe.so")
PROBE_SOURCES = [os.path.join("bench", "kcs_probe.cu")]
PROBE_HEADERS = [os.path.join(INC, "kcs_probe.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _stale(lib, sources, headers) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    return any(os.path.getmtime(d) > t for d in [os.path.join(CSRC, s) for s in sources] + headers)


def is_stale() -> bool:
    return _stale(LIB, SOURCES, HEADERS)


def _compile(lib, sources, verbose):
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", lib] + \
          [os.path.join(CSRC, s) for s in sources]
    subprocess.check_call(cmd)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or is_stale():
        _compile(LIB, SOURCES, verbose)
    return LIB


def build_probe(force: bool = False, verbose: bool = False) -> str:
    if force or _stale(PROBE_LIB, PROBE_SOURCES, PROBE_HEADERS):
        _compile(PROBE_LIB, PROBE_SOURCES, verbose)
    return PROBE_LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    print(build_probe(force="--force" in sys.argv, verbose="-v" in sys.argv))
