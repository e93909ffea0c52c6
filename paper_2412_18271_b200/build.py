"""Builds libpfc.so (the C-ABI library of include/pfc.h) in-tree with nvcc for
sm_100a.  `python -m paper_2412_18271_b200.build` or build_libpfc()."""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libpfc.so")
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "shared",
]


def _sources():
    return sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh")))


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    hdr = os.path.join(os.path.dirname(_HERE), "include", "pfc.h")
    return any(os.path.getmtime(s) > t for s in _sources() + [hdr])


def build_libpfc(force: bool = False, verbose: bool = False) -> str:
    if not (force or needs_build()):
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          ["-o", LIB, os.path.join(CSRC, "pfc_api.cu")]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build_libpfc(force="--force" in sys.argv, verbose="-v" in sys.argv))
