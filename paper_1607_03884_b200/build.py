"""Build libchem.so (the C-ABI library of include/chem.h) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libchem.so")
SOURCES = ["chem.cu"]


def _deps():
    """every source, header and .inl under csrc/ plus the C ABI header"""
    files = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cu", ".cuh", ".inl", ".h"))]
    return files + [os.path.join(HERE, "..", "include", "chem.h")]


def nvcc_cmd(extra=()):
    return ["nvcc", "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
            "-Xcompiler", "-fPIC", "-shared", *extra, "-o", LIB, *[os.path.join(CSRC, s) for s in SOURCES]]


def build(force: bool = False, verbose: bool = False) -> str:
    deps = [d for d in _deps() if os.path.exists(d)]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    cmd = nvcc_cmd(("-Xptxas", "-v") if verbose else ())
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
