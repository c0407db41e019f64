"""Build libchem.so (the C-ABI library of include/chem.h) in-tree with nvcc for sm_100a.

One object per translation unit (compiled in parallel, rebuilt only when a dependency is newer), then one link."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libchem.so")
SOURCES = ["chem.cu", "chem_tps.cu", "chem_tps_inst_a.cu", "chem_tps_inst_b.cu"]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]


def _deps():
    """every source, header and .inl under csrc/ plus the C ABI header"""
    files = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC)) if f.endswith((".cu", ".cuh", ".inl", ".h"))]
    return files + [os.path.join(HERE, "..", "include", "chem.h")]


def _compile(src, obj, verbose):
    cmd = ["nvcc", "-O3", "-std=c++17", *ARCH, "-lineinfo", "-Xcompiler", "-fPIC", *(("-Xptxas", "-v") if verbose else ()),
           "-c", os.path.join(CSRC, src), "-o", obj]
    subprocess.check_call(cmd)


def build(force: bool = False, verbose: bool = False, only=None) -> str:
    deps = [d for d in _deps() if os.path.exists(d)]
    newest = max(os.path.getmtime(d) for d in deps)
    os.makedirs(OBJ, exist_ok=True)
    todo = []
    for src in SOURCES:
        obj = os.path.join(OBJ, src.replace(".cu", ".o"))
        stale = force or not os.path.exists(obj) or os.path.getmtime(obj) < newest
        if only is not None:
            stale = src in only or not os.path.exists(obj)
        if stale:
            todo.append((src, obj))
    if not todo and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        list(ex.map(lambda so: _compile(so[0], so[1], verbose), todo))
    objs = [os.path.join(OBJ, s.replace(".cu", ".o")) for s in SOURCES]
    subprocess.check_call(["nvcc", "-shared", *ARCH, "-o", LIB, *objs])
    return LIB


if __name__ == "__main__":
    only = [a for a in sys.argv[1:] if a.endswith(".cu")] or None
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, only=only))
