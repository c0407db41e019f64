"""The C-ABI library loads and exports every symbol include/chem.h declares (no compute calls: no GPU here)."""
import ctypes
import os
import re

from paper_1607_03884_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "chem.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(chem_[a-z0-9_]+)\s*\(", text)))


def test_library_builds_and_exports_every_declared_symbol():
    path = build.build()
    L = ctypes.CDLL(path)
    syms = declared_symbols()
    assert len(syms) >= 12
    for s in syms:
        assert hasattr(L, s), s
    assert sorted(binding.EXPORTS) == syms


def test_struct_layouts_match_header():
    assert ctypes.sizeof(binding.chem_opts) == 48
    assert binding.STATS_DTYPE.itemsize == 48
    assert ctypes.sizeof(binding.chem_mech_desc) == 8 + 21 * 8


def test_product_path_does_not_touch_the_oracle():
    """neither side imports, includes or loads the other (synth.py is the shared input generator)"""
    pkg = os.path.join(ROOT, "paper_1607_03884_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".inl", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), f
                assert not re.search(r"#include\s+[\"<][^\n]*oracle", src), f
                assert "libchem_oracle" not in src and "chem_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_1607_03884_b200", src, flags=re.M), f
            assert "libchem.so" not in src and "chem.h" not in src, f
            assert not re.search(r"#include\s+[\"<][^\n]*csrc", src), f
