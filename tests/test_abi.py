"""CPU-side checks of the boundary: libcube.so builds for sm_100a, loads, exports every symbol that
include/cube.h declares, validates arguments before touching the device, and refuses to run without a GPU
(no CPU fallback).  No compute calls here."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1211_4896_b200 import build
    build.build()
    import paper_1211_4896_b200 as cube
    return cube


def test_header_symbols_are_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "cube.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(cube_[a-z_0-9]+)\s*\(", hdr))
    assert declared == set(lib.SYMBOLS), declared ^ set(lib.SYMBOLS)
    L = lib.load()
    for name in declared:
        assert getattr(L, name) is not None


def test_struct_layout_matches_header(lib):
    assert ctypes.sizeof(lib.MomentsT) == 40
    assert [f[0] for f in lib.MomentsT._fields_] == ["count", "nan_count", "min", "max", "mean", "std"]


def test_strerror(lib):
    L = lib.load()
    assert L.cube_strerror(0) == b"ok" and b"invalid" in L.cube_strerror(1)


def test_binary_is_sm100a_only(lib):
    import subprocess
    out = subprocess.run(["cuobjdump", "--list-elf", os.path.join(ROOT, "paper_1211_4896_b200", "libcube.so")],
                         capture_output=True, text=True).stdout
    assert "sm_100a" in out and "sm_90" not in out


def test_no_cpu_fallback_without_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present; this checks the GPU-less behaviour")
    with pytest.raises(lib.CubeError) as e:
        lib.Context()
    assert e.value.code == lib.ECUDA


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1211_4896_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".inl", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle", src, flags=re.M), f
                assert "cube_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_1211_4896_b200", src, flags=re.M)
            assert "libcube.so" not in src and "csrc" not in src
