"""The C-ABI library builds, loads without a GPU and exports every symbol include/hydro.h
declares; argument errors that need no device are reported through the status code."""
import ctypes as C
import os
import re

import pytest

from paper_1812_07977_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libs():
    build.build()
    return binding.load_library(False), binding.load_library(True)


def test_header_symbols_all_exported(libs):
    header = open(os.path.join(ROOT, "include", "hydro.h")).read()
    declared = set(re.findall(r"\b(hydro_[a-z_]+)\s*\(", header))
    assert declared == set(binding.SYMBOLS), declared ^ set(binding.SYMBOLS)
    for L in libs:
        for name in declared:
            assert hasattr(L, name), name


def test_build_flavours(libs):
    prod, ver = libs
    assert prod.hydro_is_verification_build() == 0
    assert ver.hydro_is_verification_build() == 1


def test_argument_errors_without_device(libs):
    L = libs[0]
    h = C.c_void_p()
    ok = (C.c_int * 6)(0, 0, 0, 0, 0, 0)
    assert L.hydro_create(1, 4, 4, 1.4, 0.1, ok, C.byref(h)) == 1          # HYDRO_ERR_ARG
    assert L.hydro_create(4, 4, 4, 1.0, 0.1, ok, C.byref(h)) == 1
    assert L.hydro_create(4, 4, 4, 1.4, -1.0, ok, C.byref(h)) == 1
    bad = (C.c_int * 6)(2, 0, 0, 0, 0, 0)
    assert L.hydro_create(4, 4, 4, 1.4, 0.1, bad, C.byref(h)) == 1
    assert b"periodic" in L.hydro_last_error()
    assert L.hydro_step(None, 0.1) == 1
    assert L.hydro_launch_count() == 0


def test_no_cpu_fallback_without_device(libs):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    L = libs[0]
    h = C.c_void_p()
    ok = (C.c_int * 6)(0, 0, 0, 0, 0, 0)
    assert L.hydro_create(4, 4, 4, 1.4, 0.1, ok, C.byref(h)) == 3          # HYDRO_ERR_CUDA
    assert not h.value
    with pytest.raises(RuntimeError):
        binding.Hydro(4, 4, 4, 1.4, 0.1, (0,) * 6)


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1812_07977_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "liboracle" not in text, f
