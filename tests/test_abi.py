"""CPU-side checks of the boundary: libfresnel.so loads, exports every symbol include/fresnel.h
declares, and refuses to create a plan without a CUDA device (no CPU fallback).  No compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_1806_06467_b200 import build, binding
    build.build()                 # nvcc cross-compiles without a GPU
    return binding


def header_symbols():
    src = open(os.path.join(ROOT, "include", "fresnel.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fresnel_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(binding):
    L = binding.lib()
    names = header_symbols()
    assert len(names) >= 15
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/fresnel.h but not exported"
    assert sorted(binding.SYMBOLS) == names


def test_status_strings_and_version(binding):
    L = binding.lib()
    assert L.fresnel_status_string(0) == b"FRESNEL_OK"
    assert L.fresnel_status_string(2) == b"FRESNEL_ERR_UNSUPPORTED"
    assert b"sm_100a" in L.fresnel_version()


def test_plan_create_argument_checks_and_no_cpu_fallback(binding):
    import torch
    L = binding.lib()
    h = ctypes.c_void_p()
    assert L.fresnel_plan_create(ctypes.byref(h), 7919, 1, 1) == 2      # a prime above the Bluestein capacity: UNSUPPORTED
    assert L.fresnel_plan_create(ctypes.byref(h), 12, 1, 1) == 2
    assert L.fresnel_plan_create(ctypes.byref(h), 16384, 1, 1) == 2
    assert L.fresnel_plan_create(ctypes.byref(h), 256, -1, 1) == 1
    assert L.fresnel_plan_create(ctypes.byref(h), 256, 1, 7) == 2
    if not torch.cuda.is_available():
        assert L.fresnel_plan_create(ctypes.byref(h), 256, 1, 1) == 4   # FRESNEL_ERR_CUDA: fails loudly
        with pytest.raises(binding.FresnelError):
            binding.Plan(256, 1, "c128")


def test_product_does_not_import_the_oracle():
    """The product path may not route through oracle/ (only tests, smoke() and bench's CPU legs may)."""
    pkg = os.path.join(ROOT, "paper_1806_06467_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f"{f} imports the oracle"
                assert "liboracle" not in txt and "fresnel_oracle" not in txt, f"{f} links the oracle"
