"""CPU-side checks of the product library: it builds for sm_100a, loads, exports every symbol
include/astra.h declares, and fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_10440_b200 import build, load_library
    build.build()
    return load_library()


def test_exports_every_declared_symbol(lib):
    from paper_2606_10440_b200 import EXPORTED_SYMBOLS
    hdr = open(os.path.join(ROOT, "include", "astra.h")).read()
    declared = sorted(set(re.findall(r"\b(astra_[a-z_]+)\s*\(", hdr)))
    assert declared == sorted(EXPORTED_SYMBOLS)
    for name in declared:
        assert getattr(lib, name) is not None


def test_sass_is_sm100a(lib):
    out = subprocess.run(["cuobjdump", "-lelf", lib._name], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_no_device_fails_loudly(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2606_10440_b200 import AstraError, Engine
    with pytest.raises(AstraError) as ei:
        Engine(0)
    assert ei.value.code == -3


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_10440_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cpp", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("oracle/", "").replace("shares nothing with oracle", "").lower() \
                    or f in ("astra_loader.cpp", "astra_internal.h"), f


def test_oracle_does_not_import_product():
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            assert "paper_2606_10440_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "paper_2606_10440_b200/csrc", "").replace("imported by paper_2606_10440_b200", "")
