"""CPU-side checks of the C-ABI library: it builds for sm_100a, loads, exports every symbol include/mipwa.h
declares, and refuses to run without a GPU (no CPU fallback).  No compute calls here."""
import ctypes
import os
import re

import pytest

from paper_1703_03284_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "mipwa.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mipwa_[a-z0-9_]+)\s*\(", text)))


def test_library_builds_and_exports_every_declared_symbol():
    build.build()
    lib = ctypes.CDLL(build.LIB)
    names = declared_symbols()
    assert len(names) >= 18
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/mipwa.h but not exported"
    assert sorted(binding.SYMBOLS) == names


def test_binary_holds_sm100a_code_only():
    import subprocess
    out = subprocess.run(["/usr/local/cuda/bin/cuobjdump", "-lelf", build.LIB], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    assert not re.search(r"sm_(?!100a)\d+", out)


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(binding.MipwaError) as ei:
        binding.Mipwa((1.86966, 0.13957, 0.13957, 0.13957), [0.1, 1.0, 2.0], [])
    assert ei.value.code == binding.ERR_CUDA
    with pytest.raises(binding.MipwaError):
        binding.measure_fp64_peak(0, 0.1)


def test_product_does_not_import_the_oracle():
    """The CUDA package and the oracle share no code and neither imports the other."""
    for base, pat in (("paper_1703_03284_b200", r"\boracle\b"), ("oracle", r"paper_1703_03284_b200|mipwa\.h|csrc")):
        for dirpath, _, files in os.walk(os.path.join(ROOT, base)):
            for f in files:
                if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                    src = open(os.path.join(dirpath, f)).read()
                    code = "\n".join(l for l in src.splitlines()
                                     if re.match(r"\s*(import|from|#include)", l))
                    assert not re.search(pat, code), f"{base}/{f} references the other side"
