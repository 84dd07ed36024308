"""Host-side checks that need no GPU: liblgf.so builds for sm_100a, loads, exports every symbol
include/lgf.h declares, validates its arguments, and fails loudly (no CPU fallback) without a device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1206_0675_b200 import binding, build

    build.build()
    return binding.load()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "lgf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lgf_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_exported(lib):
    names = declared_symbols()
    assert {"lgf_create", "lgf_iterate", "lgf_measure", "lgf_fix"} <= set(names)
    for n in names:
        assert hasattr(lib, n), "liblgf.so does not export " + n


def test_binding_covers_header():
    from paper_1206_0675_b200 import binding

    assert set(declared_symbols()) == set(binding.SIGNATURES)


def test_sass_is_sm100a_and_has_no_library_fft():
    """The product must not link cuFFT (north_star: hand-written FFT only)."""
    import subprocess

    from paper_1206_0675_b200 import binding

    out = subprocess.run(["ldd", binding.library_path()], capture_output=True, text=True).stdout
    assert "cufft" not in out.lower() and "cublas" not in out.lower()
    elf = subprocess.run(["cuobjdump", "-lelf", binding.library_path()], capture_output=True, text=True).stdout
    assert "sm_100a" in elf


def test_argument_validation_and_no_cpu_fallback(lib):
    import torch

    h = ctypes.c_void_p()
    bad = (ctypes.c_int * 4)(8, 8, 8, 10)
    assert lib.lgf_create(bad, 8, 18, ctypes.byref(h)) == -1          # LGF_EINVAL: 10 is not 2^a 3^b <= 64
    good = (ctypes.c_int * 4)(8, 8, 8, 8)
    assert lib.lgf_create(good, 3, 18, ctypes.byref(h)) == -1
    assert lib.lgf_create(good, 8, 9, ctypes.byref(h)) == -1
    if not torch.cuda.is_available():
        # no device: creation must fail with LGF_ECUDA and say why -- never compute on the CPU
        assert lib.lgf_create(good, 8, 18, ctypes.byref(h)) == -3
        assert not h.value
        assert b"no CUDA device" in lib.lgf_last_error(None)
        from paper_1206_0675_b200 import binding

        with pytest.raises(binding.LgfError):
            binding.Context((8, 8, 8, 8))


def test_product_does_not_import_oracle():
    """The CUDA path and its binding never reference oracle/ (and the oracle never references them)."""
    pkg = os.path.join(ROOT, "paper_1206_0675_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "lgf_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_1206_0675_b200\b", src, flags=re.M), f
            assert "csrc" not in src or f.endswith(".c") or "imports nothing" in src
