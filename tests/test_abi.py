"""The C-ABI boundary without a GPU: libpsg.so builds for sm_100a, loads, exports every symbol
include/*.h declare, and fails loudly (no CPU fallback) when there is no CUDA device."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "psg.h")
HEADERS = [HEADER, os.path.join(ROOT, "include", "psg_bench.h"), os.path.join(ROOT, "include", "psg_static.h")]


@pytest.fixture(scope="module")
def lib():
    from paper_2301_04835_b200 import build
    return ctypes.CDLL(build.build())


def _declared():
    src = "".join(open(h).read() for h in HEADERS)
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(psg_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    names = _declared()
    assert len(names) >= 20 and "psg_cv_eval" in names and "psg_apply_bias_forces" in names
    for n in names:
        assert hasattr(lib, n), f"{n} is declared in include/*.h but not exported by libpsg.so"
    import paper_2301_04835_b200 as p
    assert sorted(p.EXPORTS) == names


def test_header_is_plain_c():
    """the boundary is a C ABI: the header must compile as C with no CUDA or torch headers"""
    for h in HEADERS:
        r = subprocess.run(["gcc", "-std=c99", "-fsyntax-only", "-Wall", "-Werror", "-x", "c", h], capture_output=True, text=True)
        assert r.returncode == 0, r.stderr


def test_library_is_sm100a_and_uses_tma_bulk_copies():
    from paper_2301_04835_b200 import build
    so = build.build()
    out = subprocess.run(["cuobjdump", "-lelf", so], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    sass = subprocess.run(["cuobjdump", "-sass", "-fun", "_Z7k_hillsILi2ELi3ELi2ELb0EEv9SysParams10HillConsts14HillKernelArgs", so],
                          capture_output=True, text=True).stdout
    assert "UBLKCP" in sass and "MUFU.EX2" in sass and "SYNCS" in sass and "FFMA2" in sass


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = ctypes.c_void_p()
    assert lib.psg_create(ctypes.byref(h), 0, None) == -3      # PSG_ECUDA
    lib.psg_last_error.restype = ctypes.c_char_p
    assert b"no CPU fallback" in lib.psg_last_error(None)
    out = ctypes.c_double()
    assert lib.psg_measure_alu_peak(0, 0, ctypes.byref(out)) != 0
    import paper_2301_04835_b200 as p
    with pytest.raises(Exception):
        p.Context(0)


def test_product_does_not_import_oracle():
    """the product path never imports, includes or links anything under oracle/"""
    pkg = os.path.join(ROOT, "paper_2301_04835_b200")
    pat = re.compile(r"^\s*(import\s+oracle|from\s+oracle|#include\s+\".*oracle)", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(dirpath, f)).read()), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            assert "paper_2301_04835_b200 import" not in open(os.path.join(ROOT, "oracle", f)).read()
