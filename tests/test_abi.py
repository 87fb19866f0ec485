"""CPU-side checks of the boundary: libsmaug.so builds, loads, and exports every symbol include/smaug.h
declares; argument validation that needs no GPU; no CPU fallback (create fails with SMAUG_ECUDA here)."""
import ctypes as C
import os
import re

import pytest

import paper_1710_06423_b200 as pkg

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "smaug.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(smaug_[a-z_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    pkg.build()
    L = C.CDLL(pkg.LIB_PATH)
    syms = declared_symbols()
    assert len(syms) >= 17 and "smaug_step" in syms and "smaug_create" in syms
    for s in syms:
        assert hasattr(L, s), s


def test_library_exports_every_symbol_of_the_3d_header():
    src = open(os.path.join(ROOT, "include", "smaug3d.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    syms = sorted(set(re.findall(r"\b(smaug3_[a-z_]+)\s*\(", src)))
    L = C.CDLL(pkg.build())
    assert len(syms) >= 12 and "smaug3_step" in syms
    for s in syms:
        assert hasattr(L, s), s
    L = pkg.lib()
    h = C.c_void_p()
    bc = (C.c_int * 6)(0, 0, 0, 0, 0, 0)
    assert L.smaug3_workspace_bytes(0, 4, 4) == 0
    assert 14.5e9 < L.smaug3_workspace_bytes(256, 256, 256) < 15.2e9        # 94 padded volumes of 288 x 262 x 262 doubles
    assert L.smaug3_create(0, 4, 4, 1.4, bc, None, C.byref(h)) == pkg.EINVAL
    assert L.smaug3_create(4, 4, 4, 1.0, bc, None, C.byref(h)) == pkg.EINVAL
    assert L.smaug3_create(4, 4, 4, 1.4, (C.c_int * 6)(0, 0, 0, 0, 0, 1), None, C.byref(h)) == pkg.EINVAL
    assert L.smaug3_create(4, 4, 4, 1.4, bc, None, None) == pkg.EINVAL
    assert L.smaug3_step(None, 1, 0.3) == pkg.EINVAL and b"bad" in L.smaug3_last_error()
    L.smaug3_destroy(None)
    import torch
    if not torch.cuda.is_available():
        assert L.smaug3_create(8, 8, 8, 1.4, bc, None, C.byref(h)) == pkg.ECUDA and not h.value
        assert b"no CPU fallback" in L.smaug3_last_error()


def test_workspace_bytes_and_argument_validation():
    L = pkg.lib()
    assert L.smaug_workspace_bytes(0, 4, 0) == 0
    small = L.smaug_workspace_bytes(1000, 1000, 0)
    # 4 buffers x 6 planes of (1006 rows x pitch 1024 doubles)
    assert small >= 24 * 1006 * 1024 * 8 and small < 24 * 1006 * 1024 * 8 + 64 * 1024
    assert L.smaug_workspace_bytes(1000, 1000, 1) - small >= 4 * 1006 * 1024 * 8
    big = L.smaug_workspace_bytes(8000, 8000, 0)
    assert 12e9 < big < 13e9                                  # fits one B200 (180 GB) many times over
    h = C.c_void_p()
    bc = (C.c_int * 4)(0, 0, 0, 0)
    assert L.smaug_create(0, 4, 1.4, bc, None, C.byref(h)) == pkg.EINVAL
    assert L.smaug_create(4, 4, 1.0, bc, None, C.byref(h)) == pkg.EINVAL
    assert L.smaug_create(4, 4, 1.4, (C.c_int * 4)(0, 1, 0, 0), None, C.byref(h)) == pkg.EINVAL
    assert L.smaug_create(4, 4, 1.4, (C.c_int * 4)(0, 0, 5, 5), None, C.byref(h)) == pkg.EINVAL
    assert L.smaug_create(4, 4, 1.4, bc, None, None) == pkg.EINVAL
    assert L.smaug_set_param(None, 0, 1.0) == pkg.EINVAL
    assert L.smaug_step(None, 1, 0.3) == pkg.EINVAL
    assert b"NULL" in L.smaug_last_error()
    L.smaug_destroy(None)                                      # no-op


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    L = pkg.lib()
    h = C.c_void_p()
    rc = L.smaug_create(8, 8, 1.4, (C.c_int * 4)(0, 0, 0, 0), None, C.byref(h))
    assert rc == pkg.ECUDA and not h.value
    assert b"no CPU fallback" in L.smaug_last_error()


def test_product_does_not_import_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1710_06423_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt
                assert "smaug_oracle" not in txt and "liboracle" not in txt
    txt = open(os.path.join(ROOT, "oracle", "smaug_oracle.cpp")).read()
    assert "smaug.h" not in txt.replace("include/smaug.h (SURVEY", "") and "csrc/" not in txt.split("namespace")[1]
