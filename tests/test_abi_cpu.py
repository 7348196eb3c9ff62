"""CPU-side checks of the C-ABI library: it builds for sm_100a, loads, exports every symbol that
include/fkconv.h declares, validates arguments before touching CUDA, and FAILS LOUDLY (FK_ERR_CUDA)
instead of falling back to the CPU when no device is present.  No compute call succeeds here.
"""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def K():
    from paper_1909_10547_b200 import build
    build.build()
    from paper_1909_10547_b200 import fkconv
    return fkconv


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "fkconv.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fk_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(K):
    declared = _declared_symbols()
    assert len(declared) >= 20
    assert sorted(K.SYMBOLS) == declared, "fkconv.py SYMBOLS out of sync with include/fkconv.h"
    for name in declared:
        assert hasattr(K.lib, name), name
    out = subprocess.run(["nm", "-D", "--defined-only", K.LIB_PATH], capture_output=True, text=True).stdout
    exported = set(re.findall(r"\sT\s+(fk_[a-z0-9_]+)", out))
    assert set(declared) <= exported


def test_library_targets_sm100a(K):
    assert K.compiled_arch() == 100
    out = subprocess.run(["cuobjdump", "-lelf", K.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "fkconv.h"\nint main(void){return FK_OK;}\n')
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(src),
                           "-o", str(tmp_path / "t.o")])


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def test_argument_validation_happens_before_cuda(K):
    L = K.lib
    pairs = np.array([[0, 1], [1, 1]], dtype=np.int32)
    dummy = ctypes.c_void_p(4096)   # never dereferenced: validation fails first
    # null pointers
    assert L.fk_conv_hadronic(None, _p(pairs), dummy, dummy, 2, 3, 2, 2, 1, None) == K.FK_ERR_INVALID_ARG
    assert b"null" in L.fk_last_error_string()
    assert L.fk_conv_hadronic_vjp(dummy, _p(pairs), dummy, None, dummy, 2, 3, 2, 2, 1, None) == K.FK_ERR_INVALID_ARG
    # non-positive sizes
    for bad in [(0, 3, 2, 2, 1), (2, 0, 2, 2, 1), (2, 3, 0, 2, 1), (2, 3, 2, 0, 1), (2, 3, 2, 2, 0), (-1, 3, 2, 2, 1)]:
        assert L.fk_conv_hadronic(dummy, _p(pairs), dummy, dummy, *bad, None) == K.FK_ERR_INVALID_ARG
    # flavour index out of range
    badp = np.array([[0, 2], [1, 1]], dtype=np.int32)
    assert L.fk_conv_hadronic(dummy, _p(badp), dummy, dummy, 2, 3, 2, 2, 1, None) == K.FK_ERR_INVALID_ARG
    assert b"flavour index" in L.fk_last_error_string()
    negp = np.array([[0, -1], [1, 1]], dtype=np.int32)
    assert L.fk_conv_hadronic(dummy, _p(negp), dummy, dummy, 2, 3, 2, 2, 1, None) == K.FK_ERR_INVALID_ARG
    # DIS: more active flavours than flavours
    flav = np.arange(3, dtype=np.int32)
    assert L.fk_conv_dis(dummy, _p(flav), dummy, dummy, 2, 3, 2, 3, 1, None) == K.FK_ERR_INVALID_ARG
    # limits
    assert L.fk_conv_hadronic(dummy, _p(pairs), dummy, dummy, 2, 3, 300, 2, 1, None) == K.FK_ERR_UNSUPPORTED
    big = np.zeros((2000, 2), dtype=np.int32)
    assert L.fk_conv_hadronic(dummy, _p(big), dummy, dummy, 2, 3, 2, 2000, 1, None) == K.FK_ERR_UNSUPPORTED
    # misaligned device pointer
    assert L.fk_conv_hadronic(ctypes.c_void_p(4100), _p(pairs), dummy, dummy, 2, 3, 2, 2, 1, None) == K.FK_ERR_INVALID_ARG
    # handles
    h = ctypes.c_void_p()
    assert L.fk_table_create(ctypes.byref(h), 7, dummy, _p(pairs), 2, 3, 2, 2, 0, 0, 1) == K.FK_ERR_INVALID_ARG
    assert L.fk_table_create(ctypes.byref(h), 1, dummy, _p(pairs), 2, 3, 2, 2, 1, 0, 1) == K.FK_ERR_INVALID_ARG  # f32 + BORROW
    assert L.fk_table_conv(None, dummy, dummy, 1, None) == K.FK_ERR_INVALID_ARG
    assert L.fk_group_create(ctypes.byref(h), None, 0, 1) == K.FK_ERR_INVALID_ARG
    assert L.fk_table_destroy(None) == K.FK_OK and L.fk_group_destroy(None) == K.FK_OK


def test_no_cpu_fallback_without_a_device(K):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present; the loud failure is checked on the CPU box")
    pairs = np.array([[0, 1], [1, 1]], dtype=np.int32)
    dummy = ctypes.c_void_p(4096)
    rc = K.lib.fk_conv_hadronic(dummy, _p(pairs), dummy, dummy, 2, 3, 2, 2, 1, None)
    assert rc in (K.FK_ERR_CUDA, K.FK_ERR_ALLOC)
    assert K.lib.fk_last_error_string() != b""
    h = ctypes.c_void_p()
    rc = K.lib.fk_table_create(ctypes.byref(h), 1, dummy, _p(pairs), 2, 3, 2, 2, 0, 1, 1)
    assert rc in (K.FK_ERR_CUDA, K.FK_ERR_ALLOC) and not h.value


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1909_10547_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".inl", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), fn
                assert "fk_oracle" not in text or fn == "__init__.py", fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            text = open(os.path.join(ROOT, "oracle", fn)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_1909_10547_b200\.fkconv", text, flags=re.M), fn
            assert "csrc" not in text.replace("paper_1909_10547_b200/csrc)", ""), fn
