"""The C-ABI boundary without a GPU: libtomolsqr.so builds for sm_100a, loads, exports every symbol
include/tomo_lsqr.h declares, and fails loudly (status code, no crash, no CPU fallback) when there is
no CUDA device.  No compute call is made here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2604_11920_b200 import build
    build.build()
    import paper_2604_11920_b200 as tl
    return tl


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "tomo_lsqr.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tomo_(?:lsqr|lsmr|status)_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    names = declared_symbols()
    assert "tomo_lsqr_create" in names and "tomo_lsqr_solve" in names and "tomo_lsqr_destroy" in names
    assert sorted(lib.SYMBOLS) == names  # the binding covers exactly what the header declares
    cdll = lib.load()
    for name in names:
        assert hasattr(cdll, name), name


def test_status_strings(lib):
    for code in range(8):
        s = lib.tomo_status_string(code)
        assert isinstance(s, str) and s
    assert lib.tomo_status_string(0) == "ok"
    assert "unknown" in lib.tomo_status_string(99)


def test_result_struct_layout(lib):
    # int32 itn, int32 istop, 6 doubles (include/tomo_lsqr.h)
    assert ctypes.sizeof(lib.tomo_lsqr_result_t) == 8 + 6 * 8
    assert lib.tomo_lsqr_result_t.r1norm.offset == 8


def test_argument_checks_need_no_device(lib):
    cdll = lib.load()
    h = ctypes.c_void_p(123)
    # null out pointer, bad sizes, null arrays: rejected before any CUDA call
    assert cdll.tomo_lsqr_create(None, 4, 4, 0, None, None, None, 0, None) == lib.TOMO_ERR_INVALID_ARG
    assert cdll.tomo_lsqr_create(ctypes.byref(h), 0, 4, 0, None, None, None, 0, None) == lib.TOMO_ERR_INVALID_ARG
    assert h.value is None
    assert cdll.tomo_lsqr_create(ctypes.byref(h), 2**31, 4, 0, None, None, None, 0, None) == lib.TOMO_ERR_RANGE
    assert cdll.tomo_lsqr_create(ctypes.byref(h), 4, 4, 1, None, None, None, 0, None) == lib.TOMO_ERR_INVALID_ARG
    assert cdll.tomo_lsqr_create(ctypes.byref(h), 4, 4, 0, None, None, None, 7, None) == lib.TOMO_ERR_INVALID_ARG
    assert cdll.tomo_lsqr_solve(None, None, 0.0, 0.0, 0.0, 1, None, None, None, None, None) == lib.TOMO_ERR_INVALID_ARG
    assert cdll.tomo_lsqr_set_option(None, b"graph", 1) == lib.TOMO_ERR_INVALID_ARG
    cdll.tomo_lsqr_destroy(None)  # harmless


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import numpy as np
    rp = np.zeros(5, dtype=np.int64)
    with pytest.raises(lib.TomoError) as ei:
        lib.tomo_lsqr_create(4, 4, 0, rp, None, None, stream=0)
    assert ei.value.status in (lib.TOMO_ERR_CUDA, lib.TOMO_ERR_UNSUPPORTED_ARCH, lib.TOMO_ERR_NOT_DEVICE_PTR)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2604_11920_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "lsqr_oracle" not in src, f
