"""CPU-side checks of the C-ABI boundary: the library builds for sm_100a, loads, and exports every symbol that
include/thc.h declares; no compute entry point is called here (there is no GPU on the CPU test box)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "thc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(thc_[a-z_0-9]+)\s*\(", text)))


@pytest.fixture(scope="module")
def thc():
    import paper_2111_11473_b200 as thc
    thc.build()
    return thc


def test_header_and_binding_agree(thc):
    assert _declared_symbols() == sorted(thc.SYMBOLS)


def test_library_exports_every_declared_symbol(thc):
    L = ctypes.CDLL(thc.LIB_PATH)
    for name in _declared_symbols():
        assert hasattr(L, name), name


def test_strerror_and_null_handle_are_safe(thc):
    L = thc.lib()
    assert L.thc_strerror(0) == b"ok"
    for st in (-1, -2, -3, -4, -5, -99):
        assert len(L.thc_strerror(st)) > 0
    assert L.thc_destroy(None) == -1
    assert L.thc_kernel_launches(None) == 0
    assert L.thc_algorithmic_flops(None) == 0.0


def test_setup_rejects_bad_sizes_and_fails_loudly_without_gpu(thc):
    import torch
    L = thc.lib()
    h = ctypes.c_void_p()
    assert L.thc_setup(ctypes.byref(h), 0, 4, 4, 4, 4, None) == -1          # THC_ERR_INVALID_ARG
    assert L.thc_setup(None, 1, 4, 4, 4, 4, None) == -1
    assert L.thc_setup(ctypes.byref(h), 1 << 40, 4, 4, 4, 4, None) == -2    # THC_ERR_OVERFLOW
    if not torch.cuda.is_available():
        assert L.thc_setup(ctypes.byref(h), 2, 4, 4, 4, 4, None) == -5      # THC_ERR_NO_DEVICE, never a CPU fallback
        with pytest.raises(thc.ThcError):
            thc.thc_setup(2, 4, 4, 4, 4)
