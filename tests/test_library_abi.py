"""CPU-only: the C-ABI library builds, loads and exports every symbol include/realfast.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1802_03084_b200 import build as B
    path = B.build()
    return ctypes.CDLL(path)


def _declared():
    text = open(os.path.join(ROOT, "include", "realfast.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rf_[a-z_]+)\s*\(", text)))


def test_header_declares_the_boundary():
    names = _declared()
    for required in ("rf_plan_create", "rf_search", "rf_plan_destroy"):
        assert required in names
    assert len(names) >= 10


def test_every_declared_symbol_is_exported(lib):
    for name in _declared():
        assert hasattr(lib, name), name


def test_binding_lists_the_same_names():
    from paper_1802_03084_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()


def test_struct_sizes_match():
    from paper_1802_03084_b200 import binding
    assert binding.CAND_DTYPE.itemsize == 32
    assert ctypes.sizeof(binding._CandOut) == 24
    assert ctypes.sizeof(binding._Counters) == 32


def test_argument_errors_without_gpu(lib):
    """Validation happens before any CUDA call: bad arguments give RF_ERR_ARG on a CPU box."""
    lib.rf_last_error.restype = ctypes.c_char_p
    out = ctypes.c_void_p()
    assert lib.rf_plan_create(ctypes.byref(out), None, 1, None, 1, 2, 8, ctypes.c_double(0.01), 64,
                              ctypes.c_double(1e-3), None, 1, None, 1, ctypes.c_float(6.0)) == -1
    assert b"null" in lib.rf_last_error()
    assert lib.rf_plan_destroy(None) == 0
    assert lib.rf_search(None, None, None, None) == -1
