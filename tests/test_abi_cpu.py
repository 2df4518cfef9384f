"""CPU-only checks of the C-ABI boundary: the library loads, exports every symbol include/qcldpc.h declares, and
rejects bad arguments without touching a GPU.  No compute call is made here."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADERS = [os.path.join(ROOT, "include", "qcldpc.h"), os.path.join(ROOT, "include", "qcldpc_profile.h")]


@pytest.fixture(scope="module")
def lib():
    from paper_1702_07740_b200 import build
    so = build.build()
    return ctypes.CDLL(so)


def declared_functions():
    text = "\n".join(open(h).read() for h in HEADERS)
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(qcldpc_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    names = declared_functions()
    assert len(names) >= 10 and "qcldpc_code_create" in names and "qcldpc_decode" in names
    for name in names:
        assert hasattr(lib, name), f"{name} declared in include/*.h but not exported"
    from paper_1702_07740_b200 import binding
    assert sorted(binding.EXPORTED_SYMBOLS) == names


def test_status_strings(lib):
    lib.qcldpc_status_string.restype = ctypes.c_char_p
    seen = {lib.qcldpc_status_string(s) for s in (0, -1, -2, -3, -4, -5)}
    assert len(seen) == 6 and lib.qcldpc_status_string(0) == b"ok"
    assert lib.qcldpc_status_string(-99) == b"unknown status"


def test_bad_arguments_are_rejected_before_any_cuda_call(lib):
    lib.qcldpc_code_create.restype = ctypes.c_int
    lib.qcldpc_code_create.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                       ctypes.POINTER(ctypes.c_void_p)]
    h = ctypes.c_void_p()
    base = np.zeros((2, 3), dtype=np.int32)
    assert lib.qcldpc_code_create(None, 2, 3, 4, ctypes.byref(h)) == -1
    assert lib.qcldpc_code_create(base.ctypes.data, 2, 3, 4, None) == -1
    assert lib.qcldpc_code_create(base.ctypes.data, 0, 3, 4, ctypes.byref(h)) == -1
    assert lib.qcldpc_code_create(base.ctypes.data, 2, 3, 0, ctypes.byref(h)) == -1
    bad = base.copy(); bad[1, 2] = 4          # shift == Z is out of range
    assert lib.qcldpc_code_create(bad.ctypes.data, 2, 3, 4, ctypes.byref(h)) == -1
    bad[1, 2] = -2
    assert lib.qcldpc_code_create(bad.ctypes.data, 2, 3, 4, ctypes.byref(h)) == -1
    assert not h.value
    lib.qcldpc_workspace_bytes.restype = ctypes.c_size_t
    lib.qcldpc_workspace_bytes.argtypes = [ctypes.c_void_p, ctypes.c_int]
    assert lib.qcldpc_workspace_bytes(None, 4) == 0
    lib.qcldpc_decode.restype = ctypes.c_int
    lib.qcldpc_decode.argtypes = [ctypes.c_void_p] * 3 + [ctypes.c_int] * 3 + [ctypes.c_void_p] * 5 + \
        [ctypes.c_size_t, ctypes.c_void_p]
    assert lib.qcldpc_decode(None, None, None, 1, 1, 0, None, None, None, None, None, 0, None) == -1
    lib.qcldpc_code_destroy.argtypes = [ctypes.c_void_p]
    lib.qcldpc_code_destroy(None)             # no-op


def test_no_cpu_fallback_without_a_gpu():
    """On a box without a CUDA device the product path must fail loudly, not fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1702_07740_b200 import binding
    base = np.zeros((1, 2), dtype=np.int32)
    with pytest.raises(binding.QCLDPCError) as ei:
        binding.QCLDPCCode(base, 4)
    assert ei.value.status == -4


def test_product_package_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1702_07740_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), fn
                assert "liboracle" not in text and '#include "../../oracle' not in text, fn
    for dirpath, _, files in os.walk(os.path.join(ROOT, "oracle")):
        for fn in files:
            if fn.endswith((".py", ".c", ".inc")):
                text = open(os.path.join(dirpath, fn)).read()
                assert "paper_1702_07740_b200.binding" not in text and "libqcldpc" not in text, fn
