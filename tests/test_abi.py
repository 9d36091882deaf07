"""The C-ABI library builds, loads and exports every symbol include/purify_op.h declares
(no compute calls: no GPU here).  -m "not gpu" """
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols(name="purify_op.h"):
    src = open(os.path.join(ROOT, "include", name)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(purify_[a-z_0-9]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_1903_04502_b200 import build, op
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    declared = header_symbols()
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in purify_op.h but not exported"
    assert sorted(op.SYMBOLS) == declared
    from paper_1903_04502_b200 import wavelet
    wdeclared = [s for s in header_symbols("purify_wavelet.h") if s not in ("purify_last_error",)]
    assert sorted(wavelet.SYMBOLS) == wdeclared and len(wdeclared) == 7
    for name in wdeclared:
        assert hasattr(lib, name), f"{name} declared in purify_wavelet.h but not exported"
    L = op.load_library()
    assert L.purify_version() >= 100
    assert L.purify_strerror(-7).decode().startswith("no CUDA device")
    assert L.purify_strerror(0).decode() == "ok"


def test_no_device_is_a_loud_error_not_a_fallback():
    """Without a GPU create must fail with PURIFY_ERR_NO_DEVICE (there is no CPU path)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_1903_04502_b200 import op
    L = op.load_library()
    h = ctypes.c_void_p()
    uv = (ctypes.c_double * 8)()
    st = L.purify_op_create_host(ctypes.byref(h), 16, 2, 4, 4, ctypes.cast(uv, ctypes.c_void_p), None, 1, None, None)
    assert st == -7 and not h.value
    assert b"no CPU fallback" in L.purify_last_error()
    # argument validation happens before the device check
    assert L.purify_op_create_host(ctypes.byref(h), 15, 2, 4, 4, ctypes.cast(uv, ctypes.c_void_p), None, 1, None, None) == -1
    assert L.purify_op_create_host(ctypes.byref(h), 16, 3, 4, 4, ctypes.cast(uv, ctypes.c_void_p), None, 1, None, None) == -2
    assert L.purify_op_create_host(ctypes.byref(h), 16, 2, 5, 4, ctypes.cast(uv, ctypes.c_void_p), None, 1, None, None) == -1
    assert L.purify_degrid(None, None, None, None) == -1


def test_product_does_not_import_the_oracle():
    """The product path may not route through oracle/ (task rule 3)."""
    pkg = os.path.join(ROOT, "paper_1903_04502_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".hpp", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert "purify_oracle" not in txt, f
    otxt = open(os.path.join(ROOT, "oracle", "purify_oracle.cpp")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "paper_1903_04502_b200" not in otxt.replace("paper_1903_04502_b200/csrc", "").replace("paper_1903_04502_b200/op.py", "")
