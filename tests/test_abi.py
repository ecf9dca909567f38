"""The C-ABI library builds, loads, and exports every symbol include/cclr.h declares (no compute calls: no GPU here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "cclr.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(cclr_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_2307_14296_b200 import build, _lib
    build.build()
    names = declared_symbols()
    assert {"cclr_create", "cclr_sigma", "cclr_solve", "cclr_property", "cclr_destroy"} <= set(names)
    lib = ctypes.CDLL(_lib.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), n
    assert set(names) == set(_lib.SIGNATURES), set(names) ^ set(_lib.SIGNATURES)
    _lib.load()


def test_error_strings_and_argument_checks_without_gpu():
    from paper_2307_14296_b200 import _lib
    lib = _lib.load()
    assert lib.cclr_strerror(0) == b"ok"
    assert b"invalid" in lib.cclr_strerror(-1)
    h = ctypes.c_void_p()
    assert lib.cclr_create(1, 1, None, None, None, None, 0, None, ctypes.byref(h)) == -1   # CCLR_EINVAL before any CUDA call
    assert lib.cclr_sigma(None, None, None, 1, 0.0, 0.0, None, None) == -1
    assert lib.cclr_ctx_bytes(None) == 0


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2307_14296_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".inc")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("the oracle pins", ""), os.path.join(dirpath, f)
