"""CPU-only checks of the boundary: the shared library builds/loads and exports every symbol include/fhe.h declares,
and the binding's prototype table covers the same set.  No compute calls (no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _header_symbols():
    text = open(os.path.join(ROOT, "include", "fhe.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fhe_[a-z0-9_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_05920_b200 import build
    build.build()
    import paper_2607_05920_b200 as fhe
    return fhe, fhe.load_library()


def test_header_declares_the_northstar_calls():
    syms = _header_symbols()
    for name in ("fhe_ctx_create", "fhe_polymul", "fhe_he_mult", "fhe_relinearize", "fhe_rescale"):
        assert name in syms


def test_library_exports_every_declared_symbol(lib):
    fhe, cdll = lib
    syms = _header_symbols()
    assert sorted(fhe.EXPORTS) == syms
    for name in syms:
        assert isinstance(getattr(cdll, name), ctypes._CFuncPtr)


def test_null_context_calls_return_arg_errors(lib):
    """Argument checks that happen before any CUDA call are safe to exercise without a GPU."""
    fhe, cdll = lib
    assert cdll.fhe_workspace_bytes(None, 0, 4) == 0
    assert cdll.fhe_polymul(None, None, None, None, 1, None, 0, None) == fhe.FHE_ERR_ARG
    assert cdll.fhe_rescale(None, None, None, 1, 1, None) == fhe.FHE_ERR_ARG
    assert cdll.fhe_debug_launch_count(None) == 0
    out = ctypes.c_void_p()
    # unsupported parameters are rejected before the device is touched
    assert cdll.fhe_ctx_create(ctypes.byref(out), 100, 128, 128, 0) == fhe.FHE_ERR_UNSUPPORTED
    assert cdll.fhe_ctx_create(ctypes.byref(out), 1024, 128, 128, 4) == fhe.FHE_ERR_UNSUPPORTED
    assert b"power of two" in cdll.fhe_last_error(None) or b"odd" in cdll.fhe_last_error(None)
    assert out.value is None


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2607_05920_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".hpp", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
