"""Host-side checks that need no GPU: libgs.so builds, loads, and exports exactly the C ABI that
include/gs.h declares; without a CUDA device the product path fails loudly (no CPU fallback)."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built():
    from paper_2502_02460_b200 import build
    return build.build()


def _declared():
    text = open(os.path.join(ROOT, "include", "gs.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gs_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = _declared()
    for required in ("gs_plan_create", "gs_cholesky", "gs_invert_triangular", "gs_to_standard", "gs_backtransform"):
        assert required in names


def test_library_exports_every_declared_symbol(built):
    from paper_2502_02460_b200 import gs
    L = ctypes.CDLL(gs.LIB_PATH)
    for name in _declared():
        assert hasattr(L, name), f"{name} declared in include/gs.h but not exported by libgs.so"
    assert sorted(gs.EXPORTS) == _declared()


def test_binding_has_no_torch_types_in_signatures():
    text = open(os.path.join(ROOT, "include", "gs.h")).read()
    assert "torch" not in text.lower() and "at::" not in text


def test_status_strings(built):
    from paper_2502_02460_b200 import gs
    L = gs.lib()
    assert L.gs_status_string(0) == b"GS_OK"
    assert L.gs_status_string(2) == b"GS_ERR_NOT_POSDEF"
    assert L.gs_status_string(6) == b"GS_ERR_UNSUPPORTED_DEVICE"


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_device_fails_loudly(built):
    """No CPU fallback: plan creation reports GS_ERR_UNSUPPORTED_DEVICE instead of computing."""
    from paper_2502_02460_b200 import gs
    L = gs.lib()
    h = ctypes.c_void_p()
    status = L.gs_plan_create(ctypes.byref(h), 64, gs.GS_REAL64, 64)
    assert status == 6 and not h


def test_invalid_arguments_without_device(built):
    from paper_2502_02460_b200 import gs
    L = gs.lib()
    h = ctypes.c_void_p()
    assert L.gs_plan_create(ctypes.byref(h), 0, gs.GS_REAL64, 0) == 1
    assert L.gs_plan_create(ctypes.byref(h), 8, gs.GS_REAL64, 9) == 1
    assert L.gs_plan_create(None, 8, gs.GS_REAL64, 8) == 1
    assert L.gs_plan_destroy(None) == 1


def test_product_does_not_import_the_oracle():
    """The product path must not route through oracle/ (voids parity claims)."""
    pkg = os.path.join(ROOT, "paper_2502_02460_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text, f
                assert "gs_oracle" not in text and "liboracle" not in text, f
    otext = open(os.path.join(ROOT, "oracle", "gs_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "paper_2502_02460_b200" not in otext.replace("paper_2502_02460_b200/csrc, include/gs.h", "").replace(
        "imports nothing from paper_2502_02460_b200", "")
