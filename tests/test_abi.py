"""The C-ABI library loads and exports every symbol include/gf8.h declares (no compute without a GPU),
and argument errors are reported before anything touches the device."""
import ctypes as C
import os
import re

import pytest

from paper_2607_07494_b200 import build as gf8_build
from paper_2607_07494_b200 import gf8

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "gf8.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gf8_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    gf8_build.build()
    return gf8.lib()


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), f"{n} declared in gf8.h but not exported by libgf8.so"
    assert sorted(gf8.EXPORTS) == names                      # the binding covers the same surface


def test_no_torch_types_in_the_boundary():
    src = open(os.path.join(ROOT, "include", "gf8.h")).read()
    assert "torch" not in src and "at::" not in src and "#include <cuda" not in src


def test_argument_errors_before_any_launch(lib):
    h = C.c_void_p()
    d = (gf8.LayerDesc * 1)(gf8.LayerDesc(250, 256, 8, 8, 3, 0, 0, 1e-3, 0.0))      # d_out not a multiple of 16
    assert lib.gf8_create(C.byref(h), 0, d, 1, 0) == 3 and not h.value
    d = (gf8.LayerDesc * 1)(gf8.LayerDesc(256, 256, 0, 8, 3, 0, 0, 1e-3, 0.0))      # rank 0 on a used side
    assert lib.gf8_create(C.byref(h), 0, d, 1, 0) == 1
    d = (gf8.LayerDesc * 1)(gf8.LayerDesc(1024, 1024, 600, 8, 3, 0, 0, 1e-3, 0.0))   # rank > GF8_MAX_RANK
    assert lib.gf8_create(C.byref(h), 0, d, 1, 0) == 3
    d = (gf8.LayerDesc * 1)(gf8.LayerDesc(256, 256, 8, 8, 7, 0, 0, 1e-3, 0.0))      # bad side
    assert lib.gf8_create(C.byref(h), 0, d, 1, 0) == 1
    assert lib.gf8_create(None, 0, d, 1, 0) == 1
    assert lib.gf8_status_string(2) == b"bad state"
    assert lib.gf8_destroy(None) == 1


def test_binding_fails_loudly_without_library(monkeypatch, tmp_path):
    monkeypatch.setattr(gf8, "_lib", None)
    monkeypatch.setattr(gf8, "LIB_PATH", str(tmp_path / "missing.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        gf8.lib()
