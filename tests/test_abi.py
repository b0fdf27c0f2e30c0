"""CPU checks of the C-ABI boundary: the library loads, exports every symbol include/rick_b200.h
declares, and validates its arguments before touching CUDA (no compute calls here)."""
import ctypes as C
import os
import re

import pytest

from paper_2411_07321_b200 import binding as B
from paper_2411_07321_b200 import build as build_mod

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build_mod.build()
    return B.lib()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "rick_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rick_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_symbols()
    assert len(names) >= 12 and "rick_plan_create" in names and "rick_wcorrect_accumulate" in names
    for n in names:
        assert hasattr(lib, n), n
    assert set(names) == set(B.EXPORTS)


def test_argument_validation_needs_no_gpu(lib):
    h = C.c_void_p()
    bad = [
        (100, 8, 7, 1.0, -1.0, 1.0, 1e-3),     # N not a multiple of 32
        (256, 0, 7, 1.0, -1.0, 1.0, 1e-3),     # Nw < 1
        (256, 8, 8, 1.0, -1.0, 1.0, 1e-3),     # even support
        (256, 8, 17, 1.0, -1.0, 1.0, 1e-3),    # support too large
        (256, 8, 7, 0.0, -1.0, 1.0, 1e-3),     # sigma <= 0
        (256, 8, 7, 1.0, 1.0, 1.0, 1e-3),      # w_max <= w_min
        (256, 8, 7, 1.0, -1.0, 1.0, 0.0),      # dl <= 0
        (256, 8, 7, 1.0, -1.0, 1.0, 0.01),     # N dl >= sqrt 2
        (256, 8, 7, float("nan"), -1.0, 1.0, 1e-3),
    ]
    for args in bad:
        assert lib.rick_plan_create(*args, C.byref(h)) == -1, args
        assert h.value is None
    assert lib.rick_plan_create(256, 8, 7, 1.0, -1.0, 1.0, 1e-3, None) == -1
    assert lib.rick_plan_destroy(None) == -1
    assert lib.rick_grid(None, None, 1, None) == -1
    assert lib.rick_strerror(0) == b"ok"
    assert lib.rick_strerror(-1) == b"invalid argument"
    assert b"unknown" in lib.rick_strerror(-99)


def test_no_fallback_when_library_missing(monkeypatch, tmp_path):
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "library_path", lambda: str(tmp_path / "nope.so"))
    with pytest.raises(B.RickError):
        B.lib()


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2411_07321_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "rick_oracle" not in src and "import oracle" not in src and "from oracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "rick_oracle.cpp")).read() + open(os.path.join(ROOT, "oracle", "rick_oracle.py")).read()
    assert "rick_b200.h" not in osrc and "import paper_2411_07321_b200" not in osrc and "from paper_2411_07321_b200" not in osrc
