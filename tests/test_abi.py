"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol that include/gmmnlse.h declares; the binding mirrors the header.  No compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "gmmnlse.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(gmmnlse_[a-z_0-9]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1708_05324_b200 import build
    return build.build()


def test_header_declares_the_three_named_calls():
    names = _declared()
    for n in ("gmmnlse_plan_create", "gmmnlse_propagate", "gmmnlse_nonlinear_op", "gmmnlse_plan_destroy"):
        assert n in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in _declared():
        assert hasattr(lib, name), f"{name} declared in gmmnlse.h but not exported"


def test_binding_covers_header(lib_path):
    from paper_1708_05324_b200 import binding
    assert sorted(binding.SIGNATURES) == _declared()
    lib = binding.load_library(lib_path)
    assert lib.gmmnlse_abi_version() >= 1
    assert lib.gmmnlse_status_string(0) == b"ok"
    assert b"invalid" in lib.gmmnlse_status_string(-1)


def test_no_torch_types_in_signatures():
    src = open(HEADER).read()
    assert "torch" not in src and "at::" not in src and "#include <cuda" not in src


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1708_05324_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f


def test_missing_library_fails_loudly(tmp_path):
    from paper_1708_05324_b200 import binding
    with pytest.raises(binding.GmmnlseError):
        binding.load_library(str(tmp_path / "nope.so"))
