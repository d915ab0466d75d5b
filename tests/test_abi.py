"""The C-ABI library loads on a box without a GPU and exports every symbol include/hs.h declares; argument
validation that needs no device is checked here (no compute calls)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def hs():
    from paper_1812_02647_b200 import build
    build.build()
    import paper_1812_02647_b200.binding as binding
    return binding


def declared_functions():
    text = open(os.path.join(ROOT, "include", "hs.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hs_[a-z_]+)\s*\(", text)))


def test_header_declares_the_three_north_star_calls():
    names = declared_functions()
    for n in ("hs_plan_create", "hs_execute", "hs_destroy"):
        assert n in names
    assert len(names) >= 12


def test_library_exports_every_declared_symbol(hs):
    raw = ctypes.CDLL(hs.LIB_PATH)
    for name in declared_functions():
        assert hasattr(raw, name), f"libhs.so does not export {name}"
    # and the binding wraps each of them with explicit argument types
    for name in declared_functions():
        assert getattr(hs.lib, name).argtypes is not None


def test_error_strings_and_version(hs):
    for code in range(0, 7):
        assert len(hs.lib.hs_error_string(code)) > 0
    assert b"unknown" in hs.lib.hs_error_string(99)
    assert b"sm_100a" in hs.lib.hs_version()


def test_create_validation_is_checked_before_the_device(hs):
    bad = [(0, 1, 32, 0, 1), (1001, 1, 32, 0, 1), (1 << 26, 1, 32, 0, 1), (1024, 0, 32, 0, 1), (1024, 1, 3, 0, 1),
           (1024, 1, 64, 0, 1), (1024, 1, 32, 4, 1), (1024, 1, 32, -1, 1), (1024, 1, 32, 0, 0), (1024, 1, 32, 0, 4),
           (1 << 25, 1 << 16, 32, 0, 1)]
    for args in bad:
        assert not hs.lib.hs_plan_create(*args)
        assert hs.lib.hs_last_error() == hs.HS_ERR_INVALID_ARG, args


def test_null_plan_helpers(hs):
    assert hs.lib.hs_destroy(None) == hs.HS_OK
    assert hs.lib.hs_plan_levels(None) == -1
    assert hs.lib.hs_plan_algo(None) == -1
    assert hs.lib.hs_plan_launches(None) == -1
    assert hs.lib.hs_plan_workspace_bytes(None) == 0
    assert hs.lib.hs_execute(None, None, None, None, None, None) == hs.HS_ERR_NULL_POINTER
    assert hs.lib.hs_last_error() == hs.HS_ERR_NULL_POINTER


def test_no_device_means_unsupported_not_a_fallback(hs):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(hs.HsError) as e:
        hs.hs_plan_create(1024, 1, 32, "standard", "full")
    assert e.value.code == hs.HS_ERR_UNSUPPORTED


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1812_02647_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "hs_oracle" not in src, f
    osrc = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "hs_oracle.c")).read()
    assert "import paper_1812_02647_b200" not in osrc and "from paper_1812_02647_b200" not in osrc and "hs.h" not in osrc
