"""CPU-side checks of the boundary: libpmforce.so builds, loads, and exports every symbol that
include/pmforce.h declares (no compute calls without a GPU); the Python binding declares the same names."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "pmforce.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b((?:pm|nufft)_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


@pytest.fixture(scope="module")
def lib_path():
    from paper_2510_05206_b200 import build

    return build.build()


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for required in ("pm_assign", "pm_poisson_force", "pm_interp", "nufft_spread", "nufft_interp", "pm_assign_vjp",
                     "pm_poisson_force_vjp", "pm_interp_vjp", "nufft_spread_vjp", "nufft_interp_vjp", "pm_force",
                     "pm_force_vjp", "pm_bin", "pm_create", "pm_destroy"):
        assert required in names


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in declared_functions():
        assert hasattr(lib, name), f"{name} declared in pmforce.h but not exported"


def test_binding_covers_every_declared_symbol():
    from paper_2510_05206_b200 import api

    assert sorted(api.EXPORTED_SYMBOLS) == declared_functions()


def test_host_only_calls(lib_path):
    """Calls that need no device: error strings and NULL handling."""
    lib = ctypes.CDLL(lib_path)
    lib.pm_strerror.restype = ctypes.c_char_p
    assert lib.pm_strerror(0) == b"ok"
    assert lib.pm_strerror(-1) == b"invalid argument"
    assert lib.pm_create(None, None) == -1
    assert lib.pm_destroy(None) == 0


def test_no_product_import_of_the_oracle():
    """The product path must not import, read or call anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_2510_05206_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.replace("no CPU fallback", ""), f
