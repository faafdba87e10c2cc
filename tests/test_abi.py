"""The C-ABI library builds for sm_100a, loads, and exports every symbol include/tild.h declares
(no compute calls: there is no GPU on the build box)."""
import ctypes as C
import os
import re

import pytest

from paper_2302_02474_b200 import build as tbuild
from paper_2302_02474_b200 import tild

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    tbuild.build()
    return tild.load()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "tild.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(tild_[a-z_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert len(names) >= 15
    for name in names:
        assert hasattr(lib, name), name
    assert set(names) == set(tild.EXPORTS)


def test_params_struct_matches_header(lib):
    # tild_workspace_bytes validates struct_size == sizeof(tild_params) on the C side
    p = tild.make_params(1000, 2, (10.0,) * 3, (16,) * 3, 2, [[0, 1], [1, 0]], 50.0)
    nbytes = C.c_size_t(0)
    assert lib.tild_workspace_bytes(C.byref(p), C.byref(nbytes)) == tild.OK
    assert nbytes.value > 1000 * 12 * 4
    p.struct_size += 4
    assert lib.tild_workspace_bytes(C.byref(p), C.byref(nbytes)) == tild.EINVAL


@pytest.mark.parametrize("field,value", [("order", 0), ("order", 6), ("n_species", 0), ("n_species", 9), ("n", -1),
                                         ("max_bonds", 5), ("dt", 0.0), ("mass", -1.0)])
def test_invalid_params_are_rejected(lib, field, value):
    p = tild.make_params(1000, 2, (10.0,) * 3, (16,) * 3, 2, [[0, 1], [1, 0]], 50.0)
    setattr(p, field, value)
    nbytes = C.c_size_t(0)
    assert lib.tild_workspace_bytes(C.byref(p), C.byref(nbytes)) == tild.EINVAL


def test_invalid_box_and_grid(lib):
    nbytes = C.c_size_t(0)
    p = tild.make_params(10, 1, (10.0, 0.0, 10.0), (16,) * 3, 2, [[0]], 1.0)
    assert lib.tild_workspace_bytes(C.byref(p), C.byref(nbytes)) == tild.EINVAL
    p = tild.make_params(10, 1, (10.0,) * 3, (16, 3, 16), 4, [[0]], 1.0)     # grid < order
    assert lib.tild_workspace_bytes(C.byref(p), C.byref(nbytes)) == tild.EINVAL


def test_workspace_fits_180gb_for_c4(lib):
    from paper_2302_02474_b200 import inputs
    p = tild.params_from_config(inputs.C4)
    nbytes = C.c_size_t(0)
    assert lib.tild_workspace_bytes(C.byref(p), C.byref(nbytes)) == tild.OK
    assert nbytes.value < 8e9


def test_version_and_null_context(lib):
    assert b"sm_100a" in lib.tild_version()
    assert lib.tild_step(None, 1) == tild.EINVAL
    assert lib.tild_launch_count(None) == 0


def test_no_oracle_or_cpu_fallback_in_product():
    pkg = os.path.join(ROOT, "paper_2302_02474_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dirpath, f)).read()
                assert "tild_oracle" not in s and "from oracle" not in s and "import oracle" not in s, f
