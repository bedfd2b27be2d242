"""The C-ABI library loads and exports every symbol include/cst.h declares (no compute calls)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1910_12578_b200 import build, binding
    build.build()
    return ctypes.CDLL(binding.LIB_PATH)


def declared_symbols():
    txt = open(os.path.join(ROOT, "include", "cst.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(cst_[a-z_A-Z0-9]+)\s*\(", txt)))


def test_header_declares_the_path():
    syms = declared_symbols()
    for s in ("cst_create", "cst_destroy", "cst_fill_ghosts", "cst_advance_A", "cst_sdc_update",
              "cst_advance_A_update", "cst_cfl_dt", "cst_cfl_dt_device", "cst_strerror"):
        assert s in syms


def test_library_exports_every_declared_symbol(lib):
    for s in declared_symbols():
        assert hasattr(lib, s), f"libcst.so does not export {s}"


def test_binding_lists_the_same_symbols():
    from paper_1910_12578_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()


def test_params_struct_matches_header_layout():
    from paper_1910_12578_b200 import binding
    # 8 ints, 3+1+3 doubles, 6 ints, 2 doubles
    assert ctypes.sizeof(binding.CstParams) == 8 * 4 + 7 * 8 + 6 * 4 + 2 * 8


def test_strerror_and_version_without_gpu(lib):
    lib.cst_strerror.restype = ctypes.c_char_p
    lib.cst_version.restype = ctypes.c_char_p
    assert lib.cst_strerror(0) == b"ok"
    assert lib.cst_strerror(-1) == b"invalid argument"
    assert b"sm_100a" in lib.cst_version()


def test_create_rejects_bad_params_before_touching_the_gpu(lib):
    from paper_1910_12578_b200 import binding, workloads as wl
    cfg = wl.make_config(0)
    for bad in (dict(ng=3), dict(nx=2), dict(gamma=1.0), dict(dx=0.0), dict(nspec=60),
                dict(bc_lo=(0, 0, 0), bc_hi=(1, 0, 0))):
        c = dict(cfg); c.update(bad)
        h = ctypes.c_void_p()
        rc = lib.cst_create(ctypes.byref(binding.make_params(c)), ctypes.byref(h))
        assert rc == -1 and not h
    assert lib.cst_create(None, None) == -1


def test_oracle_and_product_share_no_code():
    """The product never imports the oracle, and the oracle never imports the product."""
    pk = os.path.join(ROOT, "paper_1910_12578_b200")
    for dirpath, _, files in os.walk(pk):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "orc.c" not in src.replace("oracle/", "")
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "binding" not in src and "libcst" not in src and "csrc/" not in src.replace("paper_1910_12578_b200/csrc", "")
