"""The C-ABI library loads and exports every symbol include/gpumcd.h declares (no GPU needed)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1101_1245_b200 import build
    build.build()
    import paper_1101_1245_b200 as g
    return g.load_library()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "gpumcd.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gpumcd_[a-z_]+)\s*\(", text)))


def test_header_declares_the_boundary_calls():
    syms = declared_symbols()
    for name in ("gpumcd_create", "gpumcd_set_source", "gpumcd_run"):   # BASELINE.json north_star
        assert name in syms
    assert len(syms) >= 11


def test_library_exports_every_declared_symbol(lib):
    from paper_1101_1245_b200 import binding
    for name in declared_symbols():
        assert hasattr(lib, name), name
        assert name in binding.EXPORTS


def test_struct_layouts_match_the_header(lib):
    from paper_1101_1245_b200 import binding as b
    assert ctypes.sizeof(b.gpumcd_options) == 76
    assert ctypes.sizeof(b.gpumcd_counters) == 14 * 8 + 5 * 8
    assert ctypes.sizeof(b.gpumcd_tables) == 64
    assert ctypes.sizeof(b.gpumcd_source) == 72
    opt = b.gpumcd_default_options()
    assert (opt.es_max_cm, opt.f_eloss_max, opt.pair_mode, opt.photon_only) == (0.5, 0.25, 1, 0)
    assert opt.wave_size == 1 << 20 and opt.bank_factor == 8 and opt.majorant_scale == 1.0


def test_argument_errors_do_not_need_a_device(lib):
    from paper_1101_1245_b200 import binding as b
    h = ctypes.c_void_p()
    assert lib.gpumcd_create(ctypes.byref(h), None, None, 4, 4, 4, ctypes.c_float(0.5), None, None) == b.GPUMCD_ERR_INVALID_ARG
    assert "null" in b.gpumcd_last_error(None)
    assert lib.gpumcd_default_options(None) == b.GPUMCD_ERR_INVALID_ARG
    assert lib.gpumcd_run(None, 1, 1, None, None) == b.GPUMCD_ERR_INVALID_ARG
    assert lib.gpumcd_set_source(None, None) == b.GPUMCD_ERR_INVALID_ARG
    lib.gpumcd_destroy(None)   # destroying nothing is allowed


def test_product_package_does_not_import_the_oracle():
    """The oracle is test infrastructure: nothing under the product package may reference it."""
    pkg = os.path.join(ROOT, "paper_1101_1245_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "oracle.h" not in src and "liborc" not in src, f
    ora = open(os.path.join(ROOT, "oracle", "oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "csrc" not in ora.replace("paper_1101_1245_b200/csrc", "") and "libgpumcd" not in ora
