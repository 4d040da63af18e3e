"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/dedisp.h declares; the Python binding has the same names.  No compute call is made."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "dedisp.h")


def _declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)  # drop comments
    return sorted(set(re.findall(r"\b(dedisp_[a-z_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib_path():
    from paper_1601_01165_b200 import build
    return build.build()


def test_header_declares_the_north_star_calls():
    syms = _declared_symbols()
    for name in ("dedisp_plan_create", "dedisp_shift_table", "dedisp_execute", "dedisp_plan_destroy",
                 "dedisp_tune"):
        assert name in syms


def test_library_exports_every_declared_symbol(lib_path):
    lib = ctypes.CDLL(lib_path)
    for name in _declared_symbols():
        assert hasattr(lib, name), "libdedisp_b200.so does not export %s" % name


def test_binding_lists_every_declared_symbol(lib_path):
    from paper_1601_01165_b200 import dedisp
    assert sorted(dedisp.SYMBOLS) == _declared_symbols()
    dedisp.load_library()


def test_variant_registry_is_readable_without_a_gpu(lib_path):
    from paper_1601_01165_b200 import dedisp
    n = dedisp.variant_count()
    assert n >= 4
    names = [dedisp.variant_name(v) for v in range(n)]
    assert len(set(names)) == n, "variant names are the tuning-cache keys: must be unique"
    assert names[0].startswith("generic_f32") and names[1].startswith("generic_u8")
    assert dedisp.variant_name(n) is None and dedisp.variant_name(-1) is None
    assert any(s.startswith("tree_f32") for s in names) and any(s.startswith("tree_u8") for s in names)
    assert any(s.startswith("lds_u8") for s in names)


def test_status_strings(lib_path):
    from paper_1601_01165_b200 import dedisp
    lib = dedisp.load_library()
    assert lib.dedisp_status_string(0) == b"ok"
    assert len({lib.dedisp_status_string(i) for i in range(6)}) == 6


def test_argument_errors_do_not_need_a_device(lib_path):
    """INVALID_ARG / OVERFLOW are decided before any CUDA call (header contract)."""
    from paper_1601_01165_b200 import dedisp
    lib = dedisp.load_library()
    h = ctypes.c_void_p(123)
    bad = [
        (0, 1420.0, 1.0, 1000.0, 16, 0.0, 1.0, 4, 0),      # C < 1
        (4, 1420.0, 1.0, 1000.0, 0, 0.0, 1.0, 4, 0),       # S < 1
        (4, 1420.0, 1.0, 1000.0, 16, 0.0, 1.0, 0, 0),      # D < 1
        (4, -1.0, 1.0, 1000.0, 16, 0.0, 1.0, 4, 0),        # f_low <= 0
        (4, 1420.0, 0.0, 1000.0, 16, 0.0, 1.0, 4, 0),      # bw <= 0
        (4, 1420.0, 1.0, float("nan"), 16, 0.0, 1.0, 4, 0),
        (4, 1420.0, 1.0, 1000.0, 16, -1.0, 1.0, 4, 0),     # negative DM (reading A11)
        (4, 1420.0, 1.0, 1000.0, 16, 0.0, -1.0, 4, 0),
        (4, 1420.0, 1.0, 1000.0, 16, 0.0, 1.0, 4, 7),      # unknown dtype
    ]
    for args in bad:
        h.value = 123
        rc = lib.dedisp_plan_create(ctypes.byref(h), *args)
        assert rc == 1, args
        assert h.value is None, "*plan must be NULL on error"
    assert lib.dedisp_plan_create(None, 4, 1420.0, 1.0, 1000.0, 16, 0.0, 1.0, 4, 0) == 1
    # uint8 sums must fit uint32
    rc = lib.dedisp_plan_create(ctypes.byref(h), 2 ** 25, 1420.0, 1.0, 1000.0, 16, 0.0, 1.0, 4, 1)
    assert rc == 2
    assert lib.dedisp_plan_destroy(None) == 0
    assert lib.dedisp_execute(None, None, None, 1, None) == 1
