"""Host-side checks that need no GPU: the C-ABI library loads and exports every symbol that
include/eigh.h declares; argument validation that launches nothing."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "eigh.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(eigh_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__ as ge
    ge.build()
    from paper_2310_03341_b200 import binding
    return binding.load()


def test_header_declares_the_boundary():
    names = declared_functions()
    for must in ("eigh_create", "eigh_workspace_size", "eigh_set_workspace", "eigh_solve", "eigh_destroy",
                 "eigh_last_error", "eigh_phase_times", "eigh_reduce_to_band", "eigh_band_to_tridiag",
                 "eigh_tridiag_dc", "eigh_backtransform_band", "eigh_backtransform_full"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    from paper_2310_03341_b200 import binding
    for name in declared_functions():
        assert hasattr(lib, name), f"{name} declared in include/eigh.h but not exported"
        assert name in binding.SIGNATURES, f"{name} has no binding signature"


def test_create_validates_arguments(lib):
    h = ctypes.c_void_p()
    assert lib.eigh_create(None, 4, 4) == -1
    assert lib.eigh_create(ctypes.byref(h), 0, 1) == -2
    assert lib.eigh_create(ctypes.byref(h), 4, 0) == -3
    assert lib.eigh_create(ctypes.byref(h), 4, 5) == -3
    assert lib.eigh_create(ctypes.byref(h), 4096, 4096) == 0
    assert lib.eigh_set_option(h, b"band_width", 48) == -3
    assert lib.eigh_set_option(h, b"nonsense", 1) == -2
    assert lib.eigh_set_option(h, b"band_width", 64) == 0
    ws = lib.eigh_workspace_size(h)
    assert ws > 4096 * 4096 * 8          # at least the packed reflectors
    # no workspace yet: every compute entry point refuses before launching anything
    assert lib.eigh_solve(h, None, 4096, None, None, None) == -1
    assert b"workspace" in lib.eigh_last_error(h)
    assert lib.eigh_set_workspace(h, ctypes.c_void_p(12345), ws) == -2      # misaligned
    assert lib.eigh_set_workspace(h, ctypes.c_void_p(4096), ws - 1) == -3   # too small
    assert lib.eigh_destroy(h) == 0


def test_workspace_fits_b200_at_largest_config(lib):
    """N = 49152 (config 4): A + Z + workspace must fit 180 GB of HBM3e."""
    h = ctypes.c_void_p()
    assert lib.eigh_create(ctypes.byref(h), 49152, 49152) == 0
    ws = lib.eigh_workspace_size(h)
    lib.eigh_destroy(h)
    mat = 49152 * 49152 * 16
    assert ws + 2 * mat < 176e9, (ws + 2 * mat) / 1e9


def test_option_change_invalidates_the_workspace(lib):
    """An option that grows the plan must not be usable with a workspace sized for the old plan
    (create -> workspace_size -> set_workspace -> set_option -> workspace_size -> solve)."""
    h = ctypes.c_void_p()
    assert lib.eigh_create(ctypes.byref(h), 2048, 2048) == 0
    ws_small = lib.eigh_workspace_size(h)
    assert lib.eigh_set_workspace(h, ctypes.c_void_p(1 << 20), ws_small) == 0
    assert lib.eigh_set_option(h, b"p4b_merge", 8) == 0
    ws_big = lib.eigh_workspace_size(h)
    assert ws_big > ws_small
    # nothing may be launched with the old buffer (the pointer is a dummy: a launch would fault)
    assert lib.eigh_solve(h, ctypes.c_void_p(1 << 20), 2048, ctypes.c_void_p(1 << 20), ctypes.c_void_p(1 << 20), None) == -1
    assert b"workspace" in lib.eigh_last_error(h)
    assert lib.eigh_set_workspace(h, ctypes.c_void_p(1 << 20), ws_small) == -3
    assert lib.eigh_destroy(h) == 0


def test_option_ranges_and_get_option(lib):
    h = ctypes.c_void_p()
    assert lib.eigh_create(ctypes.byref(h), 512, 512) == 0
    v = ctypes.c_int64()
    assert lib.eigh_get_option(h, b"band_width", ctypes.byref(v)) == 0 and v.value == 64
    assert lib.eigh_set_option(h, b"band_width", 128) == -3      # S2 / S4a are built for 64 only
    assert lib.eigh_set_option(h, b"dc_leaf", 4) == -3           # documented range 8..32
    assert lib.eigh_set_option(h, b"dc_leaf", 8) == 0
    assert lib.eigh_get_option(h, b"dc_leaf", ctypes.byref(v)) == 0 and v.value == 8
    assert lib.eigh_get_option(h, b"nonsense", ctypes.byref(v)) == -2
    assert lib.eigh_get_option(h, b"dc_leaf", None) == -3
    n = ctypes.c_int(-1)
    assert lib.eigh_dc_stats(h, 0, ctypes.byref(n), None, None) == 0 and n.value == 0
    assert lib.eigh_destroy(h) == 0
