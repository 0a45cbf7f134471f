"""-m "not gpu": the C-ABI library loads and exports every symbol include/dc.h declares
(no compute calls without a GPU), and the host-side logic that needs no device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1711_07663_b200._build import build_lib
    return ctypes.CDLL(build_lib())


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "dc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dc_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_entry_points():
    names = declared_symbols()
    for must in ("dc_create_grid", "dc_set_cut_surface", "dc_classify", "dc_destroy"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    names = declared_symbols()
    assert len(names) >= 10
    for n in names:
        assert hasattr(lib, n), "libdc.so does not export %s" % n


def test_binding_lists_the_same_names():
    from paper_1711_07663_b200 import binding
    assert sorted(binding.EXPORTS) == declared_symbols()


def test_workspace_bytes_and_error_strings(lib):
    lib.dc_workspace_bytes.argtypes = [ctypes.c_longlong] * 4
    lib.dc_workspace_bytes.restype = ctypes.c_size_t
    assert lib.dc_workspace_bytes(0, 10, 10, 10) == 0          # bad argument -> 0
    assert lib.dc_workspace_bytes(10, -1, 10, 10) == 0
    a = lib.dc_workspace_bytes(35937, 4096, 96, 1 << 20)
    b = lib.dc_workspace_bytes(35937, 4096, 96, 1 << 22)
    assert 0 < a < b and a % 256 == 0
    lib.dc_error_string.restype = ctypes.c_char_p
    lib.dc_error_string.argtypes = [ctypes.c_int]
    seen = {lib.dc_error_string(c) for c in (0, -1, -2, -3, -4, -5)}
    assert len(seen) == 6 and all(s for s in seen)


def test_struct_layouts_match_header():
    # sizes the binding assumes == what the header implies (doubles then ints, natural alignment)
    from paper_1711_07663_b200 import binding
    assert ctypes.sizeof(binding.dc_params) == 4 * 8 + 2 * 4
    assert ctypes.sizeof(binding.dc_stats) == 27 * 8 + 3 * 8 + 8 * 4 + 8 * 4 + 4 * 4


def test_null_arguments_are_rejected_without_a_gpu(lib):
    lib.dc_set_cut_surface.argtypes = [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]
    assert lib.dc_set_cut_surface(None, 5, None, None) == -1
    lib.dc_classify.argtypes = [ctypes.c_void_p] * 5
    assert lib.dc_classify(None, None, None, None, None) == -1
    lib.dc_get_stats.argtypes = [ctypes.c_void_p, ctypes.c_void_p]
    assert lib.dc_get_stats(None, None) == -1
    lib.dc_destroy.argtypes = [ctypes.c_void_p]
    lib.dc_destroy(None)   # no-op
