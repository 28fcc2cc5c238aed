"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol that
include/mrhs.h declares; the layout helpers that need no GPU return the documented values."""
import os
import re

import pytest

import paper_2211_13719_b200 as mrhs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "mrhs.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mrhs_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported():
    from paper_2211_13719_b200 import build
    build.build()
    lib = mrhs.lib()
    declared = _declared_symbols()
    assert len(declared) >= 20
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(mrhs.EXPORTED_SYMBOLS) == declared


def test_version_and_error_string():
    assert "sm_100a" in mrhs.version()
    assert isinstance(mrhs.last_error(), str)


def test_field_bytes_and_xblock():
    assert mrhs.field_bytes([4, 4, 4, 4], 12, 4, False) == 256 * 12 * 4 * 8
    assert mrhs.field_bytes([4, 4, 4, 4], 12, 4, True) == 128 * 12 * 4 * 8
    assert mrhs.field_bytes([8, 8, 8, 8], 24, 12, False) == 4096 * 24 * 12 * 8
    assert mrhs.field_bytes([3, 4, 4, 4], 12, 4, True) == 0      # odd extent cannot be checkerboarded
    assert mrhs.field_bytes([1, 4, 4, 4], 12, 4, False) == 0
    assert mrhs.xblock(48, 12) == 8 and mrhs.xblock(24, 12) == 8 and mrhs.xblock(12, 12) == 6
    assert mrhs.xblock(48, 24) == 4 and mrhs.xblock(48, 48) == 2 and mrhs.xblock(48, 96) == 1
    assert mrhs.xblock(48, 1) == 16 and mrhs.xblock(4, 4) == 4 and mrhs.xblock(2, 4) == 2
    assert mrhs.xblock(0, 4) == 0


def test_invalid_arguments_are_reported_without_a_gpu():
    # argument checks come before any CUDA call
    with pytest.raises(mrhs.MrhsError) as e:
        mrhs.lib()  # ensure loaded
        mrhs._check(mrhs.lib().mrhs_dhop(None, None, None))
    assert e.value.status == mrhs.ERR_INVALID_ARG
    assert "NULL" in mrhs.last_error()
    h = mrhs._vp()
    import ctypes
    st = mrhs.lib().mrhs_wilson_create(ctypes.byref(h), mrhs._dims([4, 4, 3, 4]), 4, 0.0, 1.0,
                                       mrhs._vp(16), None, None)
    assert st == mrhs.ERR_INVALID_ARG and "even" in mrhs.last_error()
    st = mrhs.lib().mrhs_wilson_create(ctypes.byref(h), mrhs._dims([4, 4, 4, 4]), 1000, 0.0, 1.0,
                                       mrhs._vp(16), None, None)
    assert st == mrhs.ERR_UNSUPPORTED
    st = mrhs.lib().mrhs_coarse_create(ctypes.byref(h), mrhs._dims([4, 4, 4, 4]), 32, 4, mrhs._vp(16), 0, None)
    assert st == mrhs.ERR_UNSUPPORTED and "nbasis" in mrhs.last_error()
    st = mrhs.lib().mrhs_coarse_create(ctypes.byref(h), mrhs._dims([4, 4, 4, 1]), 24, 4, mrhs._vp(16), 0, None)
    assert st == mrhs.ERR_INVALID_ARG
