"""No-GPU checks of the C ABI: the library loads, exports every symbol include/carve.h declares,
and validates arguments on the host before touching a device."""
import ctypes
import os
import re

import pytest

from paper_2606_27229_b200 import build, carve

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return carve.load_library()


def test_header_symbols_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "carve.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(carve_[a-z_]+)\s*\(", hdr))
    assert declared == set(carve.SYMBOLS)
    for name in declared:
        assert getattr(lib, name) is not None
    assert "sm_100a" in carve.carve_version()


def test_status_strings(lib):
    for s in range(9):
        assert len(lib.carve_status_string(s)) > 0


def _p(**kw):
    d = dict(B=1, H=1, T=64, L=64, dk=64, dv=64, r=8, dtype=carve.CARVE_F32)
    d.update(kw)
    return carve.Params(**d)


def test_workspace_and_shape_validation(lib):
    assert carve.carve_workspace_bytes(_p(), True) > 0
    assert carve.carve_workspace_bytes(_p(), False) == 0
    for bad in (dict(T=65), dict(L=48), dict(dk=96), dict(dv=512), dict(r=12), dict(dtype=7), dict(dk=256, dv=256)):
        assert carve.carve_workspace_bytes(_p(**bad), True) == 0, bad
    # backward needs dk*dv <= 16384; forward takes up to 32768
    assert carve.carve_resolved_path(_p(dk=128, dv=256, r=16), False) == carve.CARVE_PATH_SIMT
    assert carve.carve_resolved_path(_p(dk=128, dv=256, r=16), True) == -1
    assert carve.carve_num_launches(_p(), False) >= 1


def test_argument_errors_before_any_launch(lib):
    """NULL / shape / alignment / workspace errors are reported without a device (error codes 1,2,4,5)."""
    cp = _p().c()
    nul = [None] * 16
    assert lib.carve_fwd(ctypes.byref(cp), *nul, None, 0, None) == 1            # CARVE_ERR_NULL
    bad = _p(T=100).c()
    assert lib.carve_fwd(ctypes.byref(bad), *nul, None, 0, None) == 2           # CARVE_ERR_SHAPE
    for empty in (dict(T=0), dict(B=0), dict(H=0)):                             # empty inputs: refused, never launched
        e = _p(**empty).c()
        assert lib.carve_fwd(ctypes.byref(e), *nul, None, 0, None) == 2, empty
        assert carve.carve_workspace_bytes(_p(**empty), True) == 0, empty
    buf = (ctypes.c_char * 4096)()
    base = (ctypes.addressof(buf) + 255) & ~255
    ptrs = [ctypes.c_void_p(base)] * 16
    ptrs[0] = ctypes.c_void_p(base + 4)
    assert lib.carve_fwd(ctypes.byref(cp), *ptrs, None, 0, None) == 4           # CARVE_ERR_ALIGN
    ptrs[0] = ctypes.c_void_p(base)
    assert lib.carve_fwd(ctypes.byref(cp), *ptrs, ctypes.c_void_p(base), 16, None) == 5   # CARVE_ERR_WORKSPACE


def test_binding_fails_loudly_without_library(monkeypatch):
    monkeypatch.setattr(carve, "_lib", None)
    monkeypatch.setattr(carve, "LIB_PATH", "/nonexistent/libcarve.so")
    with pytest.raises(FileNotFoundError):
        carve.carve_version()
