"""CPU-side checks of the C-ABI boundary: the CUDA library builds for sm_100a, loads without a GPU and
exports every symbol include/rt.h declares.  No compute calls here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    with open(os.path.join(ROOT, "include", "rt.h")) as fh:
        text = fh.read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rt_[a-z_0-9]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = declared_symbols()
    for must in ("rt_grid_create", "rt_set_opacity", "rt_explicit_step", "rt_implicit_step", "rt_cfl_dt"):
        assert must in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2606_26268_b200 import build
    path = build.build()
    assert os.path.exists(path)
    L = ctypes.CDLL(path)
    for name in declared_symbols():
        assert hasattr(L, name), "librt_m1.so does not export %s" % name


def test_binding_covers_every_declared_symbol():
    from paper_2606_26268_b200 import rt
    assert rt.exported_symbols() == declared_symbols()


def test_structs_match_the_header_layout():
    from paper_2606_26268_b200 import rt
    # rt_params: 5 doubles + 3 int32 (+4 pad); rt_opacity: see include/rt.h
    assert ctypes.sizeof(rt.Params) == 56
    assert ctypes.sizeof(rt.Opacity) == 8 + 7 * 8 + 8 + 6 * 8 + 8


def test_null_handle_calls_fail_cleanly_without_a_gpu():
    from paper_2606_26268_b200 import rt
    L = rt.lib()
    assert L.rt_grid_destroy(None) == rt.ERR_INVALID_ARG
    assert L.rt_set_params(None, None) == rt.ERR_INVALID_ARG
    assert L.rt_get_launch_count(None) == 0
    assert b"null" in L.rt_last_error(None)


@pytest.mark.skipif(__import__("torch").cuda.is_available(), reason="checks the no-GPU behaviour")
def test_product_path_fails_loudly_without_a_gpu():
    import numpy as np
    from paper_2606_26268_b200 import rt
    with pytest.raises(RuntimeError):
        rt.Grid(rt.CARTESIAN, (8, 1, 1), np.linspace(0, 1, 9), [0, 1], [0, 1], (0,) * 6)
    # and the C call itself reports RT_ERR_CUDA instead of computing anything on the CPU
    n = (ctypes.c_int32 * 3)(8, 1, 1)
    bc = (ctypes.c_int32 * 6)(*([0] * 6))
    x1 = (ctypes.c_double * 9)(*np.linspace(0, 1, 9))
    x2 = (ctypes.c_double * 2)(0.0, 1.0)
    h = ctypes.c_void_p()
    rc = rt.lib().rt_grid_create(0, n, 2, x1, x2, x2, bc, None, ctypes.byref(h))
    assert rc == rt.ERR_CUDA and not h.value
