"""The C-ABI library loads on a CPU-only box and exports every symbol include/ibcouple.h declares."""
import ctypes
import os
import re

from paper_2503_22695_b200 import build as ibbuild
from paper_2503_22695_b200 import ibcouple

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "ibcouple.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ib_[a-z_0-9]+)\s*\(", src)))


def test_library_builds_loads_and_exports_all_declared_symbols():
    so = ibbuild.build()
    assert os.path.exists(so)
    L = ctypes.CDLL(so)
    names = _declared()
    assert len(names) >= 16
    for n in names:
        assert hasattr(L, n), n
    assert sorted(ibcouple.EXPORTS) == names          # the binding covers exactly the header
    ibcouple.lib().ib_status_string.restype = ctypes.c_char_p
    assert ibcouple.lib().ib_status_string(0) == b"IB_OK"
    assert ibcouple.lib().ib_status_string(5) == b"IB_ERR_INVERTED_ELEMENT"


def test_argument_validation_without_a_gpu():
    # invalid arguments are rejected synchronously, before any CUDA call is made
    L = ibcouple.lib()
    h = ctypes.c_void_p(None)
    g = ibcouple.GridDesc(30, 32, 32, 0.1, 0, 0, 0, 1)          # nx not a multiple of 8
    md = ibcouple.MeshDesc(0, 0, None, None, None, None, None, None, 0)
    assert L.ib_create(ctypes.byref(h), ctypes.byref(g), ctypes.byref(md), 0) == 1
    g = ibcouple.GridDesc(32, 32, 32, -0.1, 0, 0, 0, 1)
    assert L.ib_create(ctypes.byref(h), ctypes.byref(g), ctypes.byref(md), 0) == 1
    g = ibcouple.GridDesc(32, 32, 32, 0.1, 0, 0, 0, 0)          # a bounded grid is fine ...
    dummy = (ctypes.c_int32 * 3)(1, 1, 1)
    md_t = ibcouple.MeshDesc(0, 0, None, None, None, None, ctypes.cast(dummy, ctypes.c_void_p), None, 0, 1)
    assert L.ib_create(ctypes.byref(h), ctypes.byref(g), ctypes.byref(md_t), 0) == 2     # ... sub-points on tets are not
    md_bad = ibcouple.MeshDesc(0, 0, None, None, None, None, None, None, 0, 7)            # unknown element type
    assert L.ib_create(ctypes.byref(h), ctypes.byref(g), ctypes.byref(md_bad), 0) == 1
    assert L.ib_create(None, ctypes.byref(g), ctypes.byref(md), 0) == 1
    assert L.ib_fe_force(None, None, None, None) == 1
    assert L.ib_destroy(None) == 1
