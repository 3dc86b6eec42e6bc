"""Host-side checks that need no GPU: the C-ABI library loads, exports every symbol include/lst.h
declares, and validates its arguments."""
import ctypes as C
import os
import re
import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import __graft_entry__ as ge
    ge.build()
    import paper_2403_13166_b200 as P
    return P.load_library()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "lst.h")).read()
    names = set(re.findall(r"^\s*(?:int|void)\s+(lst_\w+)\s*\(", hdr, flags=re.M))
    assert {"lst_create", "lst_load_event", "lst_run", "lst_get", "lst_workspace_bytes", "lst_destroy"} <= names
    for n in names:
        assert hasattr(lib, n), n
    assert lib.lst_launches_per_run() >= 10


def _geo_struct(P, geo, w):
    from paper_2403_13166_b200.binding import _Geometry, _hp
    keep = [np.ascontiguousarray(geo.subdet, np.uint8), np.ascontiguousarray(geo.mtype, np.uint8),
            np.ascontiguousarray(geo.conn_rowptr, np.int32), np.ascontiguousarray(geo.conn_col, np.int32),
            np.ascontiguousarray(w, np.float32)]
    return _Geometry(int(geo.n_modules), *[_hp(a) for a in keep], None, 0, 0), keep


def test_workspace_bytes_and_validation(lib, geo_full):
    import paper_2403_13166_b200 as P
    from paper_2403_13166_b200.binding import _Caps
    from dataclasses import asdict
    from lstgen import xavier_weights
    g, keep = _geo_struct(P, geo_full, xavier_weights(1))
    n = C.c_size_t(0)
    c1 = _Caps(**asdict(P.default_caps(1)))
    assert lib.lst_workspace_bytes(C.byref(g), C.byref(c1), C.byref(n)) == 0
    one = n.value
    c4 = _Caps(**asdict(P.default_caps(4)))
    assert lib.lst_workspace_bytes(C.byref(g), C.byref(c4), C.byref(n)) == 0
    assert one < n.value < 4 * one + (1 << 20) and one < (1 << 28)     # per-slot state, shared geometry
    # malformed inputs -> LST_EINVAL, never a crash
    assert lib.lst_workspace_bytes(None, C.byref(c1), C.byref(n)) == -1
    bad = _Caps(**asdict(P.default_caps(1))); bad.max_md = 0
    assert lib.lst_workspace_bytes(C.byref(g), C.byref(bad), C.byref(n)) == -1
    col = keep[3].copy(); col[3], col[4] = col[4], col[3]          # unsorted row
    g2, k2 = _geo_struct(P, geo_full, xavier_weights(1)); g2.conn_col = col.ctypes.data_as(C.c_void_p)
    assert lib.lst_workspace_bytes(C.byref(g2), C.byref(c1), C.byref(n)) == -1
    col = keep[3].copy(); col[0] = geo_full.n_modules               # column out of range
    g2.conn_col = col.ctypes.data_as(C.c_void_p)
    assert lib.lst_workspace_bytes(C.byref(g2), C.byref(c1), C.byref(n)) == -1
    rp = keep[2].copy(); rp[5] = rp[4] - 1                          # non-monotone rowptr
    g3, k3 = _geo_struct(P, geo_full, xavier_weights(1)); g3.conn_rowptr = rp.ctypes.data_as(C.c_void_p)
    assert lib.lst_workspace_bytes(C.byref(g3), C.byref(c1), C.byref(n)) == -1
    # null context / bad slot on the other entry points
    assert lib.lst_run(None, 0, None) == -1
    assert lib.lst_get(None, 0, 0, None) == -1


def test_product_path_never_imports_oracle():
    import subprocess, sys
    code = ("import sys; import paper_2403_13166_b200, lstgen; "
            "assert not any(m == 'oracle' or m.startswith('oracle.') for m in sys.modules), 'oracle imported'")
    subprocess.check_call([sys.executable, "-c", code], cwd=ROOT)
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2403_13166_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"(^|\n)\s*(from|import)\s+oracle|#include\s+[\"<][^\n]*oracle|lst_oracle", txt), f
