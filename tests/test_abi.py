"""The C-ABI library builds for sm_100a, loads, and exports every symbol include/tt.h declares
(no compute calls: this runs without a GPU)."""
import ctypes
import os
import re

import numpy as np

from paper_1411_3968_b200 import _build
from paper_1411_3968_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "tt.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tt_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    path = _build.build()
    lib = ctypes.CDLL(path)
    names = _declared()
    assert {"tt_sort_slice", "tt_trigger_slice", "tt_extract_events", "tt_geometry_create"} <= set(names)
    for name in names:
        assert hasattr(lib, name), name
    assert sorted(B.EXPORTS) == names
    lib.tt_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.tt_version()


def test_struct_layouts_match_header():
    assert ctypes.sizeof(B.TTParams) == 40
    assert B.HIT_DTYPE.itemsize == 16 and B.EVENT_DTYPE.itemsize == 32
    assert B.RAW_DTYPE.itemsize == 16 and B.L1HIT_DTYPE.itemsize == 16  # tt_raw_hit, tt_l1hit: time first, like a hit
    assert B.RAW_DTYPE.fields["t_ps"][1] == 0 and B.L1HIT_DTYPE.fields["t_ps"][1] == 0 and B.L1HIT_DTYPE.fields["idx"][1] == 8
    assert [B.TTParams.lc_window_ps.offset, B.TTParams.l2_window_ps.offset, B.TTParams.event_half_ps.offset,
            B.TTParams.l2_multiplicity.offset, B.TTParams.l2_mode.offset, B.TTParams.q_thresh.offset] == [0, 8, 16, 24, 28, 32]


def test_argument_errors_without_gpu():
    """Argument validation and workspace queries are host-only and work without a device."""
    lib = B.load()
    need = ctypes.c_size_t(0)
    seg = np.array([0, 1000], dtype=np.uint32)
    z = ctypes.c_void_p(0)
    rc = lib.tt_sort_slice(z, z, z, ctypes.c_uint32(1000), z, seg.ctypes.data_as(ctypes.c_void_p), ctypes.c_uint32(1),
                           z, z, ctypes.c_uint32(0), z, ctypes.byref(need), z, z)
    assert rc == 0 and need.value > 1000 * 24
    bad = np.array([0, 999], dtype=np.uint32)  # does not end at n
    rc = lib.tt_sort_slice(z, z, z, ctypes.c_uint32(1000), z, bad.ctypes.data_as(ctypes.c_void_p), ctypes.c_uint32(1),
                           z, z, ctypes.c_uint32(0), z, ctypes.byref(need), z, z)
    assert rc == B.TT_E_INVAL
    # workspace queries of the fused call and of the by-tower / preparation calls: host-only too
    import ctypes as C

    geo_dummy = (C.c_char * 64)()
    prm = B.make_params()
    rc = lib.tt_sort_trigger_slice(z, z, z, C.c_uint32(1000), z, seg.ctypes.data_as(C.c_void_p), C.c_uint32(1), z, z,
                                   C.c_uint32(0), C.byref(geo_dummy), C.byref(prm), z, z, C.c_uint32(10), z, z, C.byref(need), z, z)
    assert rc == 0 and need.value > 1000 * 60
    rc = lib.tt_l1_export(z, C.c_uint32(1000), z, C.c_uint32(70000), z, C.c_uint32(0), z, z, C.byref(need), z, z)
    assert rc == B.TT_E_INVAL  # src must fit 16 bits
    rc = lib.tt_prepare_slice(z, z, C.c_uint32(1000), C.c_uint32(0), z, seg.ctypes.data_as(C.c_void_p), C.c_uint32(1),
                              C.c_uint32(84), z, C.c_uint32(999), z, z, C.byref(need), z, z)
    assert rc == B.TT_E_INVAL  # more raw hits than the output buffer holds
    rc = lib.tt_prepare_slice(z, z, C.c_uint32(1000), C.c_uint32(0), z, seg.ctypes.data_as(C.c_void_p), C.c_uint32(1),
                              C.c_uint32(84), z, C.c_uint32(1000), z, z, C.byref(need), z, z)
    assert rc == 0 and need.value > 1000 * 24
    # runs that straddle a segment are rejected
    seg2 = np.array([0, 500, 1000], dtype=np.uint32)
    runs = np.array([0, 400, 1000], dtype=np.uint32)
    one = ctypes.c_void_p(256)  # any non-null "device" pointer: rejected before use
    rc = lib.tt_sort_slice(z, z, z, ctypes.c_uint32(1000), z, seg2.ctypes.data_as(ctypes.c_void_p), ctypes.c_uint32(2),
                           one, runs.ctypes.data_as(ctypes.c_void_p), ctypes.c_uint32(2), z, ctypes.byref(need), z, z)
    assert rc == B.TT_E_INVAL


def test_product_path_never_imports_oracle():
    """The package and bench's product arm must not route through oracle/ (no CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_1411_3968_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f
