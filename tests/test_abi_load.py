"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every symbol
include/cdc_seedscan.h declares; the ctypes structs mirror the header; host-side validation that needs no GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1908_01949_b200 import binding as B
from paper_1908_01949_b200 import build as cdc_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "cdc_seedscan.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cdc_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    path = cdc_build.build()
    assert os.path.exists(path)
    lib = C.CDLL(path)
    names = _declared()
    assert len(names) >= 19
    for n in names:
        assert hasattr(lib, n), f"{n} declared in the header but not exported"
    assert sorted(B.EXPORTS) == names          # the binding covers the header, nothing more


def test_library_is_sm100a_native_code():
    """The fat binary must carry sm_100a SASS for the scan kernel (no PTX-JIT for another arch)."""
    import subprocess
    path = cdc_build.build()
    out = subprocess.run(["cuobjdump", "-lelf", path], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_struct_layouts_match_header():
    assert C.sizeof(B.GridSpec) == 5 * 8 + 5 * 8 + 5 * 4 + 5 * 4
    assert C.sizeof(B.ScanParams) == 56
    assert C.sizeof(B.HoughParams) == 72
    assert C.sizeof(B.ScanStats) == 80
    assert B.SEED_DEBUG_DTYPE.itemsize == 40
    assert C.sizeof(B.GeometryDesc) == 8 + 5 * 8 + 3 * 8
    assert C.sizeof(B.FieldDesc) == 64


def test_host_side_validation_without_gpu():
    lib = B.lib()
    dims = (C.c_int32 * 3)()
    assert lib.cdc_hough_dims(C.byref(B.hough_params()), dims) == 0
    assert tuple(dims) == (31, 230, 230)
    assert lib.cdc_hough_dims(C.byref(B.hough_params(bin_R_mm=0.0)), dims) == -1
    assert b"Hough" in lib.cdc_last_error()
    assert lib.cdc_hough_dims(None, dims) == -1
    # geometry validation happens before any CUDA call
    h = C.c_void_p()
    assert lib.cdc_geometry_create(None, None, C.byref(h)) == -1
    r = np.array([530.0, 546.5, 570.0]); n = np.array([198, 204, 211], dtype=np.int32)
    z = np.zeros(3); st = np.array([0.07, -0.07, 0.07])
    gd = B.GeometryDesc(3, r.ctypes.data, n.ctypes.data, z.ctypes.data, st.ctypes.data, None, 750.0, 500.0, 827.0)
    fd = B.FieldDesc(0, 1.0, 0, 0, 0.0, 0.0, 10.0, 10.0, None)
    assert lib.cdc_geometry_create(C.byref(gd), C.byref(fd), C.byref(h)) == -1     # unequal layer pitch
    assert b"equally spaced" in lib.cdc_last_error()
    assert lib.cdc_fp32_peak_probe(C.c_int32(0), None, None, None) == -1
    assert lib.cdc_scan_get_stats(None, None, None) == -1


def test_no_cpu_fallback_in_product_path():
    """The product package never imports the oracle."""
    pkg = os.path.join(ROOT, "paper_1908_01949_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f
