"""CPU checks of the C-ABI library: it builds, loads, exports every symbol include/wbmm.h
declares, validates arguments, and refuses to compute without a GPU (no CPU fallback)."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def wb():
    from paper_2607_02097_b200 import build
    build.build()
    import paper_2607_02097_b200 as wb
    return wb


def test_exports_match_header(wb):
    from paper_2607_02097_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "wbmm.h")).read()
    declared = set(re.findall(r"WBMM_API[^;(]*?\b(wbmm_\w+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    L = ctypes.CDLL(binding.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), name
    assert wb.wbmm_version() == 100


def test_desc_struct_matches_header(wb):
    assert ctypes.sizeof(wb.WbmmDesc) == 40
    names = [f[0] for f in wb.WbmmDesc._fields_]
    assert names == ["B", "C", "H", "W", "w", "shift_h", "shift_w", "dtype", "layout", "flags"]


def test_strings(wb):
    assert wb.wbmm_status_string(0) == "ok"
    assert wb.wbmm_status_string(3) == "no sm_100 CUDA device"
    assert wb.wbmm_path_string(wb.PATH_SIMT) == "simt"
    assert wb.wbmm_path_string(wb.PATH_TC_TMA) == "tcgen05+tma"


def test_argument_validation_without_gpu(wb):
    from paper_2607_02097_b200 import binding
    L = binding.lib()
    d = wb.WbmmDesc(1, 1, 4, 4, 2, 0, 0, 0, 0, 0)
    buf = (ctypes.c_float * 64)()
    p = ctypes.addressof(buf)
    assert L.wbmm_forward(None, p, p, p, None) == 1
    assert L.wbmm_forward(ctypes.byref(d), None, p, p, None) == 1
    assert L.wbmm_forward(ctypes.byref(d), p, p, p, None) == 1          # y aliases x
    for field, val in (("w", 0), ("H", 0), ("shift_h", 2), ("shift_w", -1), ("dtype", 7), ("layout", 2), ("B", -1)):
        bad = wb.WbmmDesc(1, 1, 4, 4, 2, 0, 0, 0, 0, 0)
        setattr(bad, field, val)
        assert L.wbmm_forward(ctypes.byref(bad), p, p + 128, p + 64, None) == 1, field
    assert L.wbmm_forward(ctypes.byref(d), p + 2, p + 128, p + 64, None) == 5   # misaligned fp32
    assert L.wbmm_backward(ctypes.byref(d), p, None, p + 64, p + 128, None, None) == 1  # dx needs T


def test_argument_validation_of_the_extended_entry_points(wb):
    """Hierarchical / cached-M / fused / fold entry points: argument errors are reported before any device work."""
    from paper_2607_02097_b200 import binding
    L = binding.lib()
    buf = (ctypes.c_float * 4096)()
    p = ctypes.addressof(buf)
    d14 = wb.WbmmDesc(1, 1, 14, 14, 14, 0, 0, 1, 0, 0)
    odd = wb.WbmmDesc(1, 1, 14, 14, 7, 0, 0, 1, 0, 0)
    assert L.wbmm_hier_forward(ctypes.byref(odd), p, p + 64, p + 128, p + 4096, 0, None) == 1        # w must be even
    assert L.wbmm_hier_forward(ctypes.byref(d14), p, None, p + 128, p + 4096, 0, None) == 1
    assert L.wbmm_hier_backward(ctypes.byref(d14), p, p + 64, p + 128, p + 256, None, p + 512, None, None) == 1   # dTg without dTl
    assert L.wbmm_hier_backward(ctypes.byref(odd), p, p + 64, p + 128, p + 256, p + 4096, None, None, None) == 1
    assert L.wbmm_forward_matrix(ctypes.byref(d14), p, None, None, p + 4096, 0, None) == 1
    assert L.wbmm_forward_matrix(ctypes.byref(d14), p, p + 64, None, p, 0, None) == 1                # y aliases x
    assert L.wbmm_forward_fused(ctypes.byref(d14), p, None, None, ctypes.c_float(0.0), p + 4096, 0, None) == 1
    assert L.wbmm_forward_fused(ctypes.byref(d14), p, p + 64, None, ctypes.c_float(float("nan")), p + 4096, 0, None) == 1
    assert L.wbmm_forward_fused(ctypes.byref(d14), p + 1, p + 64, None, ctypes.c_float(0.0), p + 4096, 0, None) == 5
    for ks in (0, 4, 29):                                                                            # even / too large
        assert L.wbmm_fold_dwconv(ctypes.byref(d14), p, p + 64, ks, None, p + 128, None) == 1, ks
    assert L.wbmm_fold_dwconv(ctypes.byref(d14), p, None, 3, None, p + 128, None) == 1
    assert L.wbmm_fold_dwconv(None, p, p + 64, 3, None, p + 128, None) == 1


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU behaviour")
def test_no_cpu_fallback(wb):
    """Without a device every compute entry point fails loudly."""
    x = torch.zeros(1, 1, 4, 4)
    T = torch.zeros(1, 9)
    with pytest.raises(wb.WbmmError) as e:
        wb.wbmm_forward_host(x, T, 2)
    assert e.value.status == 3
    with pytest.raises(ValueError):
        wb.wbmm_forward(x, T, 2)           # CPU tensors are rejected by the binding


def test_product_does_not_import_oracle():
    """The product path must not route through oracle/ (or any CPU implementation)."""
    pkg = os.path.join(ROOT, "paper_2607_02097_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU fallback", ""), os.path.join(dirpath, f)
    osrc = open(os.path.join(ROOT, "oracle", "wbmm_ref.py")).read() + open(os.path.join(ROOT, "oracle", "wbmm_ref.c")).read()
    assert "import paper_2607" not in osrc and "libwbmm.so" not in osrc and "wbmm.h" not in osrc
