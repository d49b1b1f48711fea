"""WBMM (Windowed Batch Matrix Multiplication, arxiv/paper_2607_02097) for NVIDIA B200.

The product is libwbmm.so (C ABI in include/wbmm.h, CUDA sources in csrc/); this package is the
thin Python binding with the same names.  Importing the package does not load the library;
the first call does, and raises if it has not been built (no CPU fallback).
"""
from .binding import (  # noqa: F401
    NCHW, NHWC, FLAG_ACCUMULATE_DT, FLAG_FORCE_SIMT, FLAG_NO_SCRATCH, FLAG_NO_FORK,
    PATH_NONE, PATH_SIMT, PATH_TC_TMA, PATH_TC_GATHER, PATH_TC_TRANSPOSED,
    WbmmDesc, WbmmError,
    wbmm_forward, wbmm_forward_static_scratch, STATUS_TOO_LARGE, wbmm_forward_rect, wbmm_backward_rect, wbmm_forward_win3d, wbmm_backward_win3d, wbmm_backward, wbmm_hier_forward, wbmm_hier_backward, wbmm_forward_matrix, wbmm_forward_int8, wbmm_forward_fp8, wbmm_fold_dwconv, wbmm_forward_fused, wbmm_materialize_weight,
    wbmm_forward_host, wbmm_backward_host, wbmm_release,
    wbmm_last_path, wbmm_path_string, wbmm_status_string, wbmm_last_error_string,
    wbmm_launch_count, wbmm_version,
)
