"""ctypes wrapper around oracle/wbmm_ref.c -- the CPU ORACLE.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It never imports the product package and shares no
code with it.  All arrays are float64 numpy arrays (callers round to the case
dtype first, then widen); see the header of wbmm_ref.c for citations and readings.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wbmm_ref.c")
# WBMM_ORACLE_SANITIZE=1: a second build with AddressSanitizer + UBSan (run the CPU pins under it with
# LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0; tests/README in DESIGN.md section 4)
_SANITIZE = os.environ.get("WBMM_ORACLE_SANITIZE") == "1"
_LIB = os.path.join(_HERE, "libwbmm_ref_asan.so" if _SANITIZE else "libwbmm_ref.so")

NCHW, NHWC = 0, 1

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no fast-math, OpenMP).  Returns the .so path."""
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if force or stale:
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-o", _LIB, _SRC, "-lm"]
        if _SANITIZE:
            cmd[1:2] = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build())
    dp = ctypes.POINTER(ctypes.c_double)
    ip = ctypes.POINTER(ctypes.c_int64)
    i = ctypes.c_int
    lib.wbmm_ref_rel_index.restype = ctypes.c_int64
    lib.wbmm_ref_rel_index.argtypes = [i, i, i]
    lib.wbmm_ref_index_matrix.restype = None
    lib.wbmm_ref_index_matrix.argtypes = [i, ip]
    lib.wbmm_ref_weight_matrix.restype = None
    lib.wbmm_ref_weight_matrix.argtypes = [i, i, dp, dp]
    for name in ("wbmm_ref_forward_matrix", "wbmm_ref_forward_direct"):
        f = getattr(lib, name)
        f.restype = i
        f.argtypes = [i] * 8 + [dp, dp, dp]
    lib.wbmm_ref_forward_rect.restype = i
    lib.wbmm_ref_forward_rect.argtypes = [i] * 9 + [dp, dp, dp]
    lib.wbmm_ref_backward_rect.restype = i
    lib.wbmm_ref_backward_rect.argtypes = [i] * 9 + [dp, dp, dp, dp, dp]
    lib.wbmm_ref_backward.restype = i
    lib.wbmm_ref_backward.argtypes = [i] * 8 + [dp, dp, dp, dp, dp]
    lib.wbmm_ref_forward_3d.argtypes = [i] * 12 + [dp, dp, dp]
    lib.wbmm_ref_forward_3d.restype = i
    lib.wbmm_ref_backward_3d.argtypes = [i] * 12 + [dp, dp, dp, dp, dp]
    lib.wbmm_ref_backward_3d.restype = i
    lib.wbmm_ref_forward_int8.argtypes = [i] * 8 + [ctypes.c_void_p] * 5
    lib.wbmm_ref_forward_int8.restype = i
    lib.wbmm_ref_hier_forward_train.restype = i
    lib.wbmm_ref_hier_forward_train.argtypes = [i] * 9 + [dp, dp, dp, dp]
    lib.wbmm_ref_hier_forward_fused.restype = i
    lib.wbmm_ref_hier_forward_fused.argtypes = [i] * 9 + [dp, dp, dp, dp, dp]
    lib.wbmm_ref_hier_backward_tables.restype = i
    lib.wbmm_ref_hier_backward_tables.argtypes = [i] * 8 + [dp, dp, dp, dp]
    lib.wbmm_ref_num_threads.restype = i
    lib.wbmm_ref_set_threads.argtypes = [i]
    _lib = lib
    return lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def num_threads() -> int:
    return int(_load().wbmm_ref_num_threads())


def set_threads(n: int) -> None:
    _load().wbmm_ref_set_threads(int(n))


def rel_index(w: int, i: int, j: int) -> int:
    """Eq. 7."""
    return int(_load().wbmm_ref_rel_index(w, i, j))


def index_matrix(w: int) -> np.ndarray:
    n = w * w
    out = np.empty((n, n), dtype=np.int64)
    _load().wbmm_ref_index_matrix(w, out.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)))
    return out


def weight_matrix(T: np.ndarray, w: int) -> np.ndarray:
    """Eq. 8: M[c] = T[c, I]."""
    T, tp = _d(T)
    C = T.shape[0]
    assert T.shape[1] == (2 * w - 1) ** 2
    n = w * w
    M = np.empty((C, n, n), dtype=np.float64)
    _load().wbmm_ref_weight_matrix(C, w, tp, M.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    return M


def _dims(x: np.ndarray, layout: int):
    if layout == NCHW:
        B, C, H, W = x.shape
    else:
        B, H, W, C = x.shape
    return B, C, H, W


def forward(x, T, w, shift=(0, 0), layout=NCHW, form="direct") -> np.ndarray:
    """y = WBMM(x; T, w).  form = "direct" | "matrix" (two independent evaluations)."""
    x, xp = _d(x)
    T, tp = _d(T)
    B, C, H, W = _dims(x, layout)
    assert T.shape == (C, (2 * w - 1) ** 2), (T.shape, C, w)
    y = np.zeros_like(x)
    fn = {"direct": _load().wbmm_ref_forward_direct, "matrix": _load().wbmm_ref_forward_matrix}[form]
    rc = fn(B, C, H, W, w, int(shift[0]), int(shift[1]), layout, xp, tp,
            y.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    if rc != 0:
        raise ValueError(f"oracle rejected arguments (rc={rc})")
    return y


def backward(x, T, dy, w, shift=(0, 0), layout=NCHW, need_dx=True, need_dT=True):
    """Returns (dx, dT) in float64; either is None when not requested."""
    x, xp = _d(x)
    T, tp = _d(T)
    dy, gp = _d(dy)
    assert dy.shape == x.shape
    B, C, H, W = _dims(x, layout)
    assert T.shape == (C, (2 * w - 1) ** 2)
    null = ctypes.POINTER(ctypes.c_double)()
    dx = np.zeros_like(x) if need_dx else None
    dT = np.zeros_like(T) if need_dT else None
    rc = _load().wbmm_ref_backward(
        B, C, H, W, w, int(shift[0]), int(shift[1]), layout, xp, tp, gp,
        dx.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if need_dx else null,
        dT.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if need_dT else null)
    if rc != 0:
        raise ValueError(f"oracle rejected arguments (rc={rc})")
    return dx, dT


def forward_rect(x, T, wh, ww, shift=(0, 0), layout=NCHW) -> np.ndarray:
    """Rectangular windows w_h x w_w (Eq. 4-7): y = WBMM(x; T), T [C,(2w_h-1)(2w_w-1)]."""
    x, xp = _d(x)
    T, tp = _d(T)
    B, C, H, W = _dims(x, layout)
    assert T.shape == (C, (2 * wh - 1) * (2 * ww - 1)), (T.shape, C, wh, ww)
    y = np.zeros_like(x)
    rc = _load().wbmm_ref_forward_rect(B, C, H, W, wh, ww, int(shift[0]), int(shift[1]), layout, xp, tp,
                                       y.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    if rc != 0:
        raise ValueError(f"oracle rejected arguments (rc={rc})")
    return y


def forward_int8(x, T, w, shift=(0, 0), layout=NCHW, scale=None) -> np.ndarray:
    """INT8 forward (NEXT-4): x, T int8, exact integer sums.  scale None: the int32 sums; scale [C]
    float32: int8 values sat_s8(rne(fp32(sum) * scale[c])) (reading A21)."""
    x = np.ascontiguousarray(x, dtype=np.int8)
    T = np.ascontiguousarray(T, dtype=np.int8)
    B, C, H, W = _dims(x, layout)
    assert T.shape == (C, (2 * w - 1) ** 2), (T.shape, C, w)
    if scale is None:
        y = np.zeros(x.shape, dtype=np.int32)
        rc = _load().wbmm_ref_forward_int8(B, C, H, W, w, int(shift[0]), int(shift[1]), layout, x.ctypes.data,
                                           T.ctypes.data, None, y.ctypes.data, None)
    else:
        scale = np.ascontiguousarray(scale, dtype=np.float32)
        assert scale.shape == (C,) and np.isfinite(scale).all()
        y = np.zeros(x.shape, dtype=np.int8)
        rc = _load().wbmm_ref_forward_int8(B, C, H, W, w, int(shift[0]), int(shift[1]), layout, x.ctypes.data,
                                           T.ctypes.data, scale.ctypes.data, None, y.ctypes.data)
    if rc != 0:
        raise ValueError(f"oracle rejected arguments (rc={rc})")
    return y


def _dims3(x, layout):
    if x.ndim != 5:
        raise ValueError("volume must be 5-D")
    if layout == NCHW:
        B, C, D, H, W = x.shape
    else:
        B, D, H, W, C = x.shape
    return B, C, D, H, W


def forward_3d(x, T, win, shift=(0, 0, 0), layout=NCHW) -> np.ndarray:
    """3-D windows win = (w_d, w_h, w_w) on [B,C,D,H,W] (layout 0) / [B,D,H,W,C] (layout 1): DESIGN.md reading A23."""
    x, xp = _d(x)
    T, tp = _d(T)
    B, C, D, H, W = _dims3(x, layout)
    wd, wh, ww = win
    assert T.shape == (C, (2 * wd - 1) * (2 * wh - 1) * (2 * ww - 1)), (T.shape, C, win)
    y = np.zeros_like(x)
    rc = _load().wbmm_ref_forward_3d(B, C, D, H, W, wd, wh, ww, int(shift[0]), int(shift[1]), int(shift[2]), layout, xp, tp,
                                     y.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    if rc != 0:
        raise ValueError(f"oracle rejected arguments (rc={rc})")
    return y


def backward_3d(x, T, dy, win, shift=(0, 0, 0), layout=NCHW, need_dx=True, need_dT=True):
    """(dx, dT) of forward_3d in float64; either is None when not requested."""
    x, xp = _d(x)
    T, tp = _d(T)
    dy, gp = _d(dy)
    assert dy.shape == x.shape
    B, C, D, H, W = _dims3(x, layout)
    wd, wh, ww = win
    assert T.shape == (C, (2 * wd - 1) * (2 * wh - 1) * (2 * ww - 1))
    null = ctypes.POINTER(ctypes.c_double)()
    dx = np.zeros_like(x) if need_dx else None
    dT = np.zeros_like(T) if need_dT else None
    rc = _load().wbmm_ref_backward_3d(
        B, C, D, H, W, wd, wh, ww, int(shift[0]), int(shift[1]), int(shift[2]), layout, xp, tp, gp,
        dx.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if need_dx else null,
        dT.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if need_dT else null)
    if rc != 0:
        raise ValueError(f"oracle rejected arguments (rc={rc})")
    return dx, dT


def e4m3_decode(codes) -> np.ndarray:
    """FP8 E4M3 ("fn" flavour: no infinities, 0x7f / 0xff are NaN; bias 7) byte codes -> float64, from the format's
    definition: sign (1) | exponent (4) | mantissa (3); exponent 0: subnormal m/8 * 2^-6; else (1 + m/8) * 2^(e-7)."""
    c = np.asarray(codes).astype(np.uint8).astype(np.int64)
    sign = np.where(c & 0x80, -1.0, 1.0)
    e = (c >> 3) & 0xF
    m = (c & 0x7).astype(np.float64)
    val = np.where(e == 0, m / 8.0 * 2.0 ** -6, (1.0 + m / 8.0) * np.exp2((e - 7).astype(np.float64)))
    val = np.where((e == 15) & ((c & 7) == 7), np.nan, val)
    return sign * val


def forward_fp8(x_codes, T_codes, w, shift=(0, 0), layout=NCHW, scale=None) -> np.ndarray:
    """FP8 (E4M3) forward, NEXT-4: the operator of `forward` on the decoded values, in float64 (every product of two
    E4M3 numbers and every sum of w*w of them is exact in float64), times scale[c] when given.  What the kernel stores
    (float32 sums, or E4M3 codes of sum * scale) is compared against THIS real number: DESIGN.md reading A22."""
    x = e4m3_decode(x_codes)
    T = e4m3_decode(T_codes)
    y = forward(x, T, w, shift, layout, form="direct")
    if scale is not None:
        sc = np.asarray(scale, dtype=np.float64)
        y = y * (sc[None, :, None, None] if layout == NCHW else sc[None, None, None, :])
    return y


def backward_rect(x, T, dy, wh, ww, shift=(0, 0), layout=NCHW, need_dx=True, need_dT=True):
    """(dx, dT) of forward_rect in float64; either is None when not requested."""
    x, xp = _d(x)
    T, tp = _d(T)
    dy, gp = _d(dy)
    assert dy.shape == x.shape
    B, C, H, W = _dims(x, layout)
    assert T.shape == (C, (2 * wh - 1) * (2 * ww - 1))
    null = ctypes.POINTER(ctypes.c_double)()
    dx = np.zeros_like(x) if need_dx else None
    dT = np.zeros_like(T) if need_dT else None
    rc = _load().wbmm_ref_backward_rect(
        B, C, H, W, wh, ww, int(shift[0]), int(shift[1]), layout, xp, tp, gp,
        dx.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if need_dx else null,
        dT.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if need_dT else null)
    if rc != 0:
        raise ValueError(f"oracle rejected arguments (rc={rc})")
    return dx, dT


def hier_forward(x, Tg, Tl, w, shift=(0, 0), layout=NCHW, form="train", transpose=False, return_matrix=False):
    """Hierarchical window reparameterisation: global w x w windows with
    table Tg[C,(2w-1)^2] plus their 2 x 2 local sub-windows with table Tl[C,(w-1)^2], identity
    shortcuts included.  form = "train" (Algorithm 2: the two scales evaluated separately) or
    "fused" (Algorithm 3: one fused matrix per channel).  transpose=True applies the transposed
    operator (dX)."""
    x, xp = _d(x)
    Tg, gp = _d(Tg)
    Tl, lp = _d(Tl)
    B, C, H, W = _dims(x, layout)
    assert w % 2 == 0 and Tg.shape == (C, (2 * w - 1) ** 2) and Tl.shape == (C, (w - 1) ** 2)
    y = np.zeros_like(x)
    yp = y.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
    args = (B, C, H, W, w, int(shift[0]), int(shift[1]), layout, 1 if transpose else 0, xp, gp, lp, yp)
    if form == "train":
        rc = _load().wbmm_ref_hier_forward_train(*args)
        M = None
    else:
        M = np.zeros((C, w * w, w * w)) if return_matrix else None
        mp = M.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if return_matrix else ctypes.POINTER(ctypes.c_double)()
        rc = _load().wbmm_ref_hier_forward_fused(*args, mp)
    if rc != 0:
        raise ValueError(f"oracle rejected arguments (rc={rc})")
    return (y, M) if return_matrix else y


def hier_backward(x, Tg, Tl, dy, w, shift=(0, 0), layout=NCHW):
    """Gradients of the hierarchical operator (the backward of Algorithm 2):
    returns (dx, dTg, dTl).  dx is the transposed operator applied to dy (training form);
    dTg[C,(2w-1)^2], dTl[C,(w-1)^2] are the table gradients by their definition."""
    dx = hier_forward(dy, Tg, Tl, w, shift, layout, form="train", transpose=True)
    x, xp = _d(x)
    dy, gp = _d(dy)
    B, C, H, W = _dims(x, layout)
    assert w % 2 == 0 and x.shape == dy.shape
    dTg = np.zeros((C, (2 * w - 1) ** 2))
    dTl = np.zeros((C, (w - 1) ** 2))
    rc = _load().wbmm_ref_hier_backward_tables(
        B, C, H, W, w, int(shift[0]), int(shift[1]), layout, xp, gp,
        dTg.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), dTl.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    if rc != 0:
        raise ValueError(f"oracle rejected arguments (rc={rc})")
    return dx, dTg, dTl


def apply_matrix(x, M, w, shift=(0, 0), layout=NCHW, transpose=False, bias=None) -> np.ndarray:
    """Cached-M mode, WBMM-C: Algorithm 1 with a GIVEN per-channel
    matrix M[C, N, N] (y_win = M_c x_win, orientation A1) instead of M = R[:, I]; optional per-channel bias
    (Eq. 1's beta_c).  Written out in the paper's order with plain numpy: pad (l.2), roll
    (A6), window partition (l.3-4), one batched matrix product (l.15), inverse reshape (l.17), un-roll, crop."""
    x = np.asarray(x, dtype=np.float64)
    M = np.asarray(M, dtype=np.float64)
    xc = x if layout == NCHW else np.transpose(x, (0, 3, 1, 2))
    B, C, H, W = xc.shape
    N = w * w
    assert M.shape == (C, N, N)
    Hp, Wp = -(-H // w) * w, -(-W // w) * w
    xp = np.zeros((B, C, Hp, Wp))
    xp[:, :, :H, :W] = xc                                              # zero padding, bottom / right (A4)
    xh = np.roll(xp, (-int(shift[0]), -int(shift[1])), axis=(2, 3))    # x^[h, v] = x~[(h + s) mod H', ...] (A6)
    nh, nw = Hp // w, Wp // w
    win = xh.reshape(B, C, nh, w, nw, w).transpose(0, 1, 2, 4, 3, 5).reshape(B, C, nh * nw, N)
    Mc = np.transpose(M, (0, 2, 1)) if transpose else M
    yw = np.einsum("cij,bcnj->bcni", Mc, win)                          # l.15: the batched product
    yh = yw.reshape(B, C, nh, nw, w, w).transpose(0, 1, 2, 4, 3, 5).reshape(B, C, Hp, Wp)
    y = np.roll(yh, (int(shift[0]), int(shift[1])), axis=(2, 3))[:, :, :H, :W]
    if bias is not None:
        y = y + np.asarray(bias, dtype=np.float64).reshape(1, C, 1, 1)
    return np.ascontiguousarray(y if layout == NCHW else np.transpose(y, (0, 2, 3, 1)))


def fold_dwconv(T, K, w, scale=None) -> np.ndarray:
    """Multi-kernel fusion (section 3.7): on a map that is ONE w x w window, a zero-padded
    depthwise conv (Eq. 1: Y[h,v] = sum_{i,j} K[i+k, j+k] X[h+i, v+j]) is the WBMM operator whose table is
    zero except T[(w-1-i)(2w-1) + (w-1-j)] = K[i+k, j+k] -- output p = (h,v) reads input q = (h+i, v+j), and
    rel(p, q) = (r_p - r_q + w-1)(2w-1) + (c_p - c_q + w-1) (Eq. 6-7).  Returns T + scale_c * (that table);
    the scale is BatchNorm's gamma / sigma (its shift becomes the bias of apply_matrix)."""
    T = np.array(T, dtype=np.float64)
    K = np.asarray(K, dtype=np.float64)
    C, kk, _ = K.shape
    k = kk // 2
    assert kk % 2 == 1 and k <= w - 1 and T.shape == (C, (2 * w - 1) ** 2)
    s = np.ones(C) if scale is None else np.asarray(scale, dtype=np.float64)
    tw = 2 * w - 1
    for i in range(-k, k + 1):
        for j in range(-k, k + 1):
            T[:, (w - 1 - i) * tw + (w - 1 - j)] += s * K[:, i + k, j + k]
    return T
