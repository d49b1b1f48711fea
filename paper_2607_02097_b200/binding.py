"""Thin ctypes binding over libwbmm.so (include/wbmm.h).  Argument marshalling only: every step
of the WBMM path runs in the CUDA kernels behind the C ABI.  torch is used for device memory and
the current stream.  There is no CPU fallback: a missing library or device raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libwbmm.so")

NCHW, NHWC = 0, 1
DTYPE_F32, DTYPE_BF16, DTYPE_F16 = 0, 1, 2
PATH_NONE, PATH_SIMT, PATH_TC_TMA, PATH_TC_GATHER, PATH_TC_TRANSPOSED = 0, 1, 2, 3, 4
FLAG_ACCUMULATE_DT, FLAG_FORCE_SIMT, FLAG_NO_SCRATCH, FLAG_NO_FORK = 1, 2, 4, 8
STATUS_OK = 0
STATUS_TOO_LARGE = 6

_DTYPES = {torch.float32: DTYPE_F32, torch.bfloat16: DTYPE_BF16, torch.float16: DTYPE_F16}

# every symbol include/wbmm.h declares
EXPORTS = (
    "wbmm_forward", "wbmm_forward_static_scratch", "wbmm_forward_rect", "wbmm_backward_rect", "wbmm_forward_win3d", "wbmm_backward_win3d", "wbmm_backward", "wbmm_hier_forward", "wbmm_hier_backward", "wbmm_forward_matrix", "wbmm_forward_int8", "wbmm_forward_fp8", "wbmm_fold_dwconv", "wbmm_forward_fused", "wbmm_materialize_weight", "wbmm_forward_host",
    "wbmm_backward_host", "wbmm_release", "wbmm_last_path", "wbmm_launch_count",
    "wbmm_status_string", "wbmm_path_string", "wbmm_last_error_string", "wbmm_version",
)


class WbmmDesc(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in
                ("B", "C", "H", "W", "w", "shift_h", "shift_w", "dtype", "layout")] + [("flags", ctypes.c_uint32)]


class WbmmError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(msg)
        self.status = status


_lib = None


def lib() -> ctypes.CDLL:
    """Loads libwbmm.so (built in-tree by paper_2607_02097_b200.build).  Raises if it is absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2607_02097_b200.build` "
                          "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, dp, i = ctypes.c_void_p, ctypes.POINTER(WbmmDesc), ctypes.c_int
    L.wbmm_forward.argtypes = [dp, vp, vp, vp, vp]
    L.wbmm_forward_static_scratch.argtypes = [dp, vp, vp, vp, vp]
    L.wbmm_forward_static_scratch.restype = i
    L.wbmm_forward_rect.argtypes = [dp, ctypes.c_int32, vp, vp, vp, vp]
    L.wbmm_forward_rect.restype = i
    L.wbmm_backward_rect.argtypes = [dp, ctypes.c_int32, vp, vp, vp, vp, vp, vp]
    L.wbmm_backward_rect.restype = i
    i32 = ctypes.c_int32
    L.wbmm_forward_win3d.argtypes = [dp, i32, i32, i32, i32, vp, vp, vp, vp]
    L.wbmm_forward_win3d.restype = i
    L.wbmm_backward_win3d.argtypes = [dp, i32, i32, i32, i32, vp, vp, vp, vp, vp, vp]
    L.wbmm_backward_win3d.restype = i
    L.wbmm_backward.argtypes = [dp, vp, vp, vp, vp, vp, vp]
    L.wbmm_hier_forward.argtypes = [dp, vp, vp, vp, vp, i, vp]
    L.wbmm_hier_forward.restype = i
    L.wbmm_hier_backward.argtypes = [dp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.wbmm_hier_backward.restype = i
    L.wbmm_materialize_weight.argtypes = [dp, vp, vp, vp]
    L.wbmm_forward_matrix.argtypes = [dp, vp, vp, vp, vp, i, vp]
    L.wbmm_forward_matrix.restype = i
    L.wbmm_forward_int8.argtypes = [dp, vp, vp, vp, vp, vp]
    L.wbmm_forward_int8.restype = i
    L.wbmm_forward_fp8.argtypes = [dp, vp, vp, vp, vp, vp]
    L.wbmm_forward_fp8.restype = i
    L.wbmm_fold_dwconv.argtypes = [dp, vp, vp, i, vp, vp, vp]
    L.wbmm_fold_dwconv.restype = i
    L.wbmm_forward_fused.argtypes = [dp, vp, vp, vp, ctypes.c_float, vp, i, vp]
    L.wbmm_forward_fused.restype = i
    L.wbmm_forward_host.argtypes = [dp, vp, vp, vp]
    L.wbmm_backward_host.argtypes = [dp, vp, vp, vp, vp, vp]
    for n in ("wbmm_forward", "wbmm_backward", "wbmm_materialize_weight", "wbmm_forward_host",
              "wbmm_backward_host", "wbmm_last_path", "wbmm_version"):
        getattr(L, n).restype = i
    L.wbmm_release.restype = None
    L.wbmm_launch_count.restype = ctypes.c_uint64
    for n in ("wbmm_status_string", "wbmm_path_string", "wbmm_last_error_string"):
        getattr(L, n).restype = ctypes.c_char_p
    L.wbmm_status_string.argtypes = [i]
    L.wbmm_path_string.argtypes = [i]
    _lib = L
    return L


def _check(st: int) -> None:
    if st != STATUS_OK:
        L = lib()
        msg = L.wbmm_status_string(st).decode()
        err = L.wbmm_last_error_string().decode()
        raise WbmmError(st, f"libwbmm: {msg}" + (f" ({err})" if st in (4, STATUS_TOO_LARGE) and err else ""))


def _dims(t: torch.Tensor, layout: int):
    if t.dim() != 4:
        raise ValueError("activation must be 4-D")
    if layout == NCHW:
        B, C, H, W = t.shape
    else:
        B, H, W, C = t.shape
    return B, C, H, W


_desc_cache = {}


def make_desc(x: torch.Tensor, w: int, shift=(0, 0), layout: int = NCHW, flags: int = 0) -> WbmmDesc:
    """The problem descriptor of a call (read-only on the C side, so descriptors are cached by their fields:
    an eager call costs the host ~7 us, of which building a ctypes structure was one)."""
    key = (x.shape, x.dtype, w, shift[0], shift[1], layout, flags)
    d = _desc_cache.get(key)
    if d is None:
        B, C, H, W = _dims(x, layout)
        if x.dtype not in _DTYPES:
            raise TypeError(f"unsupported dtype {x.dtype}")
        d = WbmmDesc(B, C, H, W, int(w), int(shift[0]), int(shift[1]), _DTYPES[x.dtype], int(layout), int(flags))
        if len(_desc_cache) < 4096:
            _desc_cache[key] = d
    return d


_raw_stream = getattr(torch._C, "_cuda_getCurrentRawStream", None)


def _stream(t: torch.Tensor) -> int:
    """cudaStream_t of torch's current stream on the tensor's device."""
    if _raw_stream is not None:
        return _raw_stream(t.device.index)
    return torch.cuda.current_stream(t.device).cuda_stream


def _dev(t: Optional[torch.Tensor], name: str) -> Optional[int]:
    if t is None:
        return None
    if not t.is_cuda:
        raise ValueError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    return t.data_ptr()


def wbmm_forward(x: torch.Tensor, T: torch.Tensor, w: int, shift=(0, 0), layout: int = NCHW,
                 flags: int = 0, out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """y = WBMM(x; T, w) on the current CUDA stream (include/wbmm.h: wbmm_forward)."""
    d = make_desc(x, w, shift, layout, flags)
    if T.dtype != x.dtype or tuple(T.shape) != (d.C, (2 * w - 1) ** 2):
        raise ValueError("T must be [C,(2w-1)^2] in the dtype of x")
    y = torch.empty_like(x) if out is None else out
    px, pT, py = _dev(x, "x"), _dev(T, "T"), _dev(y, "y")
    if x.device.index == torch.cuda.current_device():      # the common case: no device switch
        _check(lib().wbmm_forward(ctypes.byref(d), px, pT, py, _stream(x)))
    else:
        with torch.cuda.device(x.device):
            _check(lib().wbmm_forward(ctypes.byref(d), px, pT, py, _stream(x)))
    return y


def wbmm_forward_static_scratch(x: torch.Tensor, T: torch.Tensor, w: int, shift=(0, 0),
                                out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """wbmm_forward for NHWC bf16/fp16 activations of at most 16 MiB with the temporaries in the library's static
    device array: the C call allocates nothing (include/wbmm.h: wbmm_forward_static_scratch; pass `out` to keep
    the binding from allocating the result).  Calls that overlap on the GPU race on the array."""
    d = make_desc(x, w, shift, NHWC, 0)
    if T.dtype != x.dtype or tuple(T.shape) != (d.C, (2 * w - 1) ** 2):
        raise ValueError("T must be [C,(2w-1)^2] in the dtype of x")
    y = torch.empty_like(x) if out is None else out
    px, pT, py = _dev(x, "x"), _dev(T, "T"), _dev(y, "y")
    with torch.cuda.device(x.device):
        _check(lib().wbmm_forward_static_scratch(ctypes.byref(d), px, pT, py, _stream(x)))
    return y


def wbmm_forward_rect(x: torch.Tensor, T: torch.Tensor, wh: int, ww: int, shift=(0, 0), layout: int = NCHW,
                      out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Rectangular windows w_h x w_w (include/wbmm.h: wbmm_forward_rect); T is [C, (2w_h-1)(2w_w-1)]."""
    d = make_desc(x, wh, shift, layout, 0)
    if T.dtype != x.dtype or tuple(T.shape) != (d.C, (2 * wh - 1) * (2 * ww - 1)):
        raise ValueError("T must be [C,(2w_h-1)(2w_w-1)] in the dtype of x")
    y = torch.empty_like(x) if out is None else out
    px, pT, py = _dev(x, "x"), _dev(T, "T"), _dev(y, "y")
    with torch.cuda.device(x.device):
        _check(lib().wbmm_forward_rect(ctypes.byref(d), int(ww), px, pT, py, _stream(x)))
    return y


def wbmm_backward_rect(x: Optional[torch.Tensor], T: Optional[torch.Tensor], dy: torch.Tensor, wh: int, ww: int,
                       shift=(0, 0), layout: int = NCHW, flags: int = 0, need_dx: bool = True, need_dT: bool = True,
                       dT: Optional[torch.Tensor] = None):
    """(dx, dT) of wbmm_forward_rect; dT is float32 [C, (2w_h-1)(2w_w-1)]."""
    d = make_desc(dy, wh, shift, layout, flags)
    dx = torch.empty_like(dy) if need_dx else None
    if need_dT and dT is None:
        dT = torch.empty((d.C, (2 * wh - 1) * (2 * ww - 1)), dtype=torch.float32, device=dy.device)
    if not need_dT:
        dT = None
    with torch.cuda.device(dy.device):
        _check(lib().wbmm_backward_rect(ctypes.byref(d), int(ww), _dev(x, "x"), _dev(T, "T"), _dev(dy, "dy"),
                                        _dev(dx, "dx"), _dev(dT, "dT"), _stream(dy)))
    return dx, dT


def _desc3d(t: torch.Tensor, win, shift, layout: int, flags: int):
    if t.dim() != 5:
        raise ValueError("volume must be 5-D: [B,C,D,H,W] (NCHW) or [B,D,H,W,C] (NHWC)")
    if layout == NCHW:
        B, C, D, H, W = t.shape
    else:
        B, D, H, W, C = t.shape
    if t.dtype not in _DTYPES:
        raise TypeError(f"unsupported dtype {t.dtype}")
    wd, wh, ww = (int(v) for v in win)
    d = WbmmDesc(B, C, H, W, wh, int(shift[1]), int(shift[2]), _DTYPES[t.dtype], int(layout), int(flags))
    return d, D, wd, ww, int(shift[0]), (C, (2 * wd - 1) * (2 * wh - 1) * (2 * ww - 1))


def wbmm_forward_win3d(x: torch.Tensor, T: torch.Tensor, win, shift=(0, 0, 0), layout: int = NCHW,
                       out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """3-D windows win = (w_d, w_h, w_w) on a volume (include/wbmm.h: wbmm_forward_win3d)."""
    d, D, wd, ww, sd, tshape = _desc3d(x, win, shift, layout, 0)
    if T.dtype != x.dtype or tuple(T.shape) != tshape:
        raise ValueError("T must be [C,(2w_d-1)(2w_h-1)(2w_w-1)] in the dtype of x")
    y = torch.empty_like(x) if out is None else out
    with torch.cuda.device(x.device):
        _check(lib().wbmm_forward_win3d(ctypes.byref(d), D, wd, ww, sd, _dev(x, "x"), _dev(T, "T"), _dev(y, "y"), _stream(x)))
    return y


def wbmm_backward_win3d(x: Optional[torch.Tensor], T: Optional[torch.Tensor], dy: torch.Tensor, win, shift=(0, 0, 0),
                        layout: int = NCHW, flags: int = 0, need_dx: bool = True, need_dT: bool = True,
                        dT: Optional[torch.Tensor] = None):
    """(dx, dT) of wbmm_forward_win3d; dT is float32 [C, (2w_d-1)(2w_h-1)(2w_w-1)]."""
    d, D, wd, ww, sd, tshape = _desc3d(dy, win, shift, layout, flags)
    dx = torch.empty_like(dy) if need_dx else None
    if need_dT and dT is None:
        dT = torch.empty(tshape, dtype=torch.float32, device=dy.device)
    if not need_dT:
        dT = None
    with torch.cuda.device(dy.device):
        _check(lib().wbmm_backward_win3d(ctypes.byref(d), D, wd, ww, sd, _dev(x, "x"), _dev(T, "T"), _dev(dy, "dy"),
                                         _dev(dx, "dx"), _dev(dT, "dT"), _stream(dy)))
    return dx, dT


def wbmm_hier_forward(x: torch.Tensor, Tg: torch.Tensor, Tl: torch.Tensor, w: int, shift=(0, 0),
                      layout: int = NCHW, transpose: bool = False, out: Optional[torch.Tensor] = None,
                      flags: int = 0) -> torch.Tensor:
    """Fused hierarchical operator y = (M_g + diag_blocks(M_l) + 2I) x per w x w window
    (include/wbmm.h: wbmm_hier_forward); transpose=True gives dX for dy passed as x."""
    d = make_desc(x, w, shift, layout, flags)
    if Tg.dtype != x.dtype or Tl.dtype != x.dtype or tuple(Tg.shape) != (d.C, (2 * w - 1) ** 2) \
            or tuple(Tl.shape) != (d.C, (w - 1) ** 2):
        raise ValueError("Tg must be [C,(2w-1)^2] and Tl [C,(w-1)^2] in the dtype of x")
    y = torch.empty_like(x) if out is None else out
    px, pg, pl, py = _dev(x, "x"), _dev(Tg, "Tg"), _dev(Tl, "Tl"), _dev(y, "y")
    with torch.cuda.device(x.device):
        _check(lib().wbmm_hier_forward(ctypes.byref(d), px, pg, pl, py, 1 if transpose else 0, _stream(x)))
    return y


def wbmm_hier_backward(x: Optional[torch.Tensor], Tg: Optional[torch.Tensor], Tl: Optional[torch.Tensor],
                       dy: torch.Tensor, w: int, shift=(0, 0), layout: int = NCHW, flags: int = 0,
                       need_dx: bool = True, need_dT: bool = True, dTg: Optional[torch.Tensor] = None,
                       dTl: Optional[torch.Tensor] = None):
    """(dx, dTg, dTl) of wbmm_hier_forward (include/wbmm.h: wbmm_hier_backward); the table gradients
    are float32 [C,(2w-1)^2] and [C,(w-1)^2] and come from one pass over (x, dy)."""
    d = make_desc(dy, w, shift, layout, flags)
    dx = torch.empty_like(dy) if need_dx else None
    if need_dT:
        if dTg is None:
            dTg = torch.empty((d.C, (2 * w - 1) ** 2), dtype=torch.float32, device=dy.device)
        if dTl is None:
            dTl = torch.empty((d.C, (w - 1) ** 2), dtype=torch.float32, device=dy.device)
    else:
        dTg = dTl = None
    with torch.cuda.device(dy.device):
        _check(lib().wbmm_hier_backward(ctypes.byref(d), _dev(x, "x") if need_dT else None,
                                        _dev(Tg, "Tg") if need_dx else None, _dev(Tl, "Tl") if need_dx else None,
                                        _dev(dy, "dy"), _dev(dx, "dx"), _dev(dTg, "dTg"), _dev(dTl, "dTl"), _stream(dy)))
    return dx, dTg, dTl


def wbmm_backward(x: Optional[torch.Tensor], T: Optional[torch.Tensor], dy: torch.Tensor, w: int,
                  shift=(0, 0), layout: int = NCHW, flags: int = 0, need_dx: bool = True,
                  need_dT: bool = True, dT: Optional[torch.Tensor] = None, dx: Optional[torch.Tensor] = None
                  ) -> Tuple[Optional[torch.Tensor], Optional[torch.Tensor]]:
    """(dx, dT) of wbmm_forward; dT is float32 [C,(2w-1)^2] (include/wbmm.h: wbmm_backward)."""
    d = make_desc(dy, w, shift, layout, flags)
    if need_dx and dx is None:
        dx = torch.empty_like(dy)
    if not need_dx:
        dx = None
    if need_dT and dT is None:
        dT = torch.empty((d.C, (2 * w - 1) ** 2), dtype=torch.float32, device=dy.device)
    if not need_dT:
        dT = None
    with torch.cuda.device(dy.device):
        _check(lib().wbmm_backward(ctypes.byref(d), _dev(x, "x") if need_dT else None,
                                   _dev(T, "T") if need_dx else None, _dev(dy, "dy"),
                                   _dev(dx, "dx"), _dev(dT, "dT"), _stream(dy)))
    return dx, dT


def wbmm_materialize_weight(T: torch.Tensor, w: int) -> torch.Tensor:
    """Eq. 8: W[c,i,j] = T[c, rel(i,j)] as a [C,N,N] tensor (bit-exact copy of table entries)."""
    C = T.shape[0]
    d = WbmmDesc(0, C, 1, 1, int(w), 0, 0, _DTYPES[T.dtype], NCHW, 0)
    W = torch.empty((C, w * w, w * w), dtype=T.dtype, device=T.device)
    with torch.cuda.device(T.device):
        _check(lib().wbmm_materialize_weight(ctypes.byref(d), _dev(T, "T"), _dev(W, "W"), _stream(T)))
    return W


def wbmm_forward_fused(x: torch.Tensor, T: torch.Tensor, w: int, shift=(0, 0), layout: int = NCHW,
                       bias: Optional[torch.Tensor] = None, identity: float = 0.0, transpose: bool = False,
                       out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """y = WBMM(x; T) + identity * x + bias_c in one kernel (include/wbmm.h: wbmm_forward_fused)."""
    d = make_desc(x, w, shift, layout, 0)
    if T.dtype != x.dtype or tuple(T.shape) != (d.C, (2 * w - 1) ** 2):
        raise ValueError("T must be [C,(2w-1)^2] in the dtype of x")
    if bias is not None and (bias.dtype != x.dtype or tuple(bias.shape) != (d.C,)):
        raise ValueError("bias must be [C] in the dtype of x")
    y = torch.empty_like(x) if out is None else out
    with torch.cuda.device(x.device):
        _check(lib().wbmm_forward_fused(ctypes.byref(d), _dev(x, "x"), _dev(T, "T"), _dev(bias, "bias"),
                                        ctypes.c_float(identity), _dev(y, "y"), 1 if transpose else 0, _stream(x)))
    return y


def wbmm_forward_matrix(x: torch.Tensor, M: torch.Tensor, w: int, shift=(0, 0), layout: int = NCHW,
                        bias: Optional[torch.Tensor] = None, transpose: bool = False,
                        out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Cached-M mode (WBMM-C): y_win = M_c x_win (+ bias_c) with M [C,N,N] given
    (include/wbmm.h: wbmm_forward_matrix)."""
    d = make_desc(x, w, shift, layout, 0)
    if M.dtype != x.dtype or tuple(M.shape) != (d.C, w * w, w * w):
        raise ValueError("M must be [C, w*w, w*w] in the dtype of x")
    if bias is not None and (bias.dtype != x.dtype or tuple(bias.shape) != (d.C,)):
        raise ValueError("bias must be [C] in the dtype of x")
    y = torch.empty_like(x) if out is None else out
    with torch.cuda.device(x.device):
        _check(lib().wbmm_forward_matrix(ctypes.byref(d), _dev(x, "x"), _dev(M, "M"), _dev(bias, "bias"),
                                         _dev(y, "y"), 1 if transpose else 0, _stream(x)))
    return y


def wbmm_forward_int8(x: torch.Tensor, T: torch.Tensor, w: int, shift=(0, 0), layout: int = NCHW,
                      scale: Optional[torch.Tensor] = None, out: Optional[torch.Tensor] = None, flags: int = 0) -> torch.Tensor:
    """INT8 forward with exact int32 sums; scale [C] float32 requantises to int8 (include/wbmm.h: wbmm_forward_int8)."""
    if x.dtype != torch.int8 or T.dtype != torch.int8:
        raise TypeError("x and T must be int8")
    B, C, H, W = _dims(x, layout)
    if tuple(T.shape) != (C, (2 * w - 1) ** 2):
        raise ValueError("T must be [C, (2w-1)^2]")
    if scale is not None and (scale.dtype != torch.float32 or tuple(scale.shape) != (C,)):
        raise ValueError("scale must be float32 [C]")
    d = WbmmDesc(B, C, H, W, int(w), int(shift[0]), int(shift[1]), DTYPE_F32, int(layout), int(flags))
    odt = torch.int32 if scale is None else torch.int8
    y = torch.empty(x.shape, dtype=odt, device=x.device) if out is None else out
    if y.dtype != odt or y.shape != x.shape:
        raise ValueError(f"out must be {odt} with the shape of x")
    with torch.cuda.device(x.device):
        _check(lib().wbmm_forward_int8(ctypes.byref(d), _dev(x, "x"), _dev(T, "T"), _dev(scale, "scale"), _dev(y, "y"),
                                       _stream(x)))
    return y


def wbmm_forward_fp8(x: torch.Tensor, T: torch.Tensor, w: int, shift=(0, 0), layout: int = NCHW,
                     scale: Optional[torch.Tensor] = None, out: Optional[torch.Tensor] = None, flags: int = 0) -> torch.Tensor:
    """FP8 (E4M3) forward with float32 sums; scale [C] float32 gives E4M3 output (include/wbmm.h: wbmm_forward_fp8)."""
    f8 = torch.float8_e4m3fn
    if x.dtype != f8 or T.dtype != f8:
        raise TypeError("x and T must be torch.float8_e4m3fn")
    B, C, H, W = _dims(x, layout)
    if tuple(T.shape) != (C, (2 * w - 1) ** 2):
        raise ValueError("T must be [C, (2w-1)^2]")
    if scale is not None and (scale.dtype != torch.float32 or tuple(scale.shape) != (C,)):
        raise ValueError("scale must be float32 [C]")
    d = WbmmDesc(B, C, H, W, int(w), int(shift[0]), int(shift[1]), DTYPE_F32, int(layout), int(flags))
    odt = torch.float32 if scale is None else f8
    y = torch.empty(x.shape, dtype=odt, device=x.device) if out is None else out
    if y.dtype != odt or y.shape != x.shape:
        raise ValueError(f"out must be {odt} with the shape of x")
    with torch.cuda.device(x.device):
        _check(lib().wbmm_forward_fp8(ctypes.byref(d), _dev(x, "x"), _dev(T, "T"), _dev(scale, "scale"), _dev(y, "y"),
                                      _stream(x)))
    return y


def wbmm_fold_dwconv(T: torch.Tensor, K: torch.Tensor, w: int, scale: Optional[torch.Tensor] = None,
                     out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """T + scale_c * (table of the zero-padded depthwise conv K [C,k,k]) -- section 3.7's fold for
    one-window maps (include/wbmm.h: wbmm_fold_dwconv)."""
    C = T.shape[0]
    if K.dtype != T.dtype or K.dim() != 3 or K.shape[0] != C or K.shape[1] != K.shape[2]:
        raise ValueError("K must be [C, k, k] in the dtype of T")
    if scale is not None and (scale.dtype != torch.float32 or tuple(scale.shape) != (C,)):
        raise ValueError("scale must be float32 [C]")
    d = WbmmDesc(0, C, 1, 1, int(w), 0, 0, _DTYPES[T.dtype], NCHW, 0)
    Tout = torch.empty_like(T) if out is None else out
    with torch.cuda.device(T.device):
        _check(lib().wbmm_fold_dwconv(ctypes.byref(d), _dev(T, "T"), _dev(K, "K"), int(K.shape[1]),
                                      _dev(scale, "scale"), _dev(Tout, "Tout"), _stream(T)))
    return Tout


def _host(t: Optional[torch.Tensor], name: str) -> Optional[int]:
    if t is None:
        return None
    if t.is_cuda or not t.is_contiguous():
        raise ValueError(f"{name} must be a contiguous host tensor")
    return t.data_ptr()


def wbmm_forward_host(x: torch.Tensor, T: torch.Tensor, w: int, shift=(0, 0), layout: int = NCHW,
                      flags: int = 0, out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Host-buffer forward: H2D copies, kernels and the D2H copy all happen inside the C call."""
    d = make_desc(x, w, shift, layout, flags)
    y = torch.empty_like(x) if out is None else out
    _check(lib().wbmm_forward_host(ctypes.byref(d), _host(x, "x"), _host(T, "T"), _host(y, "y")))
    return y


def wbmm_backward_host(x, T, dy, w, shift=(0, 0), layout: int = NCHW, flags: int = 0,
                       need_dx: bool = True, need_dT: bool = True, dx=None, dT=None):
    d = make_desc(dy, w, shift, layout, flags)
    if need_dx and dx is None:
        dx = torch.empty_like(dy)
    if need_dT and dT is None:
        dT = torch.empty((d.C, (2 * w - 1) ** 2), dtype=torch.float32)
    _check(lib().wbmm_backward_host(ctypes.byref(d), _host(x, "x") if need_dT else None,
                                    _host(T, "T") if need_dx else None, _host(dy, "dy"),
                                    _host(dx, "dx") if need_dx else None, _host(dT, "dT") if need_dT else None))
    return (dx if need_dx else None), (dT if need_dT else None)


def wbmm_release() -> None:
    lib().wbmm_release()


def wbmm_last_path() -> int:
    return int(lib().wbmm_last_path())


def wbmm_path_string(path: int) -> str:
    return lib().wbmm_path_string(int(path)).decode()


def wbmm_status_string(status: int) -> str:
    return lib().wbmm_status_string(int(status)).decode()


def wbmm_last_error_string() -> str:
    return lib().wbmm_last_error_string().decode()


def wbmm_launch_count() -> int:
    return int(lib().wbmm_launch_count())


def wbmm_version() -> int:
    return int(lib().wbmm_version())
