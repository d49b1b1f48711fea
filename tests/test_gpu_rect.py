"""Rectangular windows w_h x w_w on the GPU (wbmm_forward_rect / wbmm_backward_rect, csrc/wbmm_rect.cu) against the
oracle's forward_rect / backward_rect (section 3.1, Eq. 4-7); w_h = 1: the 1-D windows of PAPER.md:909."""
import numpy as np
import pytest
import torch

import synth_inputs as si
from parity import TOL, max_err_over_tol, widen

pytestmark = pytest.mark.gpu

NCHW, NHWC = si.NCHW, si.NHWC
TD = {"f32": torch.float32, "bf16": torch.bfloat16, "f16": torch.float16}


@pytest.fixture(scope="module")
def wb():
    import paper_2607_02097_b200 as wb
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    wb.wbmm_version()
    return wb


def _data(B, C, H, W, wh, ww, dtype, layout, seed):
    g = torch.Generator().manual_seed(seed)
    shape = (B, C, H, W) if layout == NCHW else (B, H, W, C)
    x = torch.randn(shape, generator=g).to(TD[dtype]).cuda()
    dy = torch.randn(shape, generator=g).to(TD[dtype]).cuda()
    T = (torch.randn((C, (2 * wh - 1) * (2 * ww - 1)), generator=g) * 0.05).to(TD[dtype]).cuda()
    return x, dy, T


RECT_CASES = [
    # B, C, H, W, wh, ww, shift, dtype, layout
    (3, 5, 28, 56, 7, 14, (0, 0), "bf16", NCHW),
    (2, 6, 30, 50, 14, 7, (5, 3), "bf16", NCHW),          # ragged both ways, shift up to w_h - 1 / w_w - 1
    (2, 8, 21, 40, 7, 14, (6, 13), "f16", NHWC),
    (4, 3, 9, 10, 2, 3, (1, 2), "f32", NCHW),
    (2, 4, 5, 64, 1, 16, (0, 9), "f32", NCHW),            # 1-D windows along W
    (2, 4, 48, 6, 12, 1, (7, 0), "bf16", NHWC),           # 1-D windows along H
    (1, 2, 32, 32, 32, 32 // 4, (0, 0), "f32", NCHW),     # N = 256, 63 x 15 bins
    (3, 70, 16, 24, 4, 8, (2, 5), "f32", NHWC),
]


@pytest.mark.parametrize("B,C,H,W,wh,ww,shift,dtype,layout", RECT_CASES)
def test_rect_forward_backward_match_the_oracle(wb, oracle, B, C, H, W, wh, ww, shift, dtype, layout):
    x, dy, T = _data(B, C, H, W, wh, ww, dtype, layout, seed=700 + wh * 31 + ww)
    y = wb.wbmm_forward_rect(x, T, wh, ww, shift, layout)
    assert wb.wbmm_last_path() == wb.PATH_SIMT
    dx, dT = wb.wbmm_backward_rect(x, T, dy, wh, ww, shift, layout)
    torch.cuda.synchronize()
    ry = oracle.forward_rect(widen(x), widen(T), wh, ww, shift, layout)
    rdx, rdT = oracle.backward_rect(widen(x), widen(T), widen(dy), wh, ww, shift, layout)
    tol = TOL[dtype]
    assert max_err_over_tol(y, ry, tol) <= 1.0 and max_err_over_tol(dx, rdx, tol) <= 1.0
    nwin = B * (-(-H // wh)) * (-(-W // ww))
    scale = float(np.sqrt(nwin * wh * ww))
    g = widen(dT)
    assert float(np.max(np.abs(g - rdT) / (tol * (scale + np.abs(rdT))))) <= 1.0
    # accumulate flag: a second call doubles dT
    wb.wbmm_backward_rect(x, None, dy, wh, ww, shift, layout, wb.FLAG_ACCUMULATE_DT, need_dx=False, dT=dT)
    assert float(np.max(np.abs(widen(dT) - 2 * rdT) / (tol * (2 * scale + np.abs(2 * rdT))))) <= 1.0


@pytest.mark.parametrize("wh,ww,shift", [(7, 14, (3, 5)), (3, 5, (0, 0)), (1, 9, (0, 4))])
def test_rect_one_hot_tables_and_integer_gradients_are_exact(wb, oracle, wh, ww, shift):
    """One-hot tables make the operator a pure shift inside the window (bitwise); small-integer x, dy make every sum of
    the table gradient exact in fp32: both must EQUAL the oracle -- pins Eq. 7's rectangular index on the device."""
    C, B, H, W = 16, 3, 3 * wh - 1, 2 * ww + 3
    nb = (2 * wh - 1) * (2 * ww - 1)
    g = torch.Generator().manual_seed(wh * 100 + ww)
    x = torch.randint(-3, 4, (B, C, H, W), generator=g).to(torch.bfloat16).cuda()
    dy = torch.randint(-2, 3, (B, C, H, W), generator=g).to(torch.bfloat16).cuda()
    bins = torch.randint(0, nb, (C,), generator=g)
    bins[0], bins[1], bins[2] = 0, nb - 1, (wh - 1) * (2 * ww - 1) + ww - 1
    T = torch.zeros((C, nb), dtype=torch.bfloat16, device="cuda")
    T[torch.arange(C), bins.cuda()] = 1.0
    y = wb.wbmm_forward_rect(x, T, wh, ww, shift)
    dx, dT = wb.wbmm_backward_rect(x, T, dy, wh, ww, shift)
    assert np.array_equal(widen(y), oracle.forward_rect(widen(x), widen(T), wh, ww, shift))
    rdx, rdT = oracle.backward_rect(widen(x), widen(T), widen(dy), wh, ww, shift)
    assert np.array_equal(widen(dx), rdx) and np.array_equal(widen(dT), rdT)


def test_rect_with_equal_sides_is_the_square_operator(wb):
    """w_w == w_h goes to wbmm_forward / wbmm_backward (the tensor-core kernels): identical results."""
    case = si.Case("rsq", 6, 8, 28, 56, 14, shift=(7, 3), seed=720, backward=True)
    d = si.make(case, device="cuda")
    y = wb.wbmm_forward_rect(d["x"], d["T"], 14, 14, case.shift)
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA
    assert torch.equal(y, wb.wbmm_forward(d["x"], d["T"], 14, case.shift))
    dx, dT = wb.wbmm_backward_rect(d["x"], d["T"], d["dy"], 14, 14, case.shift)
    rdx, rdT = wb.wbmm_backward(d["x"], d["T"], d["dy"], 14, case.shift)
    assert torch.equal(dx, rdx) and torch.allclose(dT, rdT, rtol=1e-4, atol=1e-3)


def test_rect_argument_validation(wb):
    x = torch.zeros((2, 4, 8, 8), dtype=torch.bfloat16, device="cuda")
    T = torch.zeros((4, 3 * 7), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(wb.WbmmError):        # shift_w must be < w_w
        wb.wbmm_forward_rect(x, T, 2, 4, (0, 4))
    with pytest.raises(wb.WbmmError):        # shift_h must be < w_h
        wb.wbmm_forward_rect(x, T, 2, 4, (2, 0))
    big = torch.zeros((1, 1, 64, 64), dtype=torch.float32, device="cuda")
    with pytest.raises(wb.WbmmError):        # 64 x 32 = 2048 positions: beyond what the kernels stage
        wb.wbmm_forward_rect(big, torch.zeros((1, 127 * 63), dtype=torch.float32, device="cuda"), 64, 32)
