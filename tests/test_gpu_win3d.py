"""3-D windows w_d x w_h x w_w on the GPU (wbmm_forward_win3d / wbmm_backward_win3d: the FFMA kernels of csrc/wbmm_rect.cu with
a depth axis) against the oracle's forward_3d / backward_3d (reading A23)."""
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


def _data(B, C, D, H, W, win, dtype, layout, seed):
    g = torch.Generator().manual_seed(seed)
    shape = (B, C, D, H, W) if layout == NCHW else (B, D, H, W, C)
    x = torch.randn(shape, generator=g).to(TD[dtype]).cuda()
    dy = torch.randn(shape, generator=g).to(TD[dtype]).cuda()
    nb = (2 * win[0] - 1) * (2 * win[1] - 1) * (2 * win[2] - 1)
    T = (torch.randn((C, nb), generator=g) * 0.05).to(TD[dtype]).cuda()
    return x, dy, T


f64 = lambda t: t.detach().cpu().double().numpy()

CASES = [
    # B, C, D, H, W, (wd, wh, ww), shift, dtype, layout
    (2, 3, 4, 14, 14, (2, 7, 7), (0, 0, 0), "f32", NCHW),            # video-style windows 2 x 7 x 7
    (2, 5, 5, 16, 13, (2, 7, 7), (1, 3, 2), "bf16", NCHW),           # ragged on every axis + shift
    (3, 8, 6, 9, 10, (3, 3, 4), (2, 1, 3), "f16", NHWC),
    (1, 4, 8, 8, 8, (8, 2, 2), (5, 0, 1), "f32", NHWC),              # deep windows
    (2, 3, 3, 12, 12, (1, 4, 4), (0, 2, 2), "bf16", NCHW),           # w_d = 1: slices are independent
    (1, 2, 4, 28, 28, (4, 7, 7), (2, 3, 3), "f32", NCHW),            # N = 196, 1183 bins
    (9, 2, 2, 7, 7, (2, 7, 7), (0, 0, 0), "bf16", NCHW),             # one window per volume, windows across several groups
]


@pytest.mark.parametrize("B,C,D,H,W,win,shift,dtype,layout", CASES)
def test_win3d_forward_and_backward_match_oracle(wb, oracle, B, C, D, H, W, win, shift, dtype, layout):
    x, dy, T = _data(B, C, D, H, W, win, dtype, layout, seed=1000 + B + 7 * C + D)
    y = wb.wbmm_forward_win3d(x, T, win, shift, layout)
    assert wb.wbmm_last_path() == wb.PATH_SIMT
    ry = oracle.forward_3d(f64(x), f64(T), win, shift, layout)
    assert max_err_over_tol(y, ry, TOL[dtype]) <= 1.0
    dx, dT = wb.wbmm_backward_win3d(x, T, dy, win, shift, layout)
    rdx, rdT = oracle.backward_3d(f64(x), f64(T), f64(dy), win, shift, layout)
    assert max_err_over_tol(dx, rdx, TOL[dtype]) <= 1.0
    nwin = B * -(-D // win[0]) * -(-H // win[1]) * -(-W // win[2])
    scale = float(np.sqrt(nwin * win[0] * win[1] * win[2]))
    assert float(np.max(np.abs(f64(dT) - rdT) / (1e-4 * (scale + np.abs(rdT))))) <= 1.0


def test_win3d_one_hot_table_every_bin_is_a_shift(wb, oracle):
    """One-hot tables at all (2w_d-1)(2w_h-1)(2w_w-1) bins (one per channel): bitwise equal to the oracle in float32."""
    win = (2, 3, 3)
    nb = 3 * 5 * 5
    g = torch.Generator().manual_seed(1100)
    x = torch.randn((2, nb, 4, 6, 6), generator=g).cuda()
    T = torch.eye(nb).cuda()
    y = wb.wbmm_forward_win3d(x, T, win, (1, 2, 0))
    assert np.array_equal(f64(y), oracle.forward_3d(f64(x), f64(T), win, (1, 2, 0)))


def test_win3d_integer_table_gradient_is_exact(wb, oracle):
    """Small-integer x and dy: every bin of dT is an exactly representable integer -- equality, not a tolerance."""
    win, shift = (2, 3, 2), (1, 1, 0)
    g = torch.Generator().manual_seed(1101)
    x = torch.randint(-3, 4, (3, 4, 5, 7, 6), generator=g).float().cuda()
    dy = torch.randint(-3, 4, (3, 4, 5, 7, 6), generator=g).float().cuda()
    _, dT = wb.wbmm_backward_win3d(x, None, dy, win, shift, need_dx=False)
    _, rdT = oracle.backward_3d(f64(x), None if False else np.zeros((4, 3 * 5 * 3)), f64(dy), win, shift, need_dx=False)
    assert np.array_equal(f64(dT), rdT)
    dT2 = dT.clone()
    wb.wbmm_backward_win3d(x, None, dy, win, shift, need_dx=False, dT=dT2, flags=wb.FLAG_ACCUMULATE_DT)
    assert np.array_equal(f64(dT2), 2 * rdT)


def test_win3d_depth_one_equals_the_rectangular_entry_point(wb):
    """D = w_d = 1: the same numbers as wbmm_forward_rect / wbmm_backward_rect (bitwise: same kernels, same order)."""
    g = torch.Generator().manual_seed(1102)
    x = torch.randn((3, 4, 1, 13, 11), generator=g).bfloat16().cuda()
    dy = torch.randn((3, 4, 1, 13, 11), generator=g).bfloat16().cuda()
    T = (torch.randn((4, 5 * 9), generator=g) * 0.05).bfloat16().cuda()
    y3 = wb.wbmm_forward_win3d(x, T, (1, 3, 5), (0, 2, 4))
    y2 = wb.wbmm_forward_rect(x[:, :, 0].contiguous(), T, 3, 5, (2, 4))
    assert torch.equal(y3[:, :, 0], y2)
    dx3, dT3 = wb.wbmm_backward_win3d(x, T, dy, (1, 3, 5), (0, 2, 4))
    dx2, dT2 = wb.wbmm_backward_rect(x[:, :, 0].contiguous(), T, dy[:, :, 0].contiguous(), 3, 5, (2, 4))
    assert torch.equal(dx3[:, :, 0], dx2) and torch.equal(dT3, dT2)


def test_win3d_argument_errors_and_limits(wb):
    x = torch.zeros((1, 2, 4, 8, 8), device="cuda")
    n0 = wb.wbmm_launch_count()
    with pytest.raises(wb.WbmmError) as ei:                                            # 16*8*8 = 1024 ok, 9*11*11 > 1024
        wb.wbmm_forward_win3d(torch.zeros((1, 1, 9, 11, 11), device="cuda"), torch.zeros((1, 17 * 21 * 21), device="cuda"), (9, 11, 11))
    assert ei.value.status == 2
    with pytest.raises(wb.WbmmError) as ei:                                            # shift_d out of range
        wb.wbmm_forward_win3d(x, torch.zeros((2, 3 * 3 * 3), device="cuda"), (2, 2, 2), (2, 0, 0))
    assert ei.value.status == 1
    assert wb.wbmm_launch_count() == n0
    e = torch.zeros((0, 2, 4, 8, 8), device="cuda")
    assert wb.wbmm_forward_win3d(e, torch.zeros((2, 27), device="cuda"), (2, 2, 2)).numel() == 0
