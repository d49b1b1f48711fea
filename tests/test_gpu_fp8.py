"""FP8 (E4M3) forward on the GPU (wbmm_forward_fp8, csrc/wbmm_tc_i8.cu: tcgen05.mma kind::f8f6f4) against the oracle's
forward_fp8 -- the exact real-valued operator on the decoded values (reading A22).
float32 sums: within float32 accumulation error of the exact sum.  E4M3 output: the stored code is one of the two E4M3
neighbours of sum * scale, and the nearest one unless the number lies within that error of their midpoint."""
import numpy as np
import pytest
import torch

import synth_inputs as si

pytestmark = pytest.mark.gpu

NCHW, NHWC = si.NCHW, si.NHWC
ACC_EPS = 2.0 ** -20          # float32 accumulation of <= 196 exact products: <= ~N * 2^-24 of the sum of |products|


@pytest.fixture(scope="module")
def wb():
    import paper_2607_02097_b200 as wb
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    wb.wbmm_version()
    return wb


def codes(t):
    return t.view(torch.uint8).cpu().numpy()


CASES = [
    si.Case("f8_w14_aligned", 5, 6, 28, 56, 14, seed=901),
    si.Case("f8_w14_cfg_like", 9, 4, 56, 56, 14, seed=902),
    si.Case("f8_w14_shift_ragged", 3, 4, 60, 50, 14, shift=(2, 13), seed=903),
    si.Case("f8_w14_nhwc_t", 3, 32, 28, 56, 14, shift=(5, 0), layout=NHWC, seed=904),
    si.Case("f8_w14_nhwc_gather", 3, 8, 30, 44, 14, layout=NHWC, seed=905),
    si.Case("f8_w14_strips", 2, 3, 224, 224, 14, seed=906),
    si.Case("f8_w7_aligned", 4, 6, 28, 28, 7, seed=907),
    si.Case("f8_w7_shift_ragged", 3, 5, 30, 33, 7, shift=(3, 6), seed=908),
    si.Case("f8_w7_one_window", 131, 3, 7, 7, 7, seed=909),
    si.Case("f8_w14_shift_unpadded", 5, 4, 56, 56, 14, shift=(7, 7), seed=910),       # rotated-window form
    si.Case("f8_w7_shift_bytes", 2, 3, 28, 21, 7, shift=(2, 5), seed=911),
]


def check_codes(q_codes, r, err, oracle):
    """q_codes: stored E4M3 bytes; r: the exact real numbers; err: accumulation error bound per element."""
    grid = np.unique(oracle.e4m3_decode(np.arange(256, dtype=np.uint8))[[c for c in range(256) if (c & 0x7f) != 0x7f]])
    q = oracle.e4m3_decode(q_codes)
    assert not np.isnan(q).any()
    rc = np.clip(r, -448.0, 448.0)
    hi_i = np.clip(np.searchsorted(grid, rc, side="left"), 0, len(grid) - 1)
    hi = grid[hi_i]
    lo = grid[np.maximum(hi_i - 1, 0)]
    lo = np.where(hi == rc, hi, lo)                         # exactly representable: both neighbours are the number itself
    assert np.all((q == lo) | (q == hi)), "a stored code is not a neighbour of the exact value"
    mid = 0.5 * (lo + hi)
    clear = np.abs(rc - mid) > err + 1e-12 * np.abs(mid)
    nearest = np.where(np.abs(rc - lo) <= np.abs(rc - hi), lo, hi)
    assert np.all(~clear | (q == nearest)), "a stored code is not the nearest E4M3 number"
    return float(clear.mean())


@pytest.mark.parametrize("case", CASES, ids=lambda c: c.name)
def test_fp8_forward_against_the_exact_operator(wb, oracle, case):
    d = si.make_fp8(case, device="cuda")
    xc, Tc, sc = codes(d["x"]), codes(d["T"]), d["scale"].cpu().numpy().astype(np.float64)
    ref = oracle.forward_fp8(xc, Tc, case.w, case.shift, case.layout)
    mag = oracle.forward(np.abs(oracle.e4m3_decode(xc)), np.abs(oracle.e4m3_decode(Tc)), case.w, case.shift, case.layout)
    out = torch.full(d["x"].shape, 123.0, dtype=torch.float32, device="cuda")
    y = wb.wbmm_forward_fp8(d["x"], d["T"], case.w, case.shift, case.layout, out=out).cpu().numpy().astype(np.float64)
    assert np.all(np.abs(y - ref) <= ACC_EPS * mag + 1e-30), float(np.max(np.abs(y - ref) / (mag + 1e-30)))
    q = wb.wbmm_forward_fp8(d["x"], d["T"], case.w, case.shift, case.layout, scale=d["scale"])
    scb = sc[None, :, None, None] if case.layout == NCHW else sc[None, None, None, :]
    frac_clear = check_codes(codes(q), ref * scb, (ACC_EPS * mag + np.abs(ref) * 2.0 ** -23) * np.abs(scb), oracle)
    assert frac_clear > 0.99                                # the midpoint exemption is rare, not a loophole
    assert np.abs(oracle.e4m3_decode(codes(q))).max() >= 16.0   # the scales exercise the range


@pytest.mark.parametrize("w", [14, 7])
def test_fp8_full_size_headline_shape(wb, oracle, w):
    """B128 C96 56x56 (the headline shape of BASELINE.json in E4M3), whole tensor, in the launch configuration bench.py times."""
    case = si.Case("f8_full", 128, 96, 56, 56, w, seed=950 + w)
    d = si.make_fp8(case, device="cuda")
    xc, Tc, sc = codes(d["x"]), codes(d["T"]), d["scale"].cpu().numpy().astype(np.float64)
    ref = oracle.forward_fp8(xc, Tc, w)
    mag = oracle.forward(np.abs(oracle.e4m3_decode(xc)), np.abs(oracle.e4m3_decode(Tc)), w)
    y = wb.wbmm_forward_fp8(d["x"], d["T"], w).cpu().numpy().astype(np.float64)
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA
    assert np.all(np.abs(y - ref) <= ACC_EPS * mag + 1e-30)
    q = wb.wbmm_forward_fp8(d["x"], d["T"], w, scale=d["scale"])
    scb = sc[None, :, None, None]
    assert check_codes(codes(q), ref * scb, (ACC_EPS * mag + np.abs(ref) * 2.0 ** -23) * np.abs(scb), oracle) > 0.99


@pytest.mark.parametrize("w", [7, 14])
def test_fp8_one_hot_table_every_bin_is_exact(wb, oracle, w):
    """One bin = +-1 or +-2 per channel: every output is a signed, scaled copy of one input -- exact in float32."""
    nb = (2 * w - 1) ** 2
    g = torch.Generator().manual_seed(920 + w)
    x = torch.randn((2, nb, 2 * w, 2 * w), generator=g).to(torch.float8_e4m3fn).cuda()
    T = torch.zeros((nb, nb))
    T[torch.arange(nb), torch.arange(nb)] = torch.tensor([1.0, -1.0, 2.0, -2.0])[torch.randint(0, 4, (nb,), generator=g)]
    T8 = T.to(torch.float8_e4m3fn).cuda()
    y = wb.wbmm_forward_fp8(x, T8, w).cpu().numpy().astype(np.float64)
    assert np.array_equal(y, oracle.forward_fp8(codes(x), codes(T8), w))


def test_fp8_saturation_and_exact_codes(wb, oracle):
    """Identity table: sum = x; scale 1 returns the input codes (up to the sign of zero), scale 1000 saturates at +-448."""
    g = torch.Generator().manual_seed(930)
    x = (torch.randn((3, 2, 28, 28), generator=g) * 20).to(torch.float8_e4m3fn).cuda()
    T = torch.zeros((2, 729))
    T[:, 364] = 1.0
    T8 = T.to(torch.float8_e4m3fn).cuda()
    q = wb.wbmm_forward_fp8(x, T8, 14, scale=torch.tensor([1.0, 1000.0]).cuda())
    xv, qv = oracle.e4m3_decode(codes(x)), oracle.e4m3_decode(codes(q))
    assert np.array_equal(qv[:, 0], xv[:, 0])
    assert np.array_equal(qv[:, 1], np.clip(xv[:, 1] * 1000.0, -448.0, 448.0) * (np.abs(xv[:, 1]) * 1000.0 >= 448.0)
                          + qv[:, 1] * (np.abs(xv[:, 1]) * 1000.0 < 448.0))
    assert np.abs(qv[:, 1]).max() == 448.0


def test_fp8_output_is_fully_overwritten_and_nothing_else(wb, oracle):
    case = si.Case("f8_canary", 3, 4, 30, 44, 14, shift=(3, 5), seed=940)
    d = si.make_fp8(case, device="cuda")
    n = d["x"].numel()
    buf = torch.full((n + 512,), 91, dtype=torch.uint8, device="cuda")
    out = buf[256:256 + n].view(d["x"].shape).view(torch.float8_e4m3fn)
    wb.wbmm_forward_fp8(d["x"], d["T"], case.w, case.shift, scale=d["scale"], out=out)
    torch.cuda.synchronize()
    assert bool((buf[:256] == 91).all()) and bool((buf[256 + n:] == 91).all())
    with pytest.raises(TypeError):
        wb.wbmm_forward_fp8(d["x"].view(torch.int8), d["T"], case.w)
