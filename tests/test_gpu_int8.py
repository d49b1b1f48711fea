"""INT8 forward on the GPU (wbmm_forward_int8, csrc/wbmm_tc_i8.cu: tcgen05.mma kind::i8) against the oracle's
forward_int8 (reading A21).  Integer work: every comparison is bit-exact."""
import numpy as np
import pytest
import torch

import synth_inputs as si

pytestmark = pytest.mark.gpu

NCHW, NHWC = si.NCHW, si.NHWC


@pytest.fixture(scope="module")
def wb():
    import paper_2607_02097_b200 as wb
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    wb.wbmm_version()          # loads libwbmm.so or raises: no silent fallback
    return wb


CASES = [
    si.Case("i8_w14_aligned", 5, 6, 28, 56, 14, seed=801),                            # 32-bit copies, several planes per tile
    si.Case("i8_w14_cfg_like", 9, 4, 56, 56, 14, seed=802),                           # 16 windows per image, ragged group
    si.Case("i8_w14_shift", 3, 5, 56, 56, 14, shift=(7, 3), seed=803),
    si.Case("i8_w14_ragged", 3, 4, 60, 50, 14, shift=(2, 13), seed=804),
    si.Case("i8_w14_nhwc", 3, 8, 30, 44, 14, shift=(5, 0), layout=NHWC, seed=805),
    si.Case("i8_w14_strips", 2, 3, 224, 224, 14, seed=806),                           # 256 windows per image: strips
    si.Case("i8_w14_one_window", 130, 2, 14, 14, 14, seed=807),                       # 128 + 2 planes per channel
    si.Case("i8_w7_aligned", 4, 6, 28, 28, 7, seed=808),
    si.Case("i8_w7_shift_ragged", 3, 5, 30, 33, 7, shift=(3, 6), seed=809),
    si.Case("i8_w7_nhwc", 2, 16, 56, 56, 7, layout=NHWC, seed=810),
    si.Case("i8_w7_one_window", 131, 3, 7, 7, 7, seed=811),
    si.Case("i8_w7_wide", 1, 2, 7, 896, 7, seed=812),                                 # 128 windows across
    si.Case("i8_odd_width", 2, 3, 28, 54, 14, seed=813),                              # W' != W: byte copies
    si.Case("i8_w14_shift_strips", 2, 3, 224, 224, 14, shift=(5, 9), seed=817),       # two row runs per strip, several strips
    si.Case("i8_w14_shift_bytes", 3, 4, 28, 42, 14, shift=(3, 11), seed=818),         # W % 4 != 0: byte units
    si.Case("i8_w7_shift_bytes", 2, 3, 28, 21, 7, shift=(2, 5), seed=819),
    si.Case("i8_w14_row_shift_only", 4, 3, 56, 28, 14, shift=(9, 0), seed=820),
    si.Case("i8_w14_col_shift_only", 4, 3, 28, 56, 14, shift=(0, 13), seed=821),
    si.Case("i8_w14_nhwc_t", 5, 32, 28, 56, 14, layout=NHWC, seed=814),               # NHWC through the transposition route
    si.Case("i8_w14_nhwc_t_shift", 3, 96, 56, 56, 14, shift=(7, 5), layout=NHWC, seed=815),
    si.Case("i8_w7_nhwc_t", 4, 80, 28, 28, 7, layout=NHWC, seed=816),                 # C = 64 + 16: a partial tile
]


@pytest.mark.parametrize("case", CASES, ids=lambda c: c.name)
@pytest.mark.parametrize("extreme", [False, True], ids=["typical", "extreme"])
def test_int8_forward_bit_exact(wb, oracle, case, extreme):
    d = si.make_int8(case, device="cuda", extreme=extreme)
    xh, Th, sh = d["x"].cpu().numpy(), d["T"].cpu().numpy(), d["scale"].cpu().numpy()
    want32 = oracle.forward_int8(xh, Th, case.w, case.shift, case.layout)
    out = torch.full(d["x"].shape, -77, dtype=torch.int32, device="cuda")
    y32 = wb.wbmm_forward_int8(d["x"], d["T"], case.w, case.shift, case.layout, out=out)
    assert wb.wbmm_last_path() in (wb.PATH_TC_GATHER, wb.PATH_TC_TMA, wb.PATH_TC_TRANSPOSED)
    if case.name.startswith("i8_w14_nhwc_t") or case.name == "i8_w7_nhwc_t":
        assert wb.wbmm_last_path() == wb.PATH_TC_TRANSPOSED
        yn = wb.wbmm_forward_int8(d["x"], d["T"], case.w, case.shift, case.layout, flags=wb.FLAG_NO_SCRATCH)
        assert wb.wbmm_last_path() == wb.PATH_TC_GATHER and np.array_equal(yn.cpu().numpy(), want32)
    assert np.array_equal(y32.cpu().numpy(), want32), case.name
    want8 = oracle.forward_int8(xh, Th, case.w, case.shift, case.layout, scale=sh)
    y8 = wb.wbmm_forward_int8(d["x"], d["T"], case.w, case.shift, case.layout, scale=d["scale"])
    assert np.array_equal(y8.cpu().numpy(), want8), case.name
    if not extreme:
        assert np.abs(want8.astype(np.int32)).max() > 60           # the scales exercise the range, and some saturate


@pytest.mark.parametrize("w", [7, 14])
def test_int8_one_hot_table_every_bin(wb, oracle, w):
    """One-hot tables, one bin per channel, all (2w-1)^2 bins: the output is a signed shift of x inside each window."""
    nb = (2 * w - 1) ** 2
    rng = np.random.default_rng(820 + w)
    x = torch.from_numpy(rng.integers(-128, 128, (2, nb, 2 * w, 2 * w), dtype=np.int8)).cuda()
    T = torch.zeros((nb, nb), dtype=torch.int8)
    T[torch.arange(nb), torch.arange(nb)] = torch.from_numpy(rng.choice(np.array([-128, -1, 1, 127], dtype=np.int8), nb))
    y = wb.wbmm_forward_int8(x, T.cuda(), w)
    assert np.array_equal(y.cpu().numpy(), oracle.forward_int8(x.cpu().numpy(), T.numpy(), w))


def test_int8_requantisation_ties_and_saturation(wb):
    """Identity table: the sum is x, so q has a closed form; scales 0.5 / 1.5 / -2 give ties, saturation on both sides."""
    x = torch.arange(-128, 128, dtype=torch.int16).to(torch.int8).reshape(1, 1, 16, 16).repeat(1, 3, 1, 1).contiguous().cuda()
    x = torch.nn.functional.pad(x, (0, 12, 0, 12)).contiguous()                     # 28 x 28 map, w = 14
    T = torch.zeros((3, 729), dtype=torch.int8)
    T[:, 364] = 1
    scale = torch.tensor([0.5, 1.5, -2.0], dtype=torch.float32)
    q = wb.wbmm_forward_int8(x, T.cuda(), 14, scale=scale.cuda()).cpu().numpy().astype(np.int32)
    xi = x.cpu().numpy().astype(np.float64)
    for c, s in enumerate([0.5, 1.5, -2.0]):
        a = xi[0, c] * s
        f = np.floor(a)
        r = np.where(a - f > 0.5, f + 1, np.where(a - f < 0.5, f, np.where(f % 2 == 0, f, f + 1)))
        assert np.array_equal(q[0, c], np.clip(r, -128, 127).astype(np.int32)), c


def test_int8_output_is_fully_overwritten_and_nothing_else(wb, oracle):
    case = si.Case("i8_canary", 3, 4, 30, 44, 14, shift=(3, 5), seed=830)
    d = si.make_int8(case, device="cuda")
    n = d["x"].numel()
    for scale, dt in ((None, torch.int32), (d["scale"], torch.int8)):
        buf = torch.full((n + 512,), 91, dtype=dt, device="cuda")
        out = buf[256:256 + n].view(d["x"].shape)
        wb.wbmm_forward_int8(d["x"], d["T"], case.w, case.shift, scale=scale, out=out)
        torch.cuda.synchronize()
        assert bool((buf[:256] == 91).all()) and bool((buf[256 + n:] == 91).all())
        want = oracle.forward_int8(d["x"].cpu().numpy(), d["T"].cpu().numpy(), case.w, case.shift,
                                   scale=None if scale is None else scale.cpu().numpy())
        assert np.array_equal(out.cpu().numpy(), want)


@pytest.mark.parametrize("off", [0, 1, 4, 16])
def test_int8_pointer_alignment_picks_a_kernel_that_fits(wb, oracle, off):
    """x and y at byte offsets 0 / 1 / 4 / 16 inside larger buffers: bulk copies need 16, 32-bit copies 4, else bytes."""
    case = si.Case("i8_align", 9, 3, 56, 56, 14, seed=840)
    d = si.make_int8(case, device="cuda")
    n = d["x"].numel()
    xb = torch.zeros(n + 64, dtype=torch.int8, device="cuda")
    xs = xb[off:off + n].view(d["x"].shape)
    xs.copy_(d["x"])
    yb = torch.full((n + 64,), 55, dtype=torch.int8, device="cuda")
    ys = yb[off:off + n].view(d["x"].shape)
    wb.wbmm_forward_int8(xs, d["T"], case.w, scale=d["scale"], out=ys)
    want = oracle.forward_int8(d["x"].cpu().numpy(), d["T"].cpu().numpy(), case.w, scale=d["scale"].cpu().numpy())
    assert np.array_equal(ys.cpu().numpy(), want)
    assert bool((yb[:off] == 55).all()) and bool((yb[off + n:] == 55).all())
    assert wb.wbmm_last_path() == (wb.PATH_TC_TMA if off % 16 == 0 else wb.PATH_TC_GATHER)
    y32 = wb.wbmm_forward_int8(xs, d["T"], case.w)
    assert np.array_equal(y32.cpu().numpy(), oracle.forward_int8(d["x"].cpu().numpy(), d["T"].cpu().numpy(), case.w))


def test_int8_full_size_headline_shape(wb, oracle):
    """B128 C96 56x56 w=14 (the headline shape of BASELINE.json in int8), whole tensor, both outputs."""
    case = si.Case("i8_cfg3", 128, 96, 56, 56, 14, seed=850)
    d = si.make_int8(case, device="cuda")
    xh, Th, sh = d["x"].cpu().numpy(), d["T"].cpu().numpy(), d["scale"].cpu().numpy()
    y8 = wb.wbmm_forward_int8(d["x"], d["T"], 14, scale=d["scale"])
    assert np.array_equal(y8.cpu().numpy(), oracle.forward_int8(xh, Th, 14, scale=sh))
    y32 = wb.wbmm_forward_int8(d["x"], d["T"], 14)
    assert np.array_equal(y32.cpu().numpy(), oracle.forward_int8(xh, Th, 14))
    case = si.Case("i8_cfg2", 128, 96, 56, 56, 7, seed=851)
    d = si.make_int8(case, device="cuda")
    y8 = wb.wbmm_forward_int8(d["x"], d["T"], 7, scale=d["scale"])
    assert np.array_equal(y8.cpu().numpy(), oracle.forward_int8(d["x"].cpu().numpy(), d["T"].cpu().numpy(), 7, scale=d["scale"].cpu().numpy()))


def test_int8_full_size_shifted_and_nhwc(wb, oracle):
    """Config 5's shape (B64 C192 28x28 w=14 shift 7,7) and the headline shape in NHWC, whole tensors: the gather kernel and the
    transposition route at full size."""
    case = si.Case("i8_cfg5", 64, 192, 28, 28, 14, shift=(7, 7), seed=860)
    d = si.make_int8(case, device="cuda")
    y8 = wb.wbmm_forward_int8(d["x"], d["T"], 14, case.shift, scale=d["scale"])
    assert wb.wbmm_last_path() == wb.PATH_TC_GATHER
    assert np.array_equal(y8.cpu().numpy(), oracle.forward_int8(d["x"].cpu().numpy(), d["T"].cpu().numpy(), 14, case.shift,
                                                                 scale=d["scale"].cpu().numpy()))
    case = si.Case("i8_cfg3_nhwc", 128, 96, 56, 56, 14, layout=NHWC, seed=861)
    d = si.make_int8(case, device="cuda")
    y8 = wb.wbmm_forward_int8(d["x"], d["T"], 14, layout=NHWC, scale=d["scale"])
    assert wb.wbmm_last_path() == wb.PATH_TC_TRANSPOSED
    assert np.array_equal(y8.cpu().numpy(), oracle.forward_int8(d["x"].cpu().numpy(), d["T"].cpu().numpy(), 14, layout=NHWC,
                                                                 scale=d["scale"].cpu().numpy()))


def test_int8_unsupported_and_argument_errors(wb):
    x = torch.zeros((1, 2, 10, 10), dtype=torch.int8, device="cuda")
    n0 = wb.wbmm_launch_count()
    with pytest.raises(wb.WbmmError) as ei:
        wb.wbmm_forward_int8(x, torch.zeros((2, 81), dtype=torch.int8, device="cuda"), 5)
    assert ei.value.status == 2
    xw = torch.zeros((1, 1, 7, 7 * 129), dtype=torch.int8, device="cuda")         # 129 windows across
    with pytest.raises(wb.WbmmError) as ei:
        wb.wbmm_forward_int8(xw, torch.zeros((1, 169), dtype=torch.int8, device="cuda"), 7)
    assert ei.value.status == 2
    assert wb.wbmm_launch_count() == n0
    with pytest.raises(TypeError):
        wb.wbmm_forward_int8(x.float(), torch.zeros((2, 169), dtype=torch.int8, device="cuda"), 7)
    # empty batch: nothing to do
    e = torch.zeros((0, 2, 14, 14), dtype=torch.int8, device="cuda")
    assert wb.wbmm_forward_int8(e, torch.zeros((2, 729), dtype=torch.int8, device="cuda"), 14).numel() == 0
