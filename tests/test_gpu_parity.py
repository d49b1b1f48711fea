"""GPU parity: libwbmm.so (through the C ABI, via the ctypes binding) against the CPU oracle,
element by element on the same seeded inputs.  Bar (BASELINE.json north_star):
|got - ref| <= tol*(1+|ref|), tol = 1e-2 for bf16/fp16 (fp32 accumulate), 1e-4 for fp32;
relative-position indexing and data movement bit-exact.
"""
import numpy as np
import pytest
import torch

import synth_inputs as si
from parity import TOL, max_err_over_tol, plane_subset, take_planes, widen

pytestmark = pytest.mark.gpu

NCHW, NHWC = si.NCHW, si.NHWC


@pytest.fixture(scope="module")
def wb():
    import paper_2607_02097_b200 as wb
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    wb.wbmm_version()          # loads libwbmm.so or raises: no silent fallback
    global NHWC_TC_PATHS
    NHWC_TC_PATHS = (wb.PATH_TC_TMA, wb.PATH_TC_TRANSPOSED)
    return wb


def run_forward(wb, oracle, case, flags=0, sample=None, expect_path=None):
    d = si.make(case, device="cuda")
    y = wb.wbmm_forward(d["x"], d["T"], case.w, case.shift, case.layout, flags)
    torch.cuda.synchronize()
    path = wb.wbmm_last_path()
    if expect_path is not None:
        assert path == expect_path, wb.wbmm_path_string(path)
    bs = cs = None
    if sample:
        bs, cs = plane_subset(case, *sample)
    xs = take_planes(d["x"], case.layout, bs, cs)
    Ts = d["T"].cpu() if cs is None else d["T"].cpu().index_select(0, cs)
    ref = oracle.forward(widen(xs), widen(Ts), case.w, case.shift, case.layout, "direct")
    err = max_err_over_tol(take_planes(y, case.layout, bs, cs), ref, TOL[case.dtype])
    return err, path


# Table gradient (fp32 output): each bin sums n = L * mult(k) products |dy x| ~ 1 in fp32:
# rounding error ~ 2^-24 * sqrt(n) * |partial sums| -- far inside 1e-4 * (sqrt(n_max) + |ref|), n_max = L * N the
# centre bin's term count.  100 x tighter than the 1e-2 form of the 16-bit outputs; one dropped window moves a
# bin by ~sqrt(mult) >> this bound.
def dT_err_over_tol(dT, ref, case, tol=1e-4):
    g = widen(dT)
    assert g.shape == ref.shape and np.isfinite(g).all()
    nwin = case.B * (-(-case.H // case.w)) * (-(-case.W // case.w))
    scale = float(np.sqrt(nwin * case.w * case.w))
    return float(np.max(np.abs(g - ref) / (tol * (scale + np.abs(ref)))))


NHWC_TC_PATHS = ()      # filled in by the wb fixture: the tensor-core paths an NHWC call may report


def run_backward(wb, oracle, case, flags=0, sample_c=None):
    d = si.make(case, device="cuda")
    dx, dT = wb.wbmm_backward(d["x"], d["T"], d["dy"], case.w, case.shift, case.layout, flags)
    torch.cuda.synchronize()
    cs = None
    if sample_c:
        _, cs = plane_subset(case, case.B, sample_c)
    xs, gs = (take_planes(d[k], case.layout, None, cs) for k in ("x", "dy"))
    Ts = d["T"].cpu() if cs is None else d["T"].cpu().index_select(0, cs)
    rdx, rdT = oracle.backward(widen(xs), widen(Ts), widen(gs), case.w, case.shift, case.layout)
    e_dx = max_err_over_tol(take_planes(dx, case.layout, None, cs), rdx, TOL[case.dtype])
    dTs = dT.cpu() if cs is None else dT.cpu().index_select(0, cs)
    e_dT = max(max_err_over_tol(dTs, rdT, TOL[case.dtype]), dT_err_over_tol(dTs, rdT, case))
    return e_dx, e_dT


# ------------------------------------------------------------------ small cases, every variant
SMALL = [
    si.Case("s_w3", 2, 3, 6, 9, 3, dtype="f32"),
    si.Case("s_w4_ragged", 3, 5, 10, 7, 4, dtype="f32"),
    si.Case("s_w7_shift", 2, 4, 14, 21, 7, dtype="f32", shift=(3, 2)),
    si.Case("s_w14", 3, 5, 28, 42, 14, dtype="bf16"),
    si.Case("s_w14_ragged_shift", 2, 9, 30, 25, 14, dtype="bf16", shift=(7, 5)),
    si.Case("s_w7_f16", 5, 17, 21, 28, 7, dtype="f16"),
    si.Case("s_w1", 2, 3, 5, 4, 1, dtype="f32"),
    si.Case("s_w16", 1, 2, 32, 16, 16, dtype="bf16"),
    si.Case("s_w20", 1, 2, 20, 40, 20, dtype="f32"),
    si.Case("s_many_windows", 33, 3, 28, 28, 7, dtype="bf16"),     # several blocks + ragged tail
]


@pytest.mark.parametrize("case", SMALL, ids=lambda c: c.name)
@pytest.mark.parametrize("layout", [NCHW, NHWC])
@pytest.mark.parametrize("force_simt", [True, False])
def test_forward_small(wb, oracle, case, layout, force_simt):
    case = si.with_(case, layout=layout)
    err, _ = run_forward(wb, oracle, case, wb.FLAG_FORCE_SIMT if force_simt else 0)
    assert err <= 1.0, err


@pytest.mark.parametrize("case", SMALL, ids=lambda c: c.name)
@pytest.mark.parametrize("layout", [NCHW, NHWC])
@pytest.mark.parametrize("force_simt", [True, False])
def test_backward_small(wb, oracle, case, layout, force_simt):
    case = si.with_(case, layout=layout, backward=True)
    e_dx, e_dT = run_backward(wb, oracle, case, wb.FLAG_FORCE_SIMT if force_simt else 0)
    assert e_dx <= 1.0 and e_dT <= 1.0, (e_dx, e_dT)


# ------------------------------------------------------------------ the pipelined kernels, every mode
# Shapes chosen so that the warp-specialised bulk kernel (NCHW) / the 8-channel-group kernel (NHWC)
# serve them -- asserted through wbmm_last_path() -- with ragged tails in every tiling dimension:
# B not a multiple of the images per tile, several tiles and channels per CTA, strips of big maps,
# shift with odd and even column offsets, padding, fp16.
PIPE = [
    si.Case("p_w14_plain", 19, 5, 56, 56, 14),                               # 8 images per tile, tail of 3
    si.Case("p_w14_many_tiles", 40, 160, 28, 28, 14),                        # 32 images per tile, > 148 tiles
    si.Case("p_w14_shift_odd", 9, 7, 28, 56, 14, shift=(7, 7)),              # odd column start: funnel shifts
    si.Case("p_w14_shift_even", 9, 7, 28, 56, 14, shift=(3, 4)),
    si.Case("p_w14_ragged", 7, 6, 60, 60, 14),                               # 25 windows per image, W' = 70
    si.Case("p_w14_ragged_shift", 6, 5, 36, 40, 14, shift=(5, 9)),
    si.Case("p_w14_strips", 3, 4, 168, 112, 14),                             # 96 windows per image: 2 images / tile
    si.Case("p_w14_big_map", 2, 3, 224, 224, 14),                            # 256 windows per image: row strips
    si.Case("p_w14_f16", 10, 9, 42, 56, 14, dtype="f16", shift=(0, 7)),
    si.Case("p_w14_big_map_shift", 2, 3, 224, 224, 14, shift=(7, 7)),        # row strips in rolled order: two row runs
    si.Case("p_w7_strips_shift", 3, 5, 112, 112, 7, shift=(3, 4)),
    si.Case("p_w7_strips_ragged", 2, 4, 108, 112, 7, shift=(2, 0)),          # last strip partly in the padding
    si.Case("p_w7_plain", 21, 6, 56, 56, 7),                                 # 64 windows per image
    si.Case("p_w7_strips", 3, 5, 112, 112, 7),                               # 256 windows per image: strips
    si.Case("p_w7_shift", 5, 7, 28, 28, 7, shift=(3, 2)),
    si.Case("p_w7_ragged", 6, 4, 26, 30, 7, shift=(0, 3)),                   # W' = 35 is odd and columns wrap: generic path
    si.Case("p_w7_ragged_noshift", 6, 4, 30, 60, 7),                         # W' = 63 is odd, nothing wraps: pipelined
    si.Case("p_w7_ragged_rowshift", 5, 3, 60, 60, 7, shift=(3, 0)),          # rows wrap, columns do not
    si.Case("p_w7_f16", 33, 3, 28, 56, 7, dtype="f16"),
]


def _nhwc_path(wb, case, flags):
    """NHWC forward / dX: w = 7 without a shift runs in one pass straight from NHWC memory (pipelined channel-group
    kernel); otherwise transposition scratch around the NCHW kernels when C and H*W are multiples of 8, else (or with
    FLAG_NO_SCRATCH) the block-synchronous 8-channel-group kernels -- which need an even W' at odd w; what is left
    (here: W' = 63) takes the FFMA kernels."""
    if case.w == 7 and tuple(case.shift) == (0, 0) and case.C % 8 == 0:
        return wb.PATH_TC_TMA
    via_scratch = not (flags & wb.FLAG_NO_SCRATCH) and case.C % 8 == 0 and (case.H * case.W) % 8 == 0
    if via_scratch:
        return wb.PATH_TC_TRANSPOSED
    Wp = -(-case.W // case.w) * case.w
    return wb.PATH_SIMT if (case.w % 2 == 1 and Wp % 2 == 1) else wb.PATH_TC_GATHER


@pytest.mark.parametrize("case", PIPE, ids=lambda c: c.name)
@pytest.mark.parametrize("layout,no_scratch", [(NCHW, False), (NHWC, False), (NHWC, True)])
def test_pipelined_kernels_forward_backward(wb, oracle, case, layout, no_scratch):
    C = case.C if layout == NCHW else -(-case.C // 8) * 8                     # NHWC paths: 8-channel groups
    case = si.with_(case, layout=layout, C=C, backward=True)
    flags = wb.FLAG_NO_SCRATCH if no_scratch else 0
    d = si.make(case, device="cuda")
    y = wb.wbmm_forward(d["x"], d["T"], case.w, case.shift, case.layout, flags)
    torch.cuda.synchronize()
    path = wb.wbmm_last_path()
    if case.name != "p_w7_ragged":
        assert path == (wb.PATH_TC_TMA if layout == NCHW else _nhwc_path(wb, case, flags)), wb.wbmm_path_string(path)
    dx, dT = wb.wbmm_backward(d["x"], d["T"], d["dy"], case.w, case.shift, case.layout, flags)
    torch.cuda.synchronize()
    ry = oracle.forward(widen(d["x"]), widen(d["T"]), case.w, case.shift, case.layout, "direct")
    rdx, rdT = oracle.backward(widen(d["x"]), widen(d["T"]), widen(d["dy"]), case.w, case.shift, case.layout)
    tol = TOL[case.dtype]
    errs = (max_err_over_tol(y, ry, tol), max_err_over_tol(dx, rdx, tol), max_err_over_tol(dT, rdT, tol))
    assert max(errs) <= 1.0, errs


@pytest.mark.parametrize("w,shift,H,W", [(14, (0, 0), 56, 56), (14, (7, 7), 28, 56), (14, (2, 5), 60, 60),
                                         (7, (0, 0), 56, 56), (7, (3, 4), 28, 28)])
@pytest.mark.parametrize("layout,no_scratch", [(NCHW, False), (NHWC, False), (NHWC, True)])
def test_pipelined_kernels_one_hot_bins_bitwise(wb, oracle, w, shift, H, W, layout, no_scratch):
    """One-hot tables through the pipelined kernels (bulk / NHWC group kernel): pure data movement,
    so the result must equal the oracle's bitwise -- the bit-exact indexing test of the Toeplitz
    library, the word-granular shift / padding addressing and the NHWC transposition."""
    tw = 2 * w - 1
    nb = tw * tw
    C = 64
    case = si.Case("onehot_pipe", 9, C, H, W, w, dtype="bf16", layout=layout, shift=shift, seed=31)
    d = si.make(case, device="cuda")
    g = torch.Generator().manual_seed(w * 1000 + H)
    bins = torch.randint(0, nb, (C,), generator=g)
    bins[0], bins[1], bins[2] = 0, nb - 1, (w - 1) * tw + (w - 1)            # corners and the centre
    T = torch.zeros_like(d["T"])
    T[torch.arange(C), bins.to(T.device)] = 1.0
    flags = wb.FLAG_NO_SCRATCH if no_scratch else 0
    y = wb.wbmm_forward(d["x"], T, w, shift, layout, flags)
    assert wb.wbmm_last_path() == (wb.PATH_TC_TMA if layout == NCHW else _nhwc_path(wb, case, flags))
    ref = oracle.forward(widen(d["x"]), widen(T), w, shift, layout)
    assert np.array_equal(widen(y), ref)
    dx, _ = wb.wbmm_backward(None, T, d["x"], w, shift, layout, flags, need_dT=False)
    rdx, _ = oracle.backward(widen(d["x"]), widen(T), widen(d["x"]), w, shift, layout, need_dT=False)
    assert np.array_equal(widen(dx), rdx)


@pytest.mark.parametrize("case", [
    si.Case("fork_w14_shift", 24, 12, 28, 28, 14, shift=(7, 7), seed=140, backward=True),
    si.Case("fork_w7", 21, 10, 56, 56, 7, seed=141, backward=True),
    si.Case("fork_nhwc_w14", 6, 16, 28, 56, 14, layout=NHWC, seed=142, backward=True),      # scratch allocated on the internal stream
    si.Case("fork_f32", 5, 3, 56, 56, 14, dtype="f32", seed=143, backward=True),
], ids=lambda c: c.name)
def test_backward_forks_the_table_gradient_and_joins(wb, oracle, case):
    """wbmm_backward with dx and dT runs the table gradient on an internal stream forked from / joined into the
    caller's (WBMM_FLAG_NO_FORK: one after the other).  Same results either way; work queued behind the call on the
    caller's stream sees both outputs; the call can be captured into a CUDA graph and replayed."""
    d = si.make(case, device="cuda")
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        dx0, dT0 = wb.wbmm_backward(d["x"], d["T"], d["dy"], case.w, case.shift, case.layout, wb.FLAG_NO_FORK)
        dx1, dT1 = wb.wbmm_backward(d["x"], d["T"], d["dy"], case.w, case.shift, case.layout)
        after = dT1.clone()                      # queued behind the call on the caller's stream: must see the joined dT
        dxg, dTg = torch.empty_like(dx1), torch.empty_like(dT1)
        torch.cuda.synchronize()
        gr = torch.cuda.CUDAGraph()
        with torch.cuda.graph(gr, stream=s):
            wb.wbmm_backward(d["x"], d["T"], d["dy"], case.w, case.shift, case.layout, dx=dxg, dT=dTg)
        dxg.fill_(7.0); dTg.fill_(7.0)
        gr.replay()
    torch.cuda.synchronize()
    assert torch.equal(dx0, dx1) and torch.equal(dx0, dxg)
    assert torch.equal(after, dT1)
    rdx, rdT = oracle.backward(widen(d["x"]), widen(d["T"]), widen(d["dy"]), case.w, case.shift, case.layout)
    for got in (dT0, dT1, dTg):
        if case.dtype == "f32":
            assert dT_err_over_tol(got, rdT, case, 1e-4) <= 1.0
        else:
            assert max_err_over_tol(got, rdT, TOL[case.dtype]) <= 1.0
    assert max_err_over_tol(dx1, rdx, TOL[case.dtype]) <= 1.0


@pytest.mark.parametrize("case", [
    si.Case("f32_nhwc_w14", 6, 12, 56, 56, 14, dtype="f32", layout=NHWC, seed=150, backward=True),
    si.Case("f32_nhwc_w14_shift_ragged", 5, 8, 30, 44, 14, dtype="f32", layout=NHWC, shift=(7, 5), seed=151, backward=True),
    si.Case("f32_nhwc_w7", 9, 20, 28, 56, 7, dtype="f32", layout=NHWC, seed=152, backward=True),
], ids=lambda c: c.name)
def test_fp32_nhwc_through_the_transposition_route(wb, oracle, case):
    """fp32 NHWC: 32-bit transposition passes around the fp32 tensor-core kernels (forward, dX, dT); with
    WBMM_FLAG_NO_SCRATCH the FFMA kernels serve it.  Forward held to 1e-6 (the split is exact), dT to the sqrt(L*N) bound."""
    d = si.make(case, device="cuda")
    y = wb.wbmm_forward(d["x"], d["T"], case.w, case.shift, case.layout)
    assert wb.wbmm_last_path() == wb.PATH_TC_TRANSPOSED, wb.wbmm_path_string(wb.wbmm_last_path())
    dx, dT = wb.wbmm_backward(d["x"], d["T"], d["dy"], case.w, case.shift, case.layout)
    assert wb.wbmm_last_path() == wb.PATH_TC_TRANSPOSED
    y_simt = wb.wbmm_forward(d["x"], d["T"], case.w, case.shift, case.layout, wb.FLAG_NO_SCRATCH)
    assert wb.wbmm_last_path() == wb.PATH_SIMT
    torch.cuda.synchronize()
    ry = oracle.forward(widen(d["x"]), widen(d["T"]), case.w, case.shift, case.layout)
    rdx, rdT = oracle.backward(widen(d["x"]), widen(d["T"]), widen(d["dy"]), case.w, case.shift, case.layout)
    assert max_err_over_tol(y, ry, 1e-6) <= 1.0 and max_err_over_tol(dx, rdx, 1e-6) <= 1.0
    assert max_err_over_tol(y_simt, ry, 1e-4) <= 1.0
    assert dT_err_over_tol(dT, rdT, case, 1e-4) <= 1.0


@pytest.mark.parametrize("B,C,dtype", [(16, 8, "bf16"), (128, 40, "bf16"), (72, 24, "f16")])
def test_one_window_7x7_planes_on_the_pipelined_kernel(wb, oracle, B, C, dtype):
    """7 x 7 maps at w = 7 (the S4 stage): the window is the plane, 49 contiguous elements that start
    on odd elements for every other (image, channel) -- plane boxes + one funnel shift by the plane's parity
    (window_to_tmem_flat7), 2-byte stores.  One-hot tables (pure data movement: bitwise), then a dense table;
    forward and dX; canaries around the output."""
    case = si.Case("flat7", B, C, 7, 7, 7, dtype=dtype, seed=130 + C, backward=True)
    d = si.make(case, device="cuda")
    g = torch.Generator().manual_seed(C)
    bins = torch.randint(0, 169, (C,), generator=g)
    bins[0], bins[1], bins[2] = 0, 168, 84
    T1 = torch.zeros_like(d["T"])
    T1[torch.arange(C), bins.to(T1.device)] = 1.0
    n = d["x"].numel()
    buf = torch.full((n + 64,), 7.0, dtype=d["x"].dtype, device="cuda")
    y = buf[32:32 + n].view_as(d["x"])
    wb.wbmm_forward(d["x"], T1, 7, out=y)
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA, wb.wbmm_path_string(wb.wbmm_last_path())
    torch.cuda.synchronize()
    assert bool((buf[:32] == 7.0).all()) and bool((buf[32 + n:] == 7.0).all())
    assert np.array_equal(widen(y), oracle.forward(widen(d["x"]), widen(T1), 7))
    dx, _ = wb.wbmm_backward(None, T1, d["dy"], 7, need_dT=False)
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA
    rdx, _ = oracle.backward(widen(d["dy"]), widen(T1), widen(d["dy"]), 7, need_dT=False)
    assert np.array_equal(widen(dx), rdx)
    y2 = wb.wbmm_forward(d["x"], d["T"], 7)
    dx2, dT2 = wb.wbmm_backward(d["x"], d["T"], d["dy"], 7)
    ry = oracle.forward(widen(d["x"]), widen(d["T"]), 7)
    rdx2, rdT = oracle.backward(widen(d["x"]), widen(d["T"]), widen(d["dy"]), 7)
    tol = TOL[dtype]
    errs = (max_err_over_tol(y2, ry, tol), max_err_over_tol(dx2, rdx2, tol), max_err_over_tol(dT2, rdT, tol))
    assert max(errs) <= 1.0, errs


@pytest.mark.parametrize("H,W,shift", [(112, 112, (7, 7)), (112, 112, (3, 8)), (106, 112, (0, 0))])
def test_table_gradient_of_large_shifted_maps_stays_on_the_tensor_cores(wb, oracle, H, W, shift):
    """Shifted / ragged 112-row maps need whole frame images (general addressing): the dT kernel then takes one
    image per tile (half the MMA K is zero windows) instead of falling back to SIMT."""
    case = si.Case("dt_big_shift", 5, 4, H, W, 14, shift=shift, seed=72, backward=True)
    d = si.make(case, device="cuda")
    _, dT = wb.wbmm_backward(d["x"], None, d["dy"], 14, shift, need_dx=False)
    torch.cuda.synchronize()
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA, wb.wbmm_path_string(wb.wbmm_last_path())
    _, rdT = oracle.backward(widen(d["x"]), widen(d["T"]), widen(d["dy"]), 14, shift, need_dx=False)
    assert max_err_over_tol(dT, rdT, TOL["bf16"]) <= 1.0


@pytest.mark.parametrize("B,C,H,W", [(5, 6, 112, 112), (9, 3, 112, 56), (3, 4, 112, 224), (2, 3, 224, 224)])
def test_table_gradient_of_large_maps_stays_on_the_tensor_cores(wb, oracle, B, C, H, W):
    """112-row maps at w = 14: whole frame images (25 KB) of x and dy do not fit beside the operand stage, so
    the dT kernel tiles them in strips of window rows (more images per tile); it must not fall back to SIMT."""
    case = si.Case("dt_big", B, C, H, W, 14, seed=71, backward=True)
    d = si.make(case, device="cuda")
    _, dT = wb.wbmm_backward(d["x"], None, d["dy"], 14, need_dx=False)
    torch.cuda.synchronize()
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA, wb.wbmm_path_string(wb.wbmm_last_path())
    _, rdT = oracle.backward(widen(d["x"]), widen(d["T"]), widen(d["dy"]), 14, need_dx=False)
    assert max_err_over_tol(dT, rdT, TOL["bf16"]) <= 1.0


@pytest.mark.parametrize("case", [
    si.Case("pb_14_w7", 16, 6, 14, 14, 7, seed=91, backward=True),                   # 392-byte planes, 4 windows per image
    si.Case("pb_14_w7_shift", 24, 6, 14, 14, 7, shift=(3, 0), seed=92, backward=True),
    si.Case("pb_14_w14", 72, 4, 14, 14, 14, seed=93, backward=True),                 # one window per image
    si.Case("pb_14_w14_shift", 16, 6, 14, 14, 14, shift=(7, 4), seed=94, backward=True),
    si.Case("pb_14_f16", 8, 10, 14, 14, 14, dtype="f16", seed=95, backward=True),
    si.Case("pb_7x28_w7", 16, 4, 7, 28, 7, seed=96, backward=True),                  # 392-byte planes again, 1 x 4 windows
    # planes of more than 256 elements: the row of an image is viewed as (8, C*H*W/8) and the box is {8, plane/8}
    si.Case("pb2_30_w14", 24, 16, 30, 30, 14, seed=101, backward=True),              # ragged (42 x 42 padded), 12 images per tile
    si.Case("pb2_30_w14_shift", 16, 24, 30, 30, 14, shift=(7, 3), seed=102, backward=True),
    si.Case("pb2_30_w7", 12, 8, 30, 30, 7, seed=103, backward=True),                 # 25 windows per image: 4 images per tile
    si.Case("pb2_18_w7", 40, 8, 18, 18, 7, seed=104, backward=True),
    si.Case("pb2_22x38_w14_f16", 20, 12, 22, 38, 14, dtype="f16", seed=105, backward=True),
    si.Case("pb2_42_w14_many", 36, 40, 42, 42, 14, seed=106, backward=True),         # 3528-byte planes, several tiles per CTA
], ids=lambda c: c.name)
def test_planes_that_are_not_multiples_of_16_bytes(wb, oracle, case):
    """14 x 14 and 7 x 7 maps: neither a bulk copy nor a tensor map with a channel dimension can address one plane;
    the pipelined kernels load them as boxes of a map over [B][C*H*W] and store them with 8-byte stores."""
    d = si.make(case, device="cuda")
    y = wb.wbmm_forward(d["x"], d["T"], case.w, case.shift)
    torch.cuda.synchronize()
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA, wb.wbmm_path_string(wb.wbmm_last_path())
    dx, dT = wb.wbmm_backward(d["x"], d["T"], d["dy"], case.w, case.shift)
    torch.cuda.synchronize()
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA, wb.wbmm_path_string(wb.wbmm_last_path())
    ry = oracle.forward(widen(d["x"]), widen(d["T"]), case.w, case.shift)
    rdx, rdT = oracle.backward(widen(d["x"]), widen(d["T"]), widen(d["dy"]), case.w, case.shift)
    tol = TOL[case.dtype]
    errs = (max_err_over_tol(y, ry, tol), max_err_over_tol(dx, rdx, tol), max_err_over_tol(dT, rdT, tol))
    assert max(errs) <= 1.0, errs


@pytest.mark.parametrize("case", [
    si.Case("pb_7x14_w7", 16, 8, 7, 14, 7, seed=97, backward=True),                  # 196-byte planes: 4-byte store units
    si.Case("pb_7x14_w7_many", 66, 24, 7, 14, 7, seed=98, backward=True),
    si.Case("pb_14_w14_many", 130, 40, 14, 14, 14, seed=99, backward=True),          # ragged last tile, several tiles per CTA
], ids=lambda c: c.name)
def test_plane_box_store_units(wb, oracle, case):
    """Planes of 196 bytes (H*W = 98: a multiple of 2 but not of 4) are stored in 4-byte units, 392-byte planes in
    8-byte units, both by the flat (plane, chunk) walk of the store warp; canaries around the output."""
    d = si.make(case, device="cuda")
    n = d["x"].numel()
    buf = torch.full((n + 64,), 7.0, dtype=d["x"].dtype, device="cuda")
    y = buf[32:32 + n].view_as(d["x"])
    wb.wbmm_forward(d["x"], d["T"], case.w, case.shift, out=y)
    dx, _ = wb.wbmm_backward(None, d["T"], d["dy"], case.w, case.shift, need_dT=False)
    torch.cuda.synchronize()
    assert bool((buf[:32] == 7.0).all()) and bool((buf[32 + n:] == 7.0).all())
    ry = oracle.forward(widen(d["x"]), widen(d["T"]), case.w, case.shift)
    rdx, _ = oracle.backward(widen(d["x"]), widen(d["T"]), widen(d["dy"]), case.w, case.shift, need_dT=False)
    tol = TOL[case.dtype]
    assert max_err_over_tol(y, ry, tol) <= 1.0 and max_err_over_tol(dx, rdx, tol) <= 1.0


# ------------------------------------------------------------------ hierarchical reparameterisation (NEXT-1)
def _hier_case(case):
    d = si.make(case, device="cuda")
    g = torch.Generator().manual_seed(case.seed + 7)
    Tl = (torch.randn((case.C, (case.w - 1) ** 2), generator=g) * 0.02).to(d["T"].dtype).cuda()
    return d, Tl


@pytest.mark.parametrize("case", [
    si.Case("h_plain", 19, 5, 56, 56, 14, seed=41),
    si.Case("h_many", 40, 150, 28, 28, 14, seed=42),
    si.Case("h_shift", 9, 7, 28, 56, 14, shift=(7, 3), seed=43),
    si.Case("h_ragged", 7, 6, 60, 60, 14, seed=44),
    si.Case("h_strips", 2, 3, 224, 224, 14, seed=45),
    si.Case("h_f16", 10, 9, 42, 56, 14, dtype="f16", shift=(0, 7), seed=46),
    si.Case("h_nhwc_shift", 6, 16, 28, 56, 14, shift=(7, 3), layout=NHWC, seed=58),      # transposition route around the same kernel
    si.Case("h_nhwc_ragged", 5, 24, 60, 60, 14, layout=NHWC, seed=59),
], ids=lambda c: c.name)
@pytest.mark.parametrize("transpose", [False, True])
def test_hier_forward_matches_oracle(wb, oracle, case, transpose):
    """Fused hierarchical operator (Alg. 3) on the GPU against the oracle's TRAINING form (Alg. 2)."""
    d, Tl = _hier_case(case)
    y = wb.wbmm_hier_forward(d["x"], d["T"], Tl, case.w, case.shift, case.layout, transpose)
    torch.cuda.synchronize()
    assert wb.wbmm_last_path() == (wb.PATH_TC_TRANSPOSED if case.layout == NHWC else wb.PATH_TC_TMA)
    ref = oracle.hier_forward(widen(d["x"]), widen(d["T"]), widen(Tl), case.w, case.shift, case.layout, "train", transpose)
    # |y| is ~2|x| here (two identity shortcuts): same bound form, |ref| carries the scale
    assert max_err_over_tol(y, ref, TOL[case.dtype]) <= 1.0


def test_hier_zero_tables_is_exactly_two_x(wb):
    """Both tables zero => y = 2x bitwise: pins the identity blocks (14 extra N=16 MMAs) alone."""
    case = si.Case("h_2x", 9, 6, 56, 56, 14, seed=47)
    d, Tl = _hier_case(case)
    y = wb.wbmm_hier_forward(d["x"], torch.zeros_like(d["T"]), torch.zeros_like(Tl), 14)
    assert torch.equal(y, (2 * d["x"].float()).to(d["x"].dtype))


@pytest.mark.parametrize("which", ["global", "local"])
def test_hier_one_hot_tables_bitwise(wb, oracle, which):
    """One-hot global table (local zero) and one-hot local table (global zero): y - 2x is a pure shift
    inside the window / inside the 7 x 7 sub-window; small-integer x keeps every sum exact in bf16, so
    the GPU result must equal the oracle bitwise.  Pins which library (global / global+local) serves
    which (row-half, K-step) pair and the sub-window masks."""
    C = 96
    case = si.Case("h_onehot", 5, C, 28, 56, 14, seed=48)
    gen = torch.Generator().manual_seed(49)
    x = torch.randint(-3, 4, (case.B, C, case.H, case.W), generator=gen).to(torch.bfloat16).cuda()
    Tg = torch.zeros((C, 729), dtype=torch.bfloat16, device="cuda")
    Tl = torch.zeros((C, 169), dtype=torch.bfloat16, device="cuda")
    if which == "global":
        bins = torch.randint(0, 729, (C,), generator=gen)
        Tg[torch.arange(C), bins.cuda()] = 1.0
    else:
        bins = torch.randint(0, 169, (C,), generator=gen)
        bins[:4] = torch.tensor([0, 168, 84, 12])
        Tl[torch.arange(C), bins.cuda()] = 1.0
    for transpose in (False, True):
        y = wb.wbmm_hier_forward(x, Tg, Tl, 14, transpose=transpose)
        ref = oracle.hier_forward(widen(x), widen(Tg), widen(Tl), 14, form="fused", transpose=transpose)
        assert np.array_equal(widen(y), ref)


@pytest.mark.parametrize("case", [
    si.Case("hb_plain", 19, 5, 56, 56, 14, seed=51, backward=True),
    si.Case("hb_many", 40, 150, 28, 28, 14, seed=52, backward=True),          # box mode, several segments per CTA
    si.Case("hb_shift", 9, 7, 28, 56, 14, shift=(7, 3), seed=53, backward=True),
    si.Case("hb_ragged_shift", 7, 6, 60, 60, 14, shift=(5, 9), seed=54, backward=True),
    si.Case("hb_f16", 10, 9, 42, 56, 14, dtype="f16", shift=(0, 7), seed=56, backward=True),
    si.Case("hb_nhwc_shift", 6, 16, 28, 56, 14, shift=(7, 3), layout=NHWC, seed=60, backward=True),
], ids=lambda c: c.name)
def test_hier_backward_matches_oracle(wb, oracle, case):
    """dx, dTg, dTl of the hierarchical operator: one transposed fused forward and ONE pass of the
    table-gradient kernel that folds S onto both sets of bins."""
    d, Tl = _hier_case(case)
    dx, dTg, dTl = wb.wbmm_hier_backward(d["x"], d["T"], Tl, d["dy"], case.w, case.shift, case.layout)
    torch.cuda.synchronize()
    assert wb.wbmm_last_path() == (wb.PATH_TC_TRANSPOSED if case.layout == NHWC else wb.PATH_TC_TMA)
    rdx, rg, rl = oracle.hier_backward(widen(d["x"]), widen(d["T"]), widen(Tl), widen(d["dy"]), case.w, case.shift, case.layout)
    tol = TOL[case.dtype]
    errs = (max_err_over_tol(dx, rdx, tol), max_err_over_tol(dTg, rg, tol), max_err_over_tol(dTl, rl, tol))
    assert max(errs) <= 1.0, errs
    # the global table gradient is the single-scale one: same kernel, same bins
    _, dT = wb.wbmm_backward(d["x"], None, d["dy"], case.w, case.shift, case.layout, need_dx=False)
    assert max_err_over_tol(dTg, widen(dT), 1e-5) <= 1.0
    # accumulate flag: a second call doubles both
    wb.wbmm_hier_backward(d["x"], None, None, d["dy"], case.w, case.shift, case.layout, wb.FLAG_ACCUMULATE_DT,
                          need_dx=False, dTg=dTg, dTl=dTl)
    assert max_err_over_tol(dTg, 2 * rg, tol) <= 1.0 and max_err_over_tol(dTl, 2 * rl, tol) <= 1.0


def test_hier_backward_local_bins_exact_on_integers(wb, oracle):
    """Small-integer x and dy: every product and partial sum is an exact fp32 integer, so both table
    gradients must equal the oracle exactly -- pins the sub-window predicate of the second fold."""
    C = 20
    gen = torch.Generator().manual_seed(57)
    x = torch.randint(-2, 3, (8, C, 28, 28), generator=gen).to(torch.bfloat16).cuda()
    dy = torch.randint(-2, 3, (8, C, 28, 28), generator=gen).to(torch.bfloat16).cuda()
    _, dTg, dTl = wb.wbmm_hier_backward(x, None, None, dy, 14, (3, 8), need_dx=False)
    z = np.zeros((C, 729)), np.zeros((C, 169))
    _, rg, rl = oracle.hier_backward(widen(x), z[0], z[1], widen(dy), 14, (3, 8))
    assert np.array_equal(widen(dTg), rg) and np.array_equal(widen(dTl), rl)


# ------------------------------------------------------------------ cached-M mode and multi-kernel fusion (NEXT-2)
@pytest.mark.parametrize("case", [
    si.Case("m_w14", 6, 5, 56, 56, 14, seed=61),
    si.Case("m_w7_shift", 9, 7, 28, 42, 7, shift=(3, 4), seed=62),
    si.Case("m_ragged_nhwc", 3, 8, 30, 45, 14, shift=(7, 2), layout=NHWC, seed=63),
    si.Case("m_f16", 4, 3, 21, 21, 7, dtype="f16", seed=64),
    si.Case("m_w7_many", 70, 40, 56, 56, 7, seed=68),                    # pipelined kernel, several channels per CTA
    si.Case("m_w14_many", 37, 40, 56, 56, 14, seed=72),                  # w = 14: the 100 KB matrix beside the ring, channel changes
    si.Case("m_w14_boxes_shift", 40, 24, 28, 28, 14, shift=(7, 5), seed=73),
    si.Case("m_w14_f16_ragged", 6, 5, 60, 60, 14, dtype="f16", seed=74),
    si.Case("m_w7_strips_shift", 3, 4, 112, 112, 7, shift=(2, 5), seed=69),
], ids=lambda c: c.name)
def test_cached_matrix_mode_equals_the_table_mode(wb, oracle, case):
    """WBMM-C and WBMM-NC "produce identical outputs": forward and dX through
    wbmm_forward_matrix with M = materialize(T) against the oracle, and against the table path of the
    library (another kernel, so another fp32 summation order: equal to within one 16-bit ulp)."""
    d = si.make(case, device="cuda")
    M = wb.wbmm_materialize_weight(d["T"], case.w)
    for transpose in (False, True):
        y = wb.wbmm_forward_matrix(d["x"], M, case.w, case.shift, case.layout, transpose=transpose)
        # NCHW planes the pipelined kernel takes: the given matrix replaces the W_c (w = 7) / the Toeplitz library (w = 14)
        pipelined = case.layout == NCHW and case.W % 2 == 0
        assert wb.wbmm_last_path() == (wb.PATH_TC_TMA if pipelined else wb.PATH_TC_GATHER)
        if transpose:
            ref, _ = wb.wbmm_backward(None, d["T"], d["x"], case.w, case.shift, case.layout, need_dT=False)
            rdx, _ = oracle.backward(widen(d["x"]), widen(d["T"]), widen(d["x"]), case.w, case.shift, case.layout, need_dT=False)
            assert max_err_over_tol(y, rdx, TOL[case.dtype]) <= 1.0
        else:
            ref = wb.wbmm_forward(d["x"], d["T"], case.w, case.shift, case.layout)
            ry = oracle.forward(widen(d["x"]), widen(d["T"]), case.w, case.shift, case.layout)
            assert max_err_over_tol(y, ry, TOL[case.dtype]) <= 1.0
        ulp = 2.0 ** -7 if case.dtype == "bf16" else 2.0 ** -10
        diff = (y.float() - ref.float()).abs()
        assert bool((diff <= ulp * ref.float().abs() + 1e-6).all())


@pytest.mark.parametrize("case", [
    si.Case("m_any", 5, 6, 30, 44, 14, shift=(2, 9), seed=65),
    si.Case("m_any_w14_plain", 21, 10, 56, 56, 14, seed=75),             # pipelined kernel: bias at K index (row 0, column 14)
    si.Case("m_any_w7", 37, 12, 28, 56, 7, seed=70),                     # pipelined kernel: bias row at K index N + 1
    si.Case("m_any_w7_ragged_shift", 9, 5, 30, 44, 7, shift=(2, 5), seed=71),
], ids=lambda c: c.name)
def test_cached_matrix_mode_arbitrary_matrix_and_bias(wb, oracle, case):
    """A matrix that is NOT table-generated, plus a bias, against the oracle's Algorithm 1."""
    d = si.make(case, device="cuda")
    g = torch.Generator().manual_seed(66)
    N = case.w * case.w
    M = (torch.randn((case.C, N, N), generator=g) * 0.05).to(torch.bfloat16).cuda()
    bias = torch.randn((case.C,), generator=g).to(torch.bfloat16).cuda()
    for transpose in (False, True):
        y = wb.wbmm_forward_matrix(d["x"], M, case.w, case.shift, case.layout, bias, transpose)
        ref = oracle.apply_matrix(widen(d["x"]), widen(M), case.w, case.shift, case.layout, transpose, widen(bias))
        assert max_err_over_tol(y, ref, TOL["bf16"]) <= 1.0


@pytest.mark.parametrize("B", [33, 64])                  # 64: whole plane boxes -- the pipelined kernel in its flat 7 x 7 form
@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_multi_kernel_fusion_on_a_one_window_map(wb, oracle, dtype, B):
    """Section 3.7 on a 7 x 7 map: Y = WBMM(X) + BN1(DW5(X)) + BN2(DW3(X)) as ONE operator -- tables folded on
    the device (wbmm_fold_dwconv), then the cached-M forward with the BatchNorm shifts as bias (16-bit) or the
    table forward (fp32, bias added by the caller).  Reference: the oracle's fold + Algorithm 1, itself pinned
    against a library conv2d."""
    w, C = 7, 24
    td = {"bf16": torch.bfloat16, "f32": torch.float32}[dtype]
    g = torch.Generator().manual_seed(67)
    x = torch.randn((B, C, w, w), generator=g).to(td).cuda()
    T = (torch.randn((C, 169), generator=g) * 0.02).to(td).cuda()
    K5 = (torch.randn((C, 5, 5), generator=g) * 0.2).to(td).cuda()
    K3 = (torch.randn((C, 3, 3), generator=g) * 0.3).to(td).cuda()
    s1, s2 = torch.rand((C,), generator=g).cuda() + 0.5, torch.rand((C,), generator=g).cuda() + 0.5
    bias = torch.randn((C,), generator=g).to(td).cuda()
    Tf = wb.wbmm_fold_dwconv(wb.wbmm_fold_dwconv(T, K5, w, s1), K3, w, s2)
    rTf = oracle.fold_dwconv(oracle.fold_dwconv(widen(T), widen(K5), w, widen(s1)), widen(K3), w, widen(s2))
    tol = TOL[dtype]
    assert max_err_over_tol(Tf, rTf, tol) <= 1.0
    # entries the conv kernels do not touch are copied bit for bit
    far = torch.ones(169, dtype=torch.bool)
    for i in range(-2, 3):
        for j in range(-2, 3):
            far[(6 - i) * 13 + (6 - j)] = False
    assert torch.equal(Tf[:, far], T[:, far])
    if dtype == "bf16":
        y = wb.wbmm_forward_matrix(x, wb.wbmm_materialize_weight(Tf, w), w, bias=bias)
        assert wb.wbmm_last_path() == (wb.PATH_TC_TMA if B % 8 == 0 else wb.PATH_TC_GATHER)
    else:
        y = wb.wbmm_forward(x, Tf, w) + bias.view(1, C, 1, 1)
    ref = oracle.apply_matrix(widen(x), oracle.weight_matrix(widen(Tf), w), w, bias=widen(bias))
    assert max_err_over_tol(y, ref, tol) <= 1.0


# ------------------------------------------------------------------ fused bias / identity shortcut (NEXT-3)
@pytest.mark.parametrize("case,identity", [
    (si.Case("f_w14", 19, 5, 56, 56, 14, seed=81), 1.0),
    (si.Case("f_w14_box", 40, 150, 28, 28, 14, seed=82), 0.0),
    (si.Case("f_w14_shift", 9, 7, 28, 56, 14, shift=(7, 3), seed=83), 2.0),
    (si.Case("f_w14_ragged", 7, 6, 60, 60, 14, shift=(5, 8), seed=84), 0.5),
    (si.Case("f_w14_f16_nhwc", 6, 8, 42, 56, 14, dtype="f16", layout=NHWC, seed=85), 1.0),
    (si.Case("f_w7", 21, 6, 56, 56, 7, seed=86), 0.0),
    (si.Case("f_w7_shift", 5, 7, 28, 28, 7, shift=(3, 2), seed=87), 0.0),
], ids=lambda v: v.name if hasattr(v, "name") else str(v))
def test_fused_bias_and_identity(wb, oracle, case, identity):
    """y = W_c x + identity x + bias_c in the pipelined kernel (bias as one more K index, identity as the
    identity block of the library) against the oracle's Algorithm 1 with M = R[:, I] + identity I and a bias;
    transposed application without the bias."""
    d = si.make(case, device="cuda")
    td = d["x"].dtype
    bias = torch.randn((case.C,), generator=torch.Generator().manual_seed(case.seed)).to(td).cuda()
    M = oracle.weight_matrix(widen(d["T"]), case.w) + identity * np.eye(case.w ** 2)[None]
    y = wb.wbmm_forward_fused(d["x"], d["T"], case.w, case.shift, case.layout, bias, identity)
    assert wb.wbmm_last_path() == (wb.PATH_TC_TMA if case.layout == NCHW else wb.PATH_TC_TRANSPOSED)
    ref = oracle.apply_matrix(widen(d["x"]), M, case.w, case.shift, case.layout, bias=widen(bias))
    assert max_err_over_tol(y, ref, TOL[case.dtype]) <= 1.0
    dx = wb.wbmm_forward_fused(d["x"], d["T"], case.w, case.shift, case.layout, None, identity, transpose=True)
    rdx = oracle.apply_matrix(widen(d["x"]), M, case.w, case.shift, case.layout, transpose=True)
    assert max_err_over_tol(dx, rdx, TOL[case.dtype]) <= 1.0


def test_fused_bias_exact_with_zero_table(wb):
    """Zero table: y = identity * x + bias_c must be exact (one rounding of an fp32 sum of two 16-bit values)
    -- pins that the bias is added exactly once and to every output position, the identity to its own."""
    case = si.Case("f_exact", 9, 12, 28, 56, 14, shift=(7, 7), seed=88)
    d = si.make(case, device="cuda")
    bias = torch.randn((case.C,), generator=torch.Generator().manual_seed(89)).to(torch.bfloat16).cuda()
    y = wb.wbmm_forward_fused(d["x"], torch.zeros_like(d["T"]), 14, case.shift, bias=bias, identity=1.0)
    ref = (d["x"].float() + bias.float().view(1, -1, 1, 1)).to(torch.bfloat16)
    assert torch.equal(y, ref)
    y7 = wb.wbmm_forward_fused(d["x"], torch.zeros((case.C, 169), dtype=torch.bfloat16, device="cuda"), 7, bias=bias)
    assert torch.equal(y7, bias.view(1, -1, 1, 1).expand_as(d["x"]).contiguous())


@pytest.mark.parametrize("case,identity", [
    (si.Case("ff_f32_w14", 5, 6, 56, 56, 14, dtype="f32", seed=170), 1.0),                      # float32: no pipelined fused kernel
    (si.Case("ff_f32_w7_shift", 7, 5, 28, 42, 7, dtype="f32", shift=(3, 2), seed=171), 2.0),
    (si.Case("ff_bf16_w7_identity", 9, 6, 28, 28, 7, seed=172), 1.0),                           # identity at w = 7
    (si.Case("ff_f16_w5_nhwc", 4, 8, 22, 31, 5, dtype="f16", layout=NHWC, shift=(1, 4), seed=173), 0.5),
], ids=lambda v: v.name if hasattr(v, "name") else str(v))
def test_fused_and_cached_matrix_on_the_ffma_kernels(wb, oracle, case, identity):
    """wbmm_forward_fused and wbmm_forward_matrix where no tensor-core kernel applies (float32, identity at w != 14, other
    window sizes): FFMA kernels (csrc/wbmm_rect.cu) against the oracle's Algorithm 1 with M = R[:, I] + identity I and a
    bias; then the same matrix GIVEN (cached-M mode), forward and transposed."""
    d = si.make(case, device="cuda")
    td = d["x"].dtype
    g = torch.Generator().manual_seed(case.seed)
    bias = torch.randn((case.C,), generator=g).to(td).cuda()
    N = case.w * case.w
    Mref = oracle.weight_matrix(widen(d["T"]), case.w) + float(torch.tensor(identity).to(td)) * np.eye(N)[None]
    tol = TOL[case.dtype]
    y = wb.wbmm_forward_fused(d["x"], d["T"], case.w, case.shift, case.layout, bias=bias, identity=identity)
    assert wb.wbmm_last_path() == wb.PATH_SIMT
    ref = oracle.apply_matrix(widen(d["x"]), Mref, case.w, case.shift, case.layout, False, widen(bias))
    assert max_err_over_tol(y, ref, tol) <= 1.0
    yt = wb.wbmm_forward_fused(d["x"], d["T"], case.w, case.shift, case.layout, identity=identity, transpose=True)
    reft = oracle.apply_matrix(widen(d["x"]), Mref, case.w, case.shift, case.layout, True)
    assert max_err_over_tol(yt, reft, tol) <= 1.0
    if case.dtype == "f32" or case.w not in (7, 14):
        gm = torch.Generator().manual_seed(case.seed + 1)
        M = (torch.randn((case.C, N, N), generator=gm) * 0.05).to(td).cuda()
        for transpose in (False, True):
            ym = wb.wbmm_forward_matrix(d["x"], M, case.w, case.shift, case.layout, bias, transpose)
            assert wb.wbmm_last_path() == wb.PATH_SIMT
            refm = oracle.apply_matrix(widen(d["x"]), widen(M), case.w, case.shift, case.layout, transpose, widen(bias))
            assert max_err_over_tol(ym, refm, tol) <= 1.0


@pytest.mark.parametrize("case,flags", [
    (si.Case("hf_f32", 5, 6, 56, 56, 14, dtype="f32", seed=160, backward=True), 0),                      # the paper's precision
    (si.Case("hf_f32_shift_ragged", 3, 4, 30, 44, 14, dtype="f32", shift=(9, 4), seed=161, backward=True), 0),
    (si.Case("hf_f32_nhwc", 4, 5, 28, 42, 14, dtype="f32", layout=NHWC, shift=(7, 7), seed=162, backward=True), 0),
    (si.Case("hf_bf16_forced", 6, 7, 28, 56, 14, shift=(7, 3), seed=163, backward=True), 2),             # WBMM_FLAG_FORCE_SIMT
    (si.Case("hf_w8", 4, 3, 20, 24, 8, dtype="f32", shift=(5, 2), seed=164, backward=True), 0),          # w = 8: 4 x 4 sub-windows
], ids=lambda v: v.name if hasattr(v, "name") else str(v))
def test_hier_ffma_fallback_matches_oracle(wb, oracle, case, flags):
    """The hierarchical operator where the tensor-core kernel does not apply (fp32, w != 14, forced): FFMA kernels
    (csrc/wbmm_rect.cu) against the oracle's TRAINING form (Alg. 2) and its table gradients."""
    d, Tl = _hier_case(case)
    tol = TOL[case.dtype]
    for transpose in (False, True):
        y = wb.wbmm_hier_forward(d["x"], d["T"], Tl, case.w, case.shift, case.layout, transpose, flags=flags)
        torch.cuda.synchronize()
        assert wb.wbmm_last_path() == wb.PATH_SIMT
        ref = oracle.hier_forward(widen(d["x"]), widen(d["T"]), widen(Tl), case.w, case.shift, case.layout, "train", transpose)
        assert max_err_over_tol(y, ref, tol) <= 1.0
    dx, dTg, dTl = wb.wbmm_hier_backward(d["x"], d["T"], Tl, d["dy"], case.w, case.shift, case.layout, flags)
    torch.cuda.synchronize()
    assert wb.wbmm_last_path() == wb.PATH_SIMT
    rdx, rg, rl = oracle.hier_backward(widen(d["x"]), widen(d["T"]), widen(Tl), widen(d["dy"]), case.w, case.shift, case.layout)
    assert max_err_over_tol(dx, rdx, tol) <= 1.0
    if case.dtype == "f32":
        assert dT_err_over_tol(dTg, rg, case, 1e-4) <= 1.0 and dT_err_over_tol(dTl, rl, case, 1e-4) <= 1.0
    else:
        assert max_err_over_tol(dTg, rg, tol) <= 1.0 and max_err_over_tol(dTl, rl, tol) <= 1.0


def test_hier_unsupported_shapes_fail_loudly(wb):
    x = torch.zeros((2, 4, 14, 14), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(wb.WbmmError):       # w = 7 has no hierarchical tensor-core path
        wb.wbmm_hier_forward(x, torch.zeros((4, 169), dtype=torch.bfloat16, device="cuda"),
                             torch.zeros((4, 36), dtype=torch.bfloat16, device="cuda"), 7)


# ------------------------------------------------------------------ NHWC in one pass (w = 7)
NHWC7 = [
    si.Case("n7_oct4_56", 21, 32, 56, 56, 7, layout=NHWC, seed=501),                # 32-channel groups, strips of 3 window rows
    si.Case("n7_oct4_28_many", 40, 96, 28, 28, 7, layout=NHWC, seed=502),           # 2 images per tile, 3 groups, > 148 tiles
    si.Case("n7_oct4_112", 3, 64, 112, 112, 7, layout=NHWC, seed=503),              # 16 windows per row: 2 rows per tile
    si.Case("n7_oct4_ragged", 6, 32, 30, 60, 7, layout=NHWC, seed=504),             # W' = 63, H' = 35: zero fill / clipping by the copy engine
    si.Case("n7_oct2_56", 21, 16, 56, 56, 7, layout=NHWC, seed=505),                # 16-channel groups (C = 16)
    si.Case("n7_oct2_ragged_f16", 5, 48, 26, 30, 7, layout=NHWC, dtype="f16", seed=506),
    si.Case("n7_oct1_28", 33, 8, 28, 56, 7, layout=NHWC, seed=507),                 # 8-channel groups
    si.Case("n7_oct1_c24", 5, 24, 26, 30, 7, layout=NHWC, seed=508),
    si.Case("n7_tiny_maps", 50, 32, 14, 14, 7, layout=NHWC, seed=509),              # 4 windows per image, 8 images per tile
    si.Case("n7_one_window_maps", 70, 64, 7, 7, 7, layout=NHWC, seed=510),          # the S4 stage: one window per image
]


@pytest.mark.parametrize("case", NHWC7, ids=lambda c: c.name)
def test_nhwc_one_pass_w7(wb, oracle, case):
    """NHWC forward and dX straight from NHWC memory (tensor-map boxes of 32 / 16 / 8 channels per pixel, swizzled
    frames, channel octets on the TMEM lane quarters): the path BASELINE.json north_star (a) asks for."""
    d = si.make(case, device="cuda")
    y = wb.wbmm_forward(d["x"], d["T"], case.w, case.shift, case.layout)
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA, wb.wbmm_path_string(wb.wbmm_last_path())
    dx, _ = wb.wbmm_backward(None, d["T"], d["x"], case.w, case.shift, case.layout, need_dT=False)
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA
    ry = oracle.forward(widen(d["x"]), widen(d["T"]), case.w, case.shift, case.layout)
    rdx, _ = oracle.backward(widen(d["x"]), widen(d["T"]), widen(d["x"]), case.w, case.shift, case.layout, need_dT=False)
    tol = TOL[case.dtype]
    assert max_err_over_tol(y, ry, tol) <= 1.0 and max_err_over_tol(dx, rdx, tol) <= 1.0


def test_nhwc_one_pass_w7_one_hot_bins_bitwise(wb, oracle):
    """Every one of the 169 bins as a one-hot table, one bin per channel (C = 192: six 32-channel groups), on a ragged
    map: the result must equal the oracle's bitwise -- the Toeplitz blocks, the two-rows-per-K-step operand order,
    the swizzled addressing and the channel interleave of the in-place epilogue."""
    C = 192
    case = si.Case("n7_onehot", 3, C, 30, 44, 7, layout=NHWC, seed=511)
    d = si.make(case, device="cuda")
    T = torch.zeros_like(d["T"])
    bins = torch.arange(C) % 169
    T[torch.arange(C), bins.to(T.device)] = 1.0
    y = wb.wbmm_forward(d["x"], T, 7, layout=NHWC)
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA
    assert np.array_equal(widen(y), oracle.forward(widen(d["x"]), widen(T), 7, layout=NHWC))
    dx, _ = wb.wbmm_backward(None, T, d["x"], 7, layout=NHWC, need_dT=False)
    rdx, _ = oracle.backward(widen(d["x"]), widen(T), widen(d["x"]), 7, layout=NHWC, need_dT=False)
    assert np.array_equal(widen(dx), rdx)


def test_config1_fp32_tiny(wb, oracle):
    """BASELINE.json config 1: fp32 path, <= 1e-4 -- on the tensor cores (3-way bf16 split) and on the FFMA kernel."""
    err, path = run_forward(wb, oracle, si.CFG1)
    assert err <= 1.0, err
    assert path == wb.PATH_TC_TMA
    err, path = run_forward(wb, oracle, si.CFG1, wb.FLAG_FORCE_SIMT)
    assert err <= 1.0, err
    assert path == wb.PATH_SIMT


# ------------------------------------------------------------------ fp32 on the tensor cores (NEXT-4)
F32_TC = [
    si.Case("f32_w14_plain", 19, 5, 56, 56, 14, dtype="f32", seed=201),              # 8 images per tile, tail of 3
    si.Case("f32_w14_many", 40, 150, 28, 28, 14, dtype="f32", seed=202),             # 32 images per tile, > 148 tiles
    si.Case("f32_w14_shift", 9, 7, 28, 56, 14, dtype="f32", shift=(7, 5), seed=203),
    si.Case("f32_w14_ragged", 7, 6, 60, 60, 14, dtype="f32", seed=204),              # 25 windows per image, W' = 70
    si.Case("f32_w14_ragged_shift", 6, 5, 36, 40, 14, dtype="f32", shift=(5, 9), seed=205),
    si.Case("f32_w14_two_images", 5, 4, 112, 112, 14, dtype="f32", seed=206),        # 64 windows per image
    si.Case("f32_w14_strips", 2, 3, 224, 224, 14, dtype="f32", seed=207),            # 256 windows per image: row strips
    si.Case("f32_w7_plain", 21, 6, 56, 56, 7, dtype="f32", seed=208),
    si.Case("f32_w7_shift", 5, 7, 28, 28, 7, dtype="f32", shift=(3, 2), seed=209),
    si.Case("f32_w7_ragged", 6, 4, 26, 30, 7, dtype="f32", shift=(0, 3), seed=210),
    si.Case("f32_w7_strips", 3, 5, 112, 112, 7, dtype="f32", seed=211),
    si.Case("f32_w7_tiny_maps", 70, 6, 14, 14, 7, dtype="f32", seed=212),            # 784-byte planes, 32 images per tile
]


@pytest.mark.parametrize("case", F32_TC, ids=lambda c: c.name)
def test_fp32_tensor_core_path(wb, oracle, case):
    """fp32 forward and dX through six bf16 tensor passes (exact 3-way splits of windows and table): the paper's
    precision at the 1e-4 bar of BASELINE.json -- and far inside it: dropping any of the three
    2^-16-weight cross terms would leave ~2e-6, the full expansion measures ~2.5e-7 (fp32 accumulation)."""
    d = si.make(case, device="cuda")
    y = wb.wbmm_forward(d["x"], d["T"], case.w, case.shift)
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA, wb.wbmm_path_string(wb.wbmm_last_path())
    dx, _ = wb.wbmm_backward(None, d["T"], d["x"], case.w, case.shift, need_dT=False)
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA
    ry = oracle.forward(widen(d["x"]), widen(d["T"]), case.w, case.shift)
    rdx, _ = oracle.backward(widen(d["x"]), widen(d["T"]), widen(d["x"]), case.w, case.shift, need_dT=False)
    assert max_err_over_tol(y, ry, 1e-6) <= 1.0 and max_err_over_tol(dx, rdx, 1e-6) <= 1.0


@pytest.mark.parametrize("case", [c for c in F32_TC if c.name not in ("f32_w14_strips", "f32_w7_ragged")], ids=lambda c: c.name)
def test_fp32_table_gradient_on_the_tensor_cores(wb, oracle, case):
    """fp32 dT with split operands (w = 14: two bf16 terms per value, three passes; w = 7: three terms, six passes):
    the 1e-4 * (sqrt(L*N) + |ref|) bound of the table gradient (measured: 0.08-0.14 of it at w = 14, 0.002 at w = 7),
    and EXACT on small integers, which pins tiles, slots and the bin fold of this kernel."""
    case = si.with_(case, backward=True)
    d = si.make(case, device="cuda")
    _, dT = wb.wbmm_backward(d["x"], None, d["dy"], case.w, case.shift, need_dx=False)
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA, wb.wbmm_path_string(wb.wbmm_last_path())
    _, rdT = oracle.backward(widen(d["x"]), np.zeros((case.C, case.bins)), widen(d["dy"]), case.w, case.shift, need_dx=False)
    assert dT_err_over_tol(dT, rdT, case) <= 1.0
    gen = torch.Generator().manual_seed(case.seed)
    xi = torch.randint(-2, 3, d["x"].shape, generator=gen).float().cuda()
    gi = torch.randint(-2, 3, d["x"].shape, generator=gen).float().cuda()
    _, dTi = wb.wbmm_backward(xi, None, gi, case.w, case.shift, need_dx=False)
    _, ri = oracle.backward(widen(xi), np.zeros((case.C, case.bins)), widen(gi), case.w, case.shift, need_dx=False)
    assert np.array_equal(widen(dTi), ri)
    # accumulate flag and the full backward call (dX and dT in one call)
    dx, dT2 = wb.wbmm_backward(d["x"], d["T"], d["dy"], case.w, case.shift, dT=dT.clone(), flags=wb.FLAG_ACCUMULATE_DT)
    assert dT_err_over_tol(dT2, 2 * rdT, case) <= 2.0
    rdx, _ = oracle.backward(widen(d["x"]), widen(d["T"]), widen(d["dy"]), case.w, case.shift, need_dT=False)
    assert max_err_over_tol(dx, rdx, 1e-6) <= 1.0


def test_fp32_tensor_core_path_one_hot_bins_bitwise(wb, oracle):
    """One-hot tables through the fp32 tensor-core kernel: x1 + x2 + x3 is x exactly and the only non-zero weight is
    1.0, so the result must equal the oracle's bitwise at every bin -- indexing of the three libraries, of the
    window splits and of the staged row-run stores."""
    for w, H, W, shift in ((14, 28, 56, (0, 0)), (14, 30, 44, (5, 9)), (7, 28, 28, (0, 0)), (7, 26, 30, (3, 2))):
        tw = 2 * w - 1
        nb = tw * tw
        C = 64
        case = si.Case("f32_onehot", 9, C, H, W, w, dtype="f32", shift=shift, seed=213)
        d = si.make(case, device="cuda")
        bins = torch.randint(0, nb, (C,), generator=torch.Generator().manual_seed(w * 100 + H))
        bins[0], bins[1], bins[2] = 0, nb - 1, (w - 1) * tw + (w - 1)
        T = torch.zeros_like(d["T"])
        T[torch.arange(C), bins.to(T.device)] = 1.0
        y = wb.wbmm_forward(d["x"], T, w, shift)
        assert wb.wbmm_last_path() == wb.PATH_TC_TMA
        assert np.array_equal(widen(y), oracle.forward(widen(d["x"]), widen(T), w, shift))


# ------------------------------------------------------------------ exact structured tests
@pytest.mark.parametrize("dtype", ["f32", "bf16", "f16"])
@pytest.mark.parametrize("layout", [NCHW, NHWC])
@pytest.mark.parametrize("w,shift,H,W", [(7, (0, 0), 14, 21), (14, (0, 0), 28, 56), (14, (7, 7), 28, 28),
                                         (7, (3, 3), 15, 20), (14, (5, 9), 30, 60)])
@pytest.mark.parametrize("force_simt", [True, False])
def test_delta_table_is_identity_bitwise(wb, dtype, layout, w, shift, H, W, force_simt):
    """Delta at the zero-offset bin => y == x bitwise (any dtype, any path)."""
    case = si.Case("delta", 3, 6, H, W, w, dtype=dtype, layout=layout, shift=shift, seed=21)
    d = si.make(case, device="cuda")
    T = torch.zeros_like(d["T"])
    tw = 2 * w - 1
    T[:, (w - 1) * tw + (w - 1)] = 1.0
    y = wb.wbmm_forward(d["x"], T, w, shift, layout, wb.FLAG_FORCE_SIMT if force_simt else 0)
    assert torch.equal(y, d["x"])


@pytest.mark.parametrize("w", [7, 14])
@pytest.mark.parametrize("force_simt", [True, False])
def test_one_hot_table_every_bin_bitwise(wb, oracle, w, force_simt):
    """One-hot table at every bin k: the GPU result must equal the oracle's bitwise (a pure data
    movement: y[r,c] = x[r-dr,c-dc] or 0).  Channel c carries bin (c mod nb): all (2w-1)^2 bins
    are covered by C = nb channels in one launch.  This is the bit-exact indexing test."""
    tw = 2 * w - 1
    nb = tw * tw
    case = si.Case("onehot", 2, nb, 2 * w, 4 * w, w, dtype="bf16", seed=22)
    d = si.make(case, device="cuda")
    T = torch.zeros_like(d["T"])
    T[torch.arange(nb), torch.arange(nb)] = 1.0
    y = wb.wbmm_forward(d["x"], T, w, flags=wb.FLAG_FORCE_SIMT if force_simt else 0)
    ref = oracle.forward(widen(d["x"]), widen(T), w)
    assert np.array_equal(widen(y), ref)
    dx, _ = wb.wbmm_backward(None, T, d["x"], w, need_dT=False, flags=wb.FLAG_FORCE_SIMT if force_simt else 0)
    rdx, _ = oracle.backward(widen(d["x"]), widen(T), widen(d["x"]), w, need_dT=False)
    assert np.array_equal(widen(dx), rdx)


@pytest.mark.parametrize("force_simt", [True, False])
def test_all_ones_table_window_sums_exact(wb, force_simt):
    """All-ones table => every output is its window's sum; small-integer x keeps bf16 exact.
    Pins partition + zero padding on the GPU without the oracle."""
    w, B, C, H, W = 14, 2, 3, 30, 60
    g = torch.Generator().manual_seed(5)
    x = torch.randint(-2, 3, (B, C, H, W), generator=g).to(torch.bfloat16).cuda()
    T = torch.ones((C, 27 * 27), dtype=torch.bfloat16, device="cuda")
    y = wb.wbmm_forward(x, T, w, flags=wb.FLAG_FORCE_SIMT if force_simt else 0).float().cpu()
    xp = torch.zeros(B, C, 42, 70)
    xp[:, :, :H, :W] = x.float().cpu()
    sums = xp.reshape(B, C, 3, 14, 5, 14).sum(dim=(3, 5))
    exp = sums[:, :, :, None, :, None].expand(B, C, 3, 14, 5, 14).reshape(B, C, 42, 70)[:, :, :H, :W]
    assert torch.equal(y, exp)


@pytest.mark.parametrize("dtype", ["f32", "bf16", "f16"])
@pytest.mark.parametrize("w", [3, 7, 14])
def test_materialize_weight_bitwise(wb, oracle, dtype, w):
    """a1+a2: W[c,i,j] = T[c, rel(i,j)] must equal the oracle's gather bit for bit."""
    case = si.Case("mat", 1, 5, w, w, w, dtype=dtype, seed=23)
    T = si.make(case, device="cuda")["T"]
    Wg = wb.wbmm_materialize_weight(T, w)
    assert np.array_equal(widen(Wg), oracle.weight_matrix(widen(T), w))


def test_output_is_fully_overwritten_and_nothing_else(wb):
    """y is written exactly on its B*C*H*W elements: canary-filled, over-allocated buffer."""
    case = si.Case("canary", 2, 3, 30, 25, 14, dtype="bf16", shift=(7, 3), seed=24)
    d = si.make(case, device="cuda")
    n = d["x"].numel()
    for flags in (0, wb.FLAG_FORCE_SIMT):
        buf = torch.full((n + 4096,), float("nan"), dtype=torch.bfloat16, device="cuda")
        y = buf[2048:2048 + n].view_as(d["x"])
        wb.wbmm_forward(d["x"], d["T"], 14, case.shift, out=y, flags=flags)
        assert torch.isnan(buf[:2048]).all() and torch.isnan(buf[2048 + n:]).all()
        assert not torch.isnan(y).any()


def test_empty_inputs(wb):
    for shape in ((0, 4, 14, 14), (2, 0, 14, 14)):
        x = torch.zeros(shape, dtype=torch.bfloat16, device="cuda")
        T = torch.zeros((shape[1], 169), dtype=torch.bfloat16, device="cuda")
        y = wb.wbmm_forward(x, T, 7)
        assert y.shape == x.shape
        dx, dT = wb.wbmm_backward(x, T, x, 7)
        assert dT.shape == (shape[1], 169) and torch.count_nonzero(dT) == 0


def test_dT_accumulate_flag_and_run_to_run(wb, oracle):
    case = si.Case("acc", 4, 6, 28, 28, 14, dtype="bf16", seed=25, backward=True)
    d = si.make(case, device="cuda")
    _, dT1 = wb.wbmm_backward(d["x"], d["T"], d["dy"], 14, need_dx=False)
    _, dT2 = wb.wbmm_backward(d["x"], d["T"], d["dy"], 14, need_dx=False)
    assert torch.all((dT1 - dT2).abs() <= 1e-5 * (1 + dT1.abs()))     # atomics: rounding only
    acc = dT1.clone()
    wb.wbmm_backward(d["x"], d["T"], d["dy"], 14, need_dx=False, dT=acc, flags=wb.FLAG_ACCUMULATE_DT)
    assert torch.allclose(acc, 2 * dT1, rtol=1e-5, atol=1e-5)


def test_calls_from_two_threads_on_two_streams(wb, oracle):
    """The library keeps per-process caches (tile schedules, shared-memory opt-ins, tensor-map encoder): calls from
    two host threads on two streams, different shapes interleaved, must each give their own correct result."""
    import threading
    cases = [si.Case("mt_a", 24, 12, 56, 56, 14, seed=111, backward=True),
             si.Case("mt_b", 40, 20, 28, 28, 14, shift=(7, 7), seed=112, backward=True)]
    data = [si.make(c, device="cuda") for c in cases]
    out = [None, None]

    def work(i):
        c, d = cases[i], data[i]
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            for _ in range(20):
                y = wb.wbmm_forward(d["x"], d["T"], c.w, c.shift)
                dx, dT = wb.wbmm_backward(d["x"], d["T"], d["dy"], c.w, c.shift)
        st.synchronize()
        out[i] = (y, dx, dT)

    th = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    for c, d, (y, dx, dT) in zip(cases, data, out):
        ry = oracle.forward(widen(d["x"]), widen(d["T"]), c.w, c.shift)
        rdx, rdT = oracle.backward(widen(d["x"]), widen(d["T"]), widen(d["dy"]), c.w, c.shift)
        tol = TOL[c.dtype]
        assert max(max_err_over_tol(y, ry, tol), max_err_over_tol(dx, rdx, tol), max_err_over_tol(dT, rdT, tol)) <= 1.0


def test_training_step_replays_from_a_cuda_graph(wb, oracle):
    """Forward + backward (incl. the dT zeroing kernel, the NHWC scratch allocations and their programmatic
    dependent launches) captured once and replayed: the replay must reproduce the oracle on NEW input values."""
    for layout in (NCHW, NHWC):
        case = si.Case("graph", 16, 16, 28, 56, 14, shift=(7, 7), layout=layout, seed=113, backward=True)
        d = si.make(case, device="cuda")
        x, dy = d["x"].clone(), d["dy"].clone()
        y, dx = torch.empty_like(x), None
        dT = torch.empty((case.C, case.bins), dtype=torch.float32, device="cuda")
        wb.wbmm_forward(x, d["T"], case.w, case.shift, layout, out=y)            # warm-up outside the capture
        wb.wbmm_backward(x, d["T"], dy, case.w, case.shift, layout, dT=dT)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            wb.wbmm_forward(x, d["T"], case.w, case.shift, layout, out=y)
            dx, _ = wb.wbmm_backward(x, d["T"], dy, case.w, case.shift, layout, dT=dT)
        x.copy_(torch.flip(d["x"], dims=(0,)))                                   # new values in the captured buffers
        dy.copy_(torch.flip(d["dy"], dims=(0,)))
        g.replay()
        torch.cuda.synchronize()
        ry = oracle.forward(widen(x), widen(d["T"]), case.w, case.shift, layout)
        rdx, rdT = oracle.backward(widen(x), widen(d["T"]), widen(dy), case.w, case.shift, layout)
        tol = TOL[case.dtype]
        assert max(max_err_over_tol(y, ry, tol), max_err_over_tol(dx, rdx, tol), max_err_over_tol(dT, rdT, tol)) <= 1.0


def test_host_entry_points(wb, oracle):
    case = si.Case("host", 2, 5, 28, 30, 14, dtype="bf16", shift=(7, 7), seed=26, backward=True)
    d = si.make(case)
    y = wb.wbmm_forward_host(d["x"], d["T"], 14, case.shift)
    ref = oracle.forward(widen(d["x"]), widen(d["T"]), 14, case.shift)
    assert max_err_over_tol(y, ref, 1e-2) <= 1.0
    dx, dT = wb.wbmm_backward_host(d["x"], d["T"], d["dy"], 14, case.shift)
    rdx, rdT = oracle.backward(widen(d["x"]), widen(d["T"]), widen(d["dy"]), 14, case.shift)
    assert max_err_over_tol(dx, rdx, 1e-2) <= 1.0 and max_err_over_tol(dT, rdT, 1e-2) <= 1.0


def test_non_default_stream(wb, oracle):
    case = si.Case("stream", 2, 4, 28, 28, 14, dtype="bf16", seed=27)
    d = si.make(case, device="cuda")
    s = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        y = wb.wbmm_forward(d["x"], d["T"], 14)
    s.synchronize()
    ref = oracle.forward(widen(d["x"]), widen(d["T"]), 14)
    assert max_err_over_tol(y, ref, 1e-2) <= 1.0


# ------------------------------------------------------------------ BASELINE.json configs, full size
# full-TENSOR oracle parity on configs 1, 2, 3, 5 -- every element of y, dx and dT, in the
# launch configuration bench.py times (a tile dropped by the static schedule would touch 8 planes of 12 288).
def test_config2_full_size_whole_tensor(wb, oracle):
    err, path = run_forward(wb, oracle, si.CFG2)
    assert path == wb.PATH_TC_TMA
    assert err <= 1.0, err


def test_config3_headline_full_size_whole_tensor(wb, oracle):
    err, path = run_forward(wb, oracle, si.CFG3)
    assert path == wb.PATH_TC_TMA
    assert err <= 1.0, err
    err, _ = run_forward(wb, oracle, si.with_(si.CFG3, table="structured"), sample=(8, 8))
    assert err <= 1.0, err


def test_config5_training_step_full_size_whole_tensor(wb, oracle):
    """y, dx (1e-2 form, 16-bit outputs) and dT (fp32 out: the tighter DT_TOL form) over all 192 channels."""
    case = si.CFG5
    d = si.make(case, device="cuda")
    y = wb.wbmm_forward(d["x"], d["T"], case.w, case.shift, case.layout)
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA
    dx, dT = wb.wbmm_backward(d["x"], d["T"], d["dy"], case.w, case.shift, case.layout)
    assert wb.wbmm_last_path() == wb.PATH_TC_TMA
    torch.cuda.synchronize()
    xw, Tw, gw = widen(d["x"]), widen(d["T"]), widen(d["dy"])
    ry = oracle.forward(xw, Tw, case.w, case.shift, case.layout)
    rdx, rdT = oracle.backward(xw, Tw, gw, case.w, case.shift, case.layout)
    tol = TOL[case.dtype]
    assert max_err_over_tol(y, ry, tol) <= 1.0
    assert max_err_over_tol(dx, rdx, tol) <= 1.0
    assert dT_err_over_tol(dT, rdT, case) <= 1.0


SWEEP = [c for c in si.sweep_cases()]


@pytest.mark.parametrize("case", SWEEP, ids=lambda c: c.name)
def test_config4_sweep(wb, oracle, case):
    """All 82 cases of config 4 (every B): parity on a seeded sample of full planes (sampled planes
    above ~40 M elements; whole tensor below 2 M), and the dispatch -- every NCHW shape on the pipelined
    tcgen05 + TMA kernel, every NHWC shape on a tensor-core path."""
    sample = None if case.n_elem <= 2_000_000 else (3, 4)
    err, path = run_forward(wb, oracle, case, sample=sample)
    assert path in ((wb.PATH_TC_TMA,) if case.layout == NCHW else NHWC_TC_PATHS), wb.wbmm_path_string(path)
    assert err <= 1.0, err
    if case.B == 256:
        torch.cuda.empty_cache()


SWEEP_BWD = [si.with_(c, backward=True) for c in SWEEP if c.B == 128]


@pytest.mark.parametrize("case", SWEEP_BWD, ids=lambda c: c.name)
def test_config4_sweep_backward_B128(wb, oracle, case):
    """dX and dT at B = 128 for every (C, H, w) of the sweep in both layouts: all images, a seeded sample of
    channels (dT is a sum over ALL windows of a channel, so a channel is compared whole or not at all)."""
    e_dx, e_dT = run_backward(wb, oracle, case, sample_c=4)
    assert e_dx <= 1.0 and e_dT <= 1.0, (e_dx, e_dT)
    torch.cuda.empty_cache()


# ------------------------------------------------------------------ table gradient: exact on small integers
# x, dy in {-2..2}: every product and every partial sum is an integer below 2^24, so the fp32 accumulation in
# TMEM, the per-warp bins and the atomics are all exact in any order -- dT must EQUAL the oracle.  One dropped,
# duplicated or misplaced window changes a bin by an integer.  One case per mode of the table-gradient kernels.
DT_EXACT = [
    ("aligned_w14_56", si.Case("dte", 19, 5, 56, 56, 14, seed=301)),                    # bulk copies, 8 images / tile, tail of 3
    ("boxes_w14_28", si.Case("dte", 40, 24, 28, 28, 14, seed=302)),                     # tensor-map boxes of 8 images
    ("gen_shift_w14_28", si.Case("dte", 24, 9, 28, 28, 14, shift=(7, 7), seed=303)),    # general addressing (cfg5's mode)
    ("gen_shift_odd_w14", si.Case("dte", 9, 7, 28, 56, 14, shift=(3, 5), seed=304)),
    ("gen_ragged_w14_60", si.Case("dte", 7, 6, 60, 60, 14, seed=305)),                  # 25 windows / image, padding
    ("gen_ragged_shift_w14", si.Case("dte", 6, 5, 36, 40, 14, shift=(5, 9), seed=306)),
    ("strips_w14_112", si.Case("dte", 9, 4, 112, 112, 14, seed=307)),                   # strips of window rows
    ("bigmap_w14_224", si.Case("dte", 3, 3, 224, 224, 14, seed=308)),                   # one window row of 8 images / tile
    ("one_image_w14_112_shift", si.Case("dte", 5, 3, 112, 112, 14, shift=(7, 7), seed=309)),
    ("plane_boxes_w14_14", si.Case("dte", 72, 6, 14, 14, 14, seed=310)),                # 392-byte planes
    ("plane_boxes_w7_14_shift", si.Case("dte", 24, 6, 14, 14, 7, shift=(3, 0), seed=311)),
    ("plane_boxes_2d_w14_30", si.Case("dte", 24, 8, 30, 30, 14, seed=322)),            # 1800-byte planes: (8, n) boxes, 12 images / tile
    ("plane_boxes_2d_w7_30_rowshift", si.Case("dte", 12, 8, 30, 30, 7, shift=(3, 0), seed=323)),   # W' = 35 is odd: rows may roll, columns not
    ("flat_planes_w7_7", si.Case("dte", 24, 8, 7, 7, 7, seed=324)),                     # 98-byte planes: the plane is the window
    ("aligned_w7_56", si.Case("dte", 21, 6, 56, 56, 7, seed=312)),
    ("boxes_w7_28", si.Case("dte", 40, 10, 28, 28, 7, seed=313)),
    ("gen_shift_w7_28", si.Case("dte", 13, 7, 28, 28, 7, shift=(3, 2), seed=314)),
    ("gen_ragged_w7_60", si.Case("dte", 6, 4, 30, 60, 7, seed=315)),                    # W' = 63 odd, nothing wraps
    ("strips_w7_112", si.Case("dte", 5, 5, 112, 112, 7, seed=316)),
    ("strips_w7_112_shift", si.Case("dte", 4, 3, 112, 112, 7, shift=(3, 4), seed=317)), # > 128 windows / image, shifted
    ("bigmap_w14_224_shift", si.Case("dte", 2, 3, 224, 224, 14, shift=(7, 7), seed=318)),
    ("f16_w14", si.Case("dte", 10, 9, 42, 56, 14, dtype="f16", shift=(0, 7), seed=319)),
    ("simt_w4", si.Case("dte", 3, 5, 10, 7, 4, dtype="f32", seed=320)),
    ("simt_w14_f32", si.Case("dte", 5, 3, 28, 42, 14, dtype="f32", shift=(7, 3), seed=321)),
]


@pytest.mark.parametrize("name,case", DT_EXACT, ids=[n for n, _ in DT_EXACT])
@pytest.mark.parametrize("layout", [NCHW, NHWC])
def test_table_gradient_exact_on_small_integers(wb, oracle, name, case, layout):
    C = case.C if layout == NCHW else -(-case.C // 8) * 8
    gen = torch.Generator().manual_seed(case.seed)
    td = si.TORCH_DTYPES[case.dtype]
    shape = (case.B, C, case.H, case.W)
    x = torch.randint(-2, 3, shape, generator=gen).to(td)
    dy = torch.randint(-2, 3, shape, generator=gen).to(td)
    if layout == NHWC:
        x, dy = (t.permute(0, 2, 3, 1).contiguous() for t in (x, dy))
    _, dT = wb.wbmm_backward(x.cuda(), None, dy.cuda(), case.w, case.shift, layout, need_dx=False)
    torch.cuda.synchronize()
    if layout == NCHW and case.dtype != "f32":      # every 16-bit NCHW mode listed here is a tensor-core mode
        assert wb.wbmm_last_path() == wb.PATH_TC_TMA, wb.wbmm_path_string(wb.wbmm_last_path())
    _, rdT = oracle.backward(widen(x), np.zeros((C, case.bins)), widen(dy), case.w, case.shift, layout, need_dx=False)
    assert np.array_equal(widen(dT), rdT), float(np.abs(widen(dT) - rdT).max())


# ------------------------------------------------------------------ soak: thousands of launches, many shapes, two streams
SOAK = [
    si.Case("k_w14_56", 19, 5, 56, 56, 14, seed=401, backward=True),
    si.Case("k_w14_28_boxes", 40, 12, 28, 28, 14, seed=402, backward=True),
    si.Case("k_w14_28_shift", 24, 9, 28, 28, 14, shift=(7, 7), seed=403, backward=True),
    si.Case("k_w14_shift_even", 9, 7, 28, 56, 14, shift=(3, 4), seed=404, backward=True),
    si.Case("k_w14_ragged", 7, 6, 60, 60, 14, seed=405, backward=True),
    si.Case("k_w14_ragged_shift", 6, 5, 36, 40, 14, shift=(5, 9), seed=406, backward=True),
    si.Case("k_w14_112", 5, 4, 112, 112, 14, seed=407, backward=True),
    si.Case("k_w14_112_shift", 3, 3, 112, 112, 14, shift=(7, 7), seed=408, backward=True),
    si.Case("k_w14_224", 2, 3, 224, 224, 14, seed=409, backward=True),
    si.Case("k_w14_14_planes", 72, 6, 14, 14, 14, seed=410, backward=True),
    si.Case("k_w14_f16", 10, 9, 42, 56, 14, dtype="f16", shift=(0, 7), seed=411, backward=True),
    si.Case("k_w7_56", 21, 6, 56, 56, 7, seed=412, backward=True),
    si.Case("k_w7_28_shift", 13, 7, 28, 28, 7, shift=(3, 2), seed=413, backward=True),
    si.Case("k_w7_ragged", 6, 4, 30, 60, 7, seed=414, backward=True),
    si.Case("k_w7_112", 3, 5, 112, 112, 7, seed=415, backward=True),
    si.Case("k_w7_112_shift", 3, 4, 112, 112, 7, shift=(3, 4), seed=416, backward=True),
    si.Case("k_w7_14_planes", 24, 6, 14, 14, 7, shift=(3, 0), seed=417, backward=True),
    si.Case("k_nhwc_w14", 6, 16, 28, 56, 14, layout=NHWC, shift=(0, 7), seed=418, backward=True),
    si.Case("k_nhwc_w7", 9, 8, 28, 28, 7, layout=NHWC, seed=419, backward=True),
    si.Case("k_f32_w14", 9, 5, 28, 56, 14, dtype="f32", seed=420, backward=True),
    si.Case("k_f32_w7_shift", 5, 7, 28, 28, 7, dtype="f32", shift=(3, 2), seed=421, backward=True),
    si.Case("k_many_channels", 8, 300, 28, 28, 14, seed=422, backward=True),        # > 148 tiles, several channels per CTA
]


def test_soak_many_shapes_two_streams(wb, oracle):
    """>= 5000 launches cycling through 22 shapes x {forward, dX, dT, hierarchical forward} from two host threads on two
    streams, every result checked on the device against ONE oracle evaluation per shape.  The pipelined kernels hand
    work between warps through mbarrier phase parities; a protocol slip shows up as a hang or as a stale tile only
    under the right timing, which single calls with a synchronise after each do not produce."""
    import threading
    items = []
    for c in SOAK:
        d = si.make(c, device="cuda")
        xw, Tw, gw = widen(d["x"]), widen(d["T"]), widen(d["dy"])
        ry = oracle.forward(xw, Tw, c.w, c.shift, c.layout)
        rdx, rdT = oracle.backward(xw, Tw, gw, c.w, c.shift, c.layout)
        ref = {"y": torch.from_numpy(ry).cuda(), "dx": torch.from_numpy(rdx).cuda(), "dT": torch.from_numpy(rdT).cuda()}
        Tl = None
        if c.w == 14 and c.layout == NCHW and c.dtype != "f32":
            Tl = (torch.randn((c.C, 169), generator=torch.Generator().manual_seed(c.seed)) * 0.02).to(d["T"].dtype).cuda()
            ref["hy"] = torch.from_numpy(oracle.hier_forward(xw, Tw, widen(Tl), c.w, c.shift, c.layout, "train")).cuda()
        nwin = c.B * (-(-c.H // c.w)) * (-(-c.W // c.w))
        items.append((c, d, Tl, ref, float(np.sqrt(nwin * c.w * c.w))))
    torch.cuda.synchronize()
    n_per_thread = 2600
    fails, counts = [], [0, 0]

    def err(got, ref, tol, scale=1.0):      # stays on the device: launches of different kernels run back to back
        return ((got.double() - ref).abs() / (tol * (scale + ref.abs()))).max()

    def work(tid):
        st = torch.cuda.Stream()
        with torch.cuda.stream(st):
            worst = torch.zeros((), dtype=torch.float64, device="cuda")
            for it in range(n_per_thread):
                c, d, Tl, ref, dscale = items[(it * 7 + tid * 11) % len(items)]
                op = (it // len(items) + tid) % 4
                tol = TOL[c.dtype]
                if op == 0:
                    e = err(wb.wbmm_forward(d["x"], d["T"], c.w, c.shift, c.layout), ref["y"], tol)
                elif op == 1:
                    e = err(wb.wbmm_backward(None, d["T"], d["dy"], c.w, c.shift, c.layout, need_dT=False)[0], ref["dx"], tol)
                elif op == 2:
                    e = err(wb.wbmm_backward(d["x"], None, d["dy"], c.w, c.shift, c.layout, need_dx=False)[1], ref["dT"], 1e-4, dscale)
                elif Tl is not None:
                    e = err(wb.wbmm_hier_forward(d["x"], d["T"], Tl, c.w, c.shift, c.layout), ref["hy"], tol)
                else:
                    e = err(wb.wbmm_forward(d["x"], d["T"], c.w, c.shift, c.layout), ref["y"], tol)
                worst = torch.maximum(worst, torch.nan_to_num(e, nan=1e30))
                counts[tid] += 1
                if it % 200 == 199 and not float(worst) <= 1.0:
                    fails.append((tid, it, c.name, float(worst)))
                    return
            if not float(worst) <= 1.0:
                fails.append((tid, "end", float(worst)))
        st.synchronize()

    th = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not fails, fails
    assert sum(counts) >= 5000
