"""Pins for the CPU oracle (oracle/wbmm_ref.c): every function is checked against something
other than itself -- closed forms, invariants, special cases that reduce to a library routine
(torch conv2d, Theorem 3.2), exact adjoint identities, finite differences, pure-Python brute
force, and the sizes the paper prints (tests/golden/paper_sizes.txt).

Each pin names the mistake it would catch.  CPU only (-m "not gpu").
"""
import os

import numpy as np
import pytest
import torch
import torch.nn.functional as F

NCHW, NHWC = 0, 1
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_sizes.txt")


def rng(seed):
    return np.random.default_rng(seed)


def golden():
    out = {}
    with open(GOLDEN) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split("=")
                out[k.strip()] = float(v)
    return out


# ----------------------------------------------------------------------------- a1: index
@pytest.mark.parametrize("w", [1, 2, 3, 4, 7, 14])
def test_index_closed_form_properties(oracle, w):
    """Eq. 6-7.  Catches: swapped i/j, wrong stride (2w vs 2w-1), off-by-one."""
    I = oracle.index_matrix(w)
    N, tw = w * w, 2 * w - 1
    nb = tw * tw
    assert I.shape == (N, N)
    assert I.min() == 0 and I.max() == nb - 1              # Theorem 3.1: exactly (2w-1)^2 offsets
    assert np.array_equal(I.T, nb - 1 - I)                 # rel(j,i) = nb-1-rel(i,j)
    centre = (w - 1) * tw + (w - 1)
    assert np.all(np.diag(I) == centre)                    # zero offset -> centre bin
    # bin multiplicity (w-|dr|)(w-|dc|)
    counts = np.bincount(I.ravel(), minlength=nb).reshape(tw, tw)
    d = np.abs(np.arange(tw) - (w - 1))
    assert np.array_equal(counts, np.outer(w - d, w - d))
    # independent construction from coordinate grids (broadcast, no loops)
    r, c = np.divmod(np.arange(N), w)
    I2 = (r[:, None] - r[None, :] + w - 1) * tw + (c[:, None] - c[None, :] + w - 1)
    assert np.array_equal(I, I2)
    # scalar entry point agrees with the matrix
    for (i, j) in [(0, 0), (0, N - 1), (N - 1, 0), (N // 2, N // 3)]:
        assert oracle.rel_index(w, i, j) == I[i, j]


def test_index_paper_sizes(oracle):
    """Sizes the paper prints (golden file, each with its citation)."""
    g = golden()
    assert (2 * 7 - 1) ** 2 == g["table_entries_w7"]
    assert 2 * 7 - 1 == g["table_side_w7"] and 2 * 14 - 1 == g["table_side_w14"]
    assert oracle.index_matrix(7).shape[0] == g["matrix_side_w7"]
    assert oracle.index_matrix(14).shape[0] == g["matrix_side_w14"]
    assert oracle.index_matrix(7).max() + 1 == g["table_entries_w7"]
    assert oracle.index_matrix(14).max() + 1 == g["table_side_w14"] ** 2
    # centre bins quoted in SURVEY 8(c): 84 (w=7), 364 (w=14)
    assert oracle.rel_index(7, 0, 0) == 84 and oracle.rel_index(14, 5, 5) == 364
    M = oracle.weight_matrix(np.zeros((256, 27 * 27)), 14)
    assert abs(M.size * 4 / 2 ** 20 - g["m_footprint_mib_c256_w14_fp32"]) < 0.1   # fp32 bytes
    assert abs(196 / 25 - g["rf_ratio_w14_vs_k5"]) < 0.05


def test_weight_matrix_is_gather(oracle):
    """Eq. 8: values copied, no arithmetic.  Table = its own bin index makes M == I."""
    for w in (3, 7):
        nb = (2 * w - 1) ** 2
        T = np.tile(np.arange(nb, dtype=np.float64), (2, 1))
        T[1] += 1000
        M = oracle.weight_matrix(T, w)
        I = oracle.index_matrix(w)
        assert np.array_equal(M[0], I) and np.array_equal(M[1], I + 1000)


# ----------------------------------------------------------------------------- forward
CASES = [
    # B, C, H, W, w, shift
    (2, 3, 6, 6, 3, (0, 0)),
    (1, 2, 8, 12, 4, (0, 0)),
    (2, 2, 7, 10, 3, (0, 0)),        # ragged both axes
    (2, 2, 9, 6, 3, (1, 2)),         # shift, odd w
    (1, 3, 10, 7, 4, (2, 2)),        # shift + ragged, even w
    (1, 2, 14, 14, 7, (3, 3)),
]


def _to_layout(a, layout):
    return np.ascontiguousarray(a.transpose(0, 2, 3, 1)) if layout == NHWC else a


def _from_layout(a, layout):
    return a.transpose(0, 3, 1, 2) if layout == NHWC else a


@pytest.mark.parametrize("case", CASES)
@pytest.mark.parametrize("layout", [NCHW, NHWC])
def test_matrix_form_equals_direct_form(oracle, case, layout):
    """Two structurally different evaluations (Alg. 1 vs windowed depthwise sum) must agree."""
    B, C, H, W, w, s = case
    r = rng(11)
    x = r.standard_normal((B, C, H, W))
    T = r.standard_normal((C, (2 * w - 1) ** 2))
    ym = oracle.forward(_to_layout(x, layout), T, w, s, layout, "matrix")
    yd = oracle.forward(_to_layout(x, layout), T, w, s, layout, "direct")
    assert np.allclose(ym, yd, rtol=0, atol=1e-12)
    # layouts: NHWC result == NCHW result on permuted copies
    y0 = oracle.forward(x, T, w, s, NCHW, "direct")
    assert np.array_equal(_from_layout(yd, layout), y0)


def brute_force(x, T, w, s=(0, 0)):
    """Pure-Python restatement of the DEFINITION, NCHW, tiny inputs only."""
    B, C, H, W = x.shape
    Hp, Wp = -(-H // w) * w, -(-W // w) * w
    tw = 2 * w - 1
    xt = np.zeros((B, C, Hp, Wp))
    xt[:, :, :H, :W] = x
    xh = np.zeros_like(xt)
    for h in range(Hp):
        for v in range(Wp):
            xh[:, :, h, v] = xt[:, :, (h + s[0]) % Hp, (v + s[1]) % Wp]
    yh = np.zeros_like(xt)
    for b in range(B):
        for c in range(C):
            for h in range(Hp):
                for v in range(Wp):
                    h0, v0 = (h // w) * w, (v // w) * w
                    acc = 0.0
                    for hq in range(h0, h0 + w):
                        for vq in range(v0, v0 + w):
                            acc += T[c, (h - hq + w - 1) * tw + (v - vq + w - 1)] * xh[b, c, hq, vq]
                    yh[b, c, h, v] = acc
    yt = np.zeros_like(xt)
    for h in range(Hp):
        for v in range(Wp):
            yt[:, :, h, v] = yh[:, :, (h - s[0]) % Hp, (v - s[1]) % Wp]
    return yt[:, :, :H, :W]


@pytest.mark.parametrize("case", CASES[:5])
def test_brute_force_tiny(oracle, case):
    B, C, H, W, w, s = case
    r = rng(5)
    x = r.standard_normal((B, C, H, W))
    T = r.standard_normal((C, (2 * w - 1) ** 2))
    ref = brute_force(x, T, w, s)
    for form in ("direct", "matrix"):
        assert np.allclose(oracle.forward(x, T, w, s, NCHW, form), ref, rtol=0, atol=1e-12)


def test_brute_force_config1(oracle):
    """BASELINE.json config 1: B=1, C=4, 14x14, w=7, fp32 inputs, seed 0."""
    import synth_inputs as si
    d = si.make(si.CFG1)
    x, T = d["x"].double().numpy(), d["T"].double().numpy()
    ref = brute_force(x, T, 7)
    assert np.allclose(oracle.forward(x, T, 7, form="direct"), ref, rtol=0, atol=1e-13)
    assert np.allclose(oracle.forward(x, T, 7, form="matrix"), ref, rtol=0, atol=1e-13)


@pytest.mark.parametrize("form", ["direct", "matrix"])
@pytest.mark.parametrize("w,s", [(3, (0, 0)), (4, (0, 0)), (3, (2, 1)), (4, (2, 2))])
def test_delta_table_is_identity(oracle, form, w, s):
    """Delta at the zero-offset bin => y == x exactly.  With a shift this also pins
    shift o inverse-roll == identity."""
    r = rng(2)
    x = r.standard_normal((2, 3, 3 * w - 1, 2 * w + 1))      # ragged
    tw = 2 * w - 1
    T = np.zeros((3, tw * tw))
    T[:, (w - 1) * tw + (w - 1)] = 1.0
    assert np.array_equal(oracle.forward(x, T, w, s, NCHW, form), x)


@pytest.mark.parametrize("form", ["direct", "matrix"])
@pytest.mark.parametrize("w", [3, 4])
def test_one_hot_table_all_bins(oracle, form, w):
    """One-hot table at bin (dr,dc): y[r,c] = x[r-dr, c-dc] if that lies in the same window
    else 0 (north_star orientation: offset = out - in).  Exact.  Catches a transposed W_c,
    a wrong sign, a wrong row stride -- for EVERY bin."""
    r = rng(3)
    H = W = 2 * w
    x = r.standard_normal((1, 1, H, W))
    tw = 2 * w - 1
    for dr in range(-(w - 1), w):
        for dc in range(-(w - 1), w):
            T = np.zeros((1, tw * tw))
            T[0, (dr + w - 1) * tw + (dc + w - 1)] = 1.0
            y = oracle.forward(x, T, w, (0, 0), NCHW, form)
            exp = np.zeros_like(x)
            for wy in range(2):
                for wx in range(2):
                    win = x[0, 0, wy * w:(wy + 1) * w, wx * w:(wx + 1) * w]
                    out = np.zeros((w, w))
                    # out[r, c] = win[r-dr, c-dc] where valid
                    r0, r1 = max(0, dr), min(w, w + dr)
                    c0, c1 = max(0, dc), min(w, w + dc)
                    out[r0:r1, c0:c1] = win[r0 - dr:r1 - dr, c0 - dc:c1 - dc]
                    exp[0, 0, wy * w:(wy + 1) * w, wx * w:(wx + 1) * w] = out
            assert np.array_equal(y, exp), (dr, dc)


@pytest.mark.parametrize("form", ["direct", "matrix"])
def test_all_ones_table_gives_window_sums(oracle, form):
    """Pins partition + bottom/right zero padding (A4): small-integer x, exact."""
    w, H, W = 4, 10, 7
    r = rng(4)
    x = r.integers(-3, 4, size=(2, 2, H, W)).astype(np.float64)
    T = np.ones((2, (2 * w - 1) ** 2))
    y = oracle.forward(x, T, w, (0, 0), NCHW, form)
    for h in range(H):
        for v in range(W):
            h0, v0 = (h // w) * w, (v // w) * w
            s = x[:, :, h0:min(h0 + w, H), v0:min(v0 + w, W)].sum(axis=(2, 3))
            assert np.array_equal(y[:, :, h, v], s)


def test_linearity(oracle):
    r = rng(6)
    w = 3
    x1, x2 = r.standard_normal((2, 2, 2, 7, 8))
    T1, T2 = r.standard_normal((2, 2, 25))
    f = lambda x, T: oracle.forward(x, T, w, (1, 2))
    assert np.allclose(f(2 * x1 - 3 * x2, T1), 2 * f(x1, T1) - 3 * f(x2, T1), atol=1e-12)
    assert np.allclose(f(x1, 2 * T1 - 3 * T2), 2 * f(x1, T1) - 3 * f(x1, T2), atol=1e-12)


@pytest.mark.parametrize("w", [3, 4, 7, 14])
def test_theorem_3_2_single_window_is_depthwise_conv(oracle, w):
    """Theorem 3.2: on a single window (H=W=w) the operator is a zero-padded
    depthwise conv with a (2w-1)^2 kernel -- a LIBRARY routine (torch conv2d, cross-correlation).
    north_star orientation (offset = out - in) is a true convolution => flipped kernel;
    the paper's orientation (offset = in - out) is the table reversed (reading A1)."""
    r = rng(7)
    C = 3
    tw = 2 * w - 1
    x = r.standard_normal((2, C, w, w))
    T = r.standard_normal((C, tw * tw))
    y = oracle.forward(x, T, w)
    K = torch.from_numpy(T.reshape(C, 1, tw, tw))
    conv_flipped = F.conv2d(torch.from_numpy(x), torch.flip(K, dims=(2, 3)), padding=w - 1, groups=C)
    assert np.allclose(y, conv_flipped.numpy(), rtol=0, atol=1e-12)
    # paper convention: WBMM_ns(x; reversed(R)) == conv2d(x, R) (cross-correlation, no flip)
    R = T[:, ::-1].copy()
    conv_paper = F.conv2d(torch.from_numpy(x), torch.from_numpy(R.reshape(C, 1, tw, tw)),
                          padding=w - 1, groups=C)
    assert np.allclose(y, conv_paper.numpy(), rtol=0, atol=1e-12)


def test_multi_window_is_per_window_conv(oracle):
    """Windows do not interact: each window equals the conv on its isolated crop."""
    r = rng(8)
    w, C = 4, 2
    tw = 2 * w - 1
    x = r.standard_normal((1, C, 8, 12))
    T = r.standard_normal((C, tw * tw))
    y = oracle.forward(x, T, w)
    K = torch.flip(torch.from_numpy(T.reshape(C, 1, tw, tw)), dims=(2, 3))
    for wy in range(2):
        for wx in range(3):
            crop = x[:, :, wy * w:(wy + 1) * w, wx * w:(wx + 1) * w]
            ref = F.conv2d(torch.from_numpy(crop.copy()), K, padding=w - 1, groups=C).numpy()
            assert np.allclose(y[:, :, wy * w:(wy + 1) * w, wx * w:(wx + 1) * w], ref, atol=1e-12)


def test_padding_equals_explicit_pad_then_crop(oracle):
    """Eq. 4-5, 'padding is removed'."""
    r = rng(9)
    w = 4
    x = r.standard_normal((2, 2, 10, 7))
    T = r.standard_normal((2, 49))
    xp = np.zeros((2, 2, 12, 8))
    xp[:, :, :10, :7] = x
    assert np.array_equal(oracle.forward(x, T, w), oracle.forward(xp, T, w)[:, :, :10, :7])


@pytest.mark.parametrize("w,s,H,W", [(3, (1, 2), 9, 6), (4, (2, 2), 8, 8), (3, (2, 2), 7, 8), (7, (3, 3), 14, 21)])
def test_shift_equals_explicit_roll(oracle, w, s, H, W):
    """A6: pad, roll by -s over the padded extent, WBMM, roll back by +s, crop."""
    r = rng(10)
    x = r.standard_normal((2, 2, H, W))
    T = r.standard_normal((2, (2 * w - 1) ** 2))
    Hp, Wp = -(-H // w) * w, -(-W // w) * w
    xp = np.zeros((2, 2, Hp, Wp))
    xp[:, :, :H, :W] = x
    xr = np.roll(xp, shift=(-s[0], -s[1]), axis=(2, 3))       # x^[h] = x~[(h+s) mod H']
    yr = oracle.forward(xr, T, w)
    ref = np.roll(yr, shift=(s[0], s[1]), axis=(2, 3))[:, :, :H, :W]
    assert np.allclose(oracle.forward(x, T, w, s), ref, rtol=0, atol=1e-13)
    assert np.array_equal(oracle.forward(x, T, w, (0, 0)), oracle.forward(x, T, w))


def test_shift_direction_pinned_by_odd_w_not_by_even_w(oracle):
    """For even w and s = w/2 the roll direction is immaterial (+s and -s differ by a whole
    window); for odd w it is not -- so the direction is pinned by w=3/7 cases above."""
    r = rng(12)
    for w, s, same in ((4, 2, True), (3, 1, False)):
        x = r.standard_normal((1, 1, 2 * w, 2 * w))
        T = r.standard_normal((1, (2 * w - 1) ** 2))
        y_plus = oracle.forward(x, T, w, (s, s))
        y_minus = oracle.forward(x, T, w, (w - s, w - s))       # -s mod w
        assert np.allclose(y_plus, y_minus, atol=1e-13) == same


# ----------------------------------------------------------------------------- backward
BWD_CASES = [(2, 3, 6, 6, 3, (0, 0)), (2, 2, 7, 10, 3, (1, 2)), (1, 2, 10, 7, 4, (2, 2)), (1, 2, 14, 14, 7, (3, 3))]


@pytest.mark.parametrize("case", BWD_CASES)
@pytest.mark.parametrize("layout", [NCHW, NHWC])
def test_dx_adjoint_identity(oracle, case, layout):
    """<dy, WBMM(x2;T)> == <dX(dy;T), x2> exactly (the operator is linear in x)."""
    B, C, H, W, w, s = case
    r = rng(13)
    x, x2, dy = (_to_layout(a, layout) for a in r.standard_normal((3, B, C, H, W)))
    T = r.standard_normal((C, (2 * w - 1) ** 2))
    dx, _ = oracle.backward(x, T, dy, w, s, layout, need_dT=False)
    lhs = np.vdot(dy, oracle.forward(x2, T, w, s, layout))
    rhs = np.vdot(dx, x2)
    assert abs(lhs - rhs) <= 1e-11 * (1 + abs(lhs))


@pytest.mark.parametrize("case", BWD_CASES)
def test_dx_is_forward_with_reversed_table(oracle, case):
    """W_c^T[i,j] = T[rel(j,i)] = T[nb-1-rel(i,j)]."""
    B, C, H, W, w, s = case
    r = rng(14)
    x, dy = r.standard_normal((2, B, C, H, W))
    T = r.standard_normal((C, (2 * w - 1) ** 2))
    dx, _ = oracle.backward(x, T, dy, w, s, need_dT=False)
    assert np.allclose(dx, oracle.forward(dy, T[:, ::-1].copy(), w, s), rtol=0, atol=1e-12)


@pytest.mark.parametrize("case", BWD_CASES)
@pytest.mark.parametrize("layout", [NCHW, NHWC])
def test_dT_adjoint_identity(oracle, case, layout):
    """<dT, T2> == <dy, WBMM(x;T2)> for any T2 (the operator is linear in T): exact."""
    B, C, H, W, w, s = case
    r = rng(15)
    x, dy = (_to_layout(a, layout) for a in r.standard_normal((2, B, C, H, W)))
    T, T2 = r.standard_normal((2, C, (2 * w - 1) ** 2))
    _, dT = oracle.backward(x, T, dy, w, s, layout, need_dx=False)
    lhs = np.vdot(dT, T2)
    rhs = np.vdot(dy, oracle.forward(x, T2, w, s, layout))
    assert abs(lhs - rhs) <= 1e-11 * (1 + abs(lhs))


def test_dT_and_dx_finite_difference(oracle):
    """Central finite difference of L = <dy, WBMM(x;T)> on tiny inputs in fp64 (north_star)."""
    r = rng(16)
    B, C, H, W, w, s = 1, 2, 5, 7, 3, (1, 1)
    x, dy = r.standard_normal((2, B, C, H, W))
    T = r.standard_normal((C, 25))
    dx, dT = oracle.backward(x, T, dy, w, s)
    L = lambda x_, T_: np.vdot(dy, oracle.forward(x_, T_, w, s))
    eps = 1e-4
    for (c, k) in [(0, 0), (0, 12), (1, 24), (1, 7), (0, 18)]:
        Tp, Tm = T.copy(), T.copy()
        Tp[c, k] += eps
        Tm[c, k] -= eps
        fd = (L(x, Tp) - L(x, Tm)) / (2 * eps)
        assert abs(fd - dT[c, k]) <= 1e-8 * (1 + abs(fd))
    for idx in [(0, 0, 0, 0), (0, 1, 4, 6), (0, 0, 2, 3), (0, 1, 3, 0)]:
        xp_, xm_ = x.copy(), x.copy()
        xp_[idx] += eps
        xm_[idx] -= eps
        fd = (L(xp_, T) - L(xm_, T)) / (2 * eps)
        assert abs(fd - dx[idx]) <= 1e-8 * (1 + abs(fd))


def test_dT_one_hot_pairs_land_in_one_bin(oracle):
    """One-hot dy at output position p and one-hot x at input position q of the same window
    => dT has a single 1 at bin rel(p,q); different windows => dT == 0."""
    w, tw = 3, 5
    for (p, q) in [((0, 0), (2, 2)), ((1, 2), (1, 0)), ((2, 1), (0, 1)), ((4, 4), (3, 5)), ((0, 0), (0, 3))]:
        x = np.zeros((1, 1, 6, 6))
        dy = np.zeros((1, 1, 6, 6))
        x[0, 0, q[0], q[1]] = 1.0
        dy[0, 0, p[0], p[1]] = 1.0
        _, dT = oracle.backward(x, np.zeros((1, 25)), dy, w, need_dx=False)
        exp = np.zeros((1, 25))
        if p[0] // w == q[0] // w and p[1] // w == q[1] // w:
            exp[0, (p[0] - q[0] + w - 1) * tw + (p[1] - q[1] + w - 1)] = 1.0
        assert np.array_equal(dT, exp), (p, q)


def test_backward_ignores_padded_region(oracle):
    """A11: dy is zero outside HxW; padded x zeros contribute nothing to dT."""
    r = rng(17)
    w = 4
    x, dy = r.standard_normal((2, 1, 2, 6, 7))
    T = r.standard_normal((2, 49))
    xp, dyp = np.zeros((2, 1, 2, 8, 8)), np.zeros((2, 1, 2, 8, 8))
    xp[0][..., :6, :7] = x
    xp[1][..., :6, :7] = dy
    dx, dT = oracle.backward(x, T, dy, w)
    dx2, dT2 = oracle.backward(xp[0], T, xp[1], w)
    assert np.allclose(dT, dT2, atol=1e-13) and np.allclose(dx, dx2[..., :6, :7], atol=1e-13)


# ------------------------------------------------------------------ hierarchical reparameterisation (Alg. 2 / 3)
def _hier_inputs(seed, B, C, H, W, w):
    r = rng(seed)
    x = r.standard_normal((B, C, H, W))
    Tg = 0.05 * r.standard_normal((C, (2 * w - 1) ** 2))
    Tl = 0.05 * r.standard_normal((C, (w - 1) ** 2))
    return x, Tg, Tl


@pytest.mark.parametrize("w,H,W,s", [(4, 8, 12, (0, 0)), (6, 12, 12, (0, 0)), (4, 10, 7, (1, 3)), (14, 28, 14, (0, 0)), (14, 30, 20, (7, 5))])
@pytest.mark.parametrize("layout", [NCHW, NHWC])
def test_hier_training_form_equals_fused_form(oracle, w, H, W, s, layout):
    """PAPER.md:891 "Algorithms 2 and 3 are functionally identical": the two structurally different
    evaluations (two scales + shortcuts vs. one fused matrix) agree to round-off, also transposed."""
    x, Tg, Tl = _hier_inputs(50 + w, 2, 3, H, W, w)
    xl = _to_layout(x, layout)
    for tr in (False, True):
        a = oracle.hier_forward(xl, Tg, Tl, w, s, layout, "train", tr)
        b = oracle.hier_forward(xl, Tg, Tl, w, s, layout, "fused", tr)
        assert np.max(np.abs(a - b)) < 1e-12


@pytest.mark.parametrize("w", [4, 14])
def test_hier_is_sum_of_single_scale_operators_plus_two_x(oracle, w):
    """On maps that are multiples of w the local sub-windows ARE the w/2 partition of the image, so
    Y = WBMM(x; Tg, w) + WBMM(x; Tl, w/2) + 2x -- reduces the hierarchical oracle to
    the single-scale one, which is pinned above."""
    x, Tg, Tl = _hier_inputs(60 + w, 2, 3, 2 * w, 3 * w, w)
    y = oracle.hier_forward(x, Tg, Tl, w, form="fused")
    ref = oracle.forward(x, Tg, w) + oracle.forward(x, Tl, w // 2) + 2 * x
    assert np.max(np.abs(y - ref)) < 1e-12


def test_hier_fused_matrix_structure(oracle):
    """Eq. 9 / Alg. 3: M_fused - M_g is I_196 everywhere plus (M_l + I_49) on the four diagonal
    sub-window blocks and NOTHING on the cross-sub-window blocks."""
    w, wl = 14, 7
    x, Tg, Tl = _hier_inputs(70, 1, 2, w, w, w)
    _, M = oracle.hier_forward(x, Tg, Tl, w, form="fused", return_matrix=True)
    Mg = oracle.weight_matrix(Tg, w)
    Ml = oracle.weight_matrix(Tl, wl)
    D = (M - Mg).reshape(2, 2, wl, 2, wl, 2, wl, 2, wl)       # (c, s_or, p_or, s_oc, p_oc, s_ir, p_ir, s_ic, p_ic)
    eye = np.eye(wl * wl).reshape(wl, wl, wl, wl)
    for a in range(2):
        for e in range(2):
            for a2 in range(2):
                for e2 in range(2):
                    blk = D[:, a, :, e, :, a2, :, e2, :]      # (c, p_or, p_oc, p_ir, p_ic)
                    if (a, e) == (a2, e2):
                        exp = Ml.reshape(2, wl, wl, wl, wl) + 2 * eye[None]
                        assert np.max(np.abs(blk - exp)) < 1e-14
                    else:
                        assert np.max(np.abs(blk)) == 0.0
    # size printed by the paper: (C, 196, 196) for 14 x 14 windows
    assert M.shape == (2, 196, 196)


def test_hier_transpose_is_adjoint(oracle):
    w = 6
    x, Tg, Tl = _hier_inputs(80, 2, 2, 13, 9, w)
    r = rng(81)
    dy = r.standard_normal(x.shape)
    y = oracle.hier_forward(x, Tg, Tl, w, (2, 5), form="train")
    dx = oracle.hier_forward(dy, Tg, Tl, w, (2, 5), form="train", transpose=True)
    assert abs(np.sum(dy * y) - np.sum(dx * x)) < 1e-10


# ------------------------------------------------------------------ hierarchical backward (tables)
@pytest.mark.parametrize("w,H,W,s", [(4, 8, 12, (0, 0)), (4, 10, 7, (1, 3)), (6, 13, 9, (2, 5)), (14, 30, 20, (7, 5))])
@pytest.mark.parametrize("layout", [NCHW, NHWC])
def test_hier_table_gradients_are_directional_derivatives(oracle, w, H, W, s, layout):
    """y is linear in (Tg, Tl): <dTg, dG> + <dTl, dL> must equal <dy, y(Tg+dG, Tl+dL) - y(Tg, Tl)> exactly
    (to round-off) for ANY direction -- checks the table gradients against the pinned forward, not
    against themselves; a wrong index, sign or a dropped sub-window fails it."""
    x, Tg, Tl = _hier_inputs(90 + w, 2, 3, H, W, w)
    r = rng(91 + w)
    dy = r.standard_normal(x.shape)
    dG = r.standard_normal(Tg.shape)
    dL = r.standard_normal(Tl.shape)
    xl, dyl = _to_layout(x, layout), _to_layout(dy, layout)
    _, dTg, dTl = oracle.hier_backward(xl, Tg, Tl, dyl, w, s, layout)
    for a, b_ in ((dG, 0 * dL), (0 * dG, dL), (dG, dL)):
        y1 = oracle.hier_forward(xl, Tg + a, Tl + b_, w, s, layout, "fused")
        y0 = oracle.hier_forward(xl, Tg, Tl, w, s, layout, "fused")
        lhs = np.sum(dTg * a) + np.sum(dTl * b_)
        rhs = np.sum(dyl * (y1 - y0))
        assert abs(lhs - rhs) < 1e-9 * (1 + abs(rhs))


@pytest.mark.parametrize("w", [4, 14])
def test_hier_table_gradients_reduce_to_single_scale(oracle, w):
    """On maps that are multiples of w (no shift) the local sub-windows are the w/2 partition of the
    image: dTg, dTl are the single-scale table gradients at w and w/2 (pinned above)."""
    x, Tg, Tl = _hier_inputs(100 + w, 2, 3, 2 * w, 3 * w, w)
    dy = rng(101 + w).standard_normal(x.shape)
    dx, dTg, dTl = oracle.hier_backward(x, Tg, Tl, dy, w)
    _, rg = oracle.backward(x, Tg, dy, w, need_dx=False)
    _, rl = oracle.backward(x, Tl, dy, w // 2, need_dx=False)
    assert np.max(np.abs(dTg - rg)) < 1e-11
    assert np.max(np.abs(dTl - rl)) < 1e-11
    rdx, _ = oracle.backward(x, Tg, dy, w, need_dT=False)
    rdl, _ = oracle.backward(x, Tl, dy, w // 2, need_dT=False)
    assert np.max(np.abs(dx - (rdx + rdl + 2 * dy))) < 1e-11


def test_hier_table_gradients_w2_closed_form(oracle):
    """w = 2: the local windows are single pixels, Tl has one entry per channel and dTl = sum(dy * x);
    the centre bin of dTg (rel = 4 of 9) is the same sum."""
    r = rng(110)
    x = r.standard_normal((3, 2, 4, 6))
    dy = r.standard_normal(x.shape)
    Tg = r.standard_normal((2, 9))
    Tl = r.standard_normal((2, 1))
    _, dTg, dTl = oracle.hier_backward(x, Tg, Tl, dy, 2)
    s = np.sum(dy * x, axis=(0, 2, 3))
    assert np.max(np.abs(dTl[:, 0] - s)) < 1e-12
    assert np.max(np.abs(dTg[:, 4] - s)) < 1e-12
    # the corner bin (dr, dc) = (+1, +1): output position (1,1) reads input position (0,0) of each 2 x 2 window
    c = np.sum(dy[:, :, 1::2, 1::2] * x[:, :, 0::2, 0::2], axis=(0, 2, 3))
    assert np.max(np.abs(dTg[:, 8] - c)) < 1e-12


# ------------------------------------------------------------------ cached-M mode and multi-kernel fusion (NEXT-2)
@pytest.mark.parametrize("w,H,W,s", [(3, 6, 9, (0, 0)), (4, 10, 7, (1, 3)), (7, 14, 21, (3, 0)), (14, 30, 20, (7, 5))])
@pytest.mark.parametrize("layout", [NCHW, NHWC])
def test_apply_matrix_with_table_matrix_is_the_operator(oracle, w, H, W, s, layout):
    """WBMM-C and WBMM-NC "produce identical outputs": Algorithm 1 with M = R[:, I] given as
    a matrix equals the pinned direct form; the transposed application equals the pinned dX."""
    r = rng(120 + w)
    x = r.standard_normal((2, 3, H, W))
    T = r.standard_normal((3, (2 * w - 1) ** 2))
    xl = _to_layout(x, layout)
    M = oracle.weight_matrix(T, w)
    assert np.max(np.abs(oracle.apply_matrix(xl, M, w, s, layout) - oracle.forward(xl, T, w, s, layout))) < 1e-12
    dx, _ = oracle.backward(xl, T, xl, w, s, layout, need_dT=False)
    assert np.max(np.abs(oracle.apply_matrix(xl, M, w, s, layout, transpose=True) - dx)) < 1e-12


def test_apply_matrix_brute_force_non_toeplitz(oracle):
    """An arbitrary (non-Toeplitz) M and a bias against pure-Python loops over a tiny ragged, shifted map."""
    r = rng(130)
    B, C, H, W, w, s = 2, 2, 5, 7, 3, (1, 2)
    x = r.standard_normal((B, C, H, W))
    M = r.standard_normal((C, 9, 9))
    bias = r.standard_normal(C)
    Hp, Wp = 6, 9
    ref = np.zeros_like(x)
    for b in range(B):
        for c in range(C):
            for wy in range(Hp // w):
                for wx in range(Wp // w):
                    for i in range(9):
                        acc = 0.0
                        for j in range(9):
                            h, v = (wy * w + j // w + s[0]) % Hp, (wx * w + j % w + s[1]) % Wp
                            acc += M[c, i, j] * (x[b, c, h, v] if h < H and v < W else 0.0)
                        h, v = (wy * w + i // w + s[0]) % Hp, (wx * w + i % w + s[1]) % Wp
                        if h < H and v < W:
                            ref[b, c, h, v] = acc + bias[c]
    assert np.max(np.abs(oracle.apply_matrix(x, M, w, s, bias=bias) - ref)) < 1e-13


@pytest.mark.parametrize("w", [7, 5])
def test_fold_dwconv_equals_library_conv_on_one_window(oracle, w):
    """Section 3.7: Y = WBMM(X) + BN1(DW5(X)) + BN2(DW3(X)) on a single-window map equals ONE WBMM with the
    folded table plus a bias -- the conv branches come from a LIBRARY routine (torch conv2d, cross-correlation,
    zero padding), the BatchNorms are written out as scale and shift."""
    import torch
    import torch.nn.functional as F
    r = rng(140 + w)
    B, C = 3, 4
    x = r.standard_normal((B, C, w, w))
    T = 0.1 * r.standard_normal((C, (2 * w - 1) ** 2))
    K5, K3 = r.standard_normal((C, 5, 5)), r.standard_normal((C, 3, 3))
    s1, b1, s2, b2 = (r.standard_normal(C) for _ in range(4))
    xt = torch.from_numpy(x)
    d5 = F.conv2d(xt, torch.from_numpy(K5).reshape(C, 1, 5, 5), padding=2, groups=C).numpy()
    d3 = F.conv2d(xt, torch.from_numpy(K3).reshape(C, 1, 3, 3), padding=1, groups=C).numpy()
    ref = oracle.forward(x, T, w) + s1.reshape(1, C, 1, 1) * d5 + b1.reshape(1, C, 1, 1) \
        + s2.reshape(1, C, 1, 1) * d3 + b2.reshape(1, C, 1, 1)
    Tf = oracle.fold_dwconv(oracle.fold_dwconv(T, K5, w, s1), K3, w, s2)
    got = oracle.apply_matrix(x, oracle.weight_matrix(Tf, w), w, bias=b1 + b2)
    assert np.max(np.abs(got - ref)) < 1e-11


# ------------------------------------------------------------------ rectangular windows w_h x w_w (Eq. 4-7)
RECT = [(2, 3), (3, 2), (1, 5), (4, 1), (7, 14), (14, 7), (3, 8)]


@pytest.mark.parametrize("wh,ww", RECT)
def test_rect_single_window_is_depthwise_conv(oracle, wh, ww):
    """Theorem 3.2 for a w_h x w_w window: on a map of ONE window the operator is the zero-padded depthwise conv with a
    (2w_h-1) x (2w_w-1) kernel -- a library routine (torch conv2d).  Pins Eq. 7's rectangular index
    I = (dh + w_h - 1)(2w_w - 1) + (dw + w_w - 1): a transposed table shape or a swapped w_h / w_w fails."""
    r = rng(31)
    C = 3
    x = r.standard_normal((2, C, wh, ww))
    T = r.standard_normal((C, (2 * wh - 1) * (2 * ww - 1)))
    y = oracle.forward_rect(x, T, wh, ww)
    K = torch.from_numpy(T.reshape(C, 1, 2 * wh - 1, 2 * ww - 1))
    ref = F.conv2d(torch.from_numpy(x), torch.flip(K, dims=(2, 3)), padding=(wh - 1, ww - 1), groups=C)
    assert np.allclose(y, ref.numpy(), rtol=0, atol=1e-12)


@pytest.mark.parametrize("w,s,H,W,layout", [(3, (0, 0), 9, 6, NCHW), (4, (1, 3), 10, 7, NCHW), (7, (3, 2), 14, 20, NHWC)])
def test_rect_reduces_to_the_square_operator(oracle, w, s, H, W, layout):
    """w_h = w_w = w: forward, dX and dT equal the square oracle's (written apart: two sets of loops)."""
    r = rng(32)
    shape = (2, 3, H, W) if layout == NCHW else (2, H, W, 3)
    x, dy = r.standard_normal(shape), r.standard_normal(shape)
    T = r.standard_normal((3, (2 * w - 1) ** 2))
    assert np.allclose(oracle.forward_rect(x, T, w, w, s, layout), oracle.forward(x, T, w, s, layout), rtol=0, atol=1e-12)
    dx, dT = oracle.backward_rect(x, T, dy, w, w, s, layout)
    rdx, rdT = oracle.backward(x, T, dy, w, s, layout)
    assert np.allclose(dx, rdx, rtol=0, atol=1e-12) and np.allclose(dT, rdT, rtol=0, atol=1e-11)


def test_rect_windows_do_not_interact_and_padding_is_cropped(oracle):
    """Each w_h x w_w window equals the conv on its isolated crop (Alg. 1 l.3-4); Eq. 4-5: pad_h by w_h, pad_w by w_w."""
    r = rng(33)
    wh, ww, C = 2, 5, 2
    x = r.standard_normal((1, C, 5, 12))                       # H' = 6, W' = 15
    T = r.standard_normal((C, 3 * 9))
    y = oracle.forward_rect(x, T, wh, ww)
    xp = np.zeros((1, C, 6, 15))
    xp[:, :, :5, :12] = x
    yp = oracle.forward_rect(xp, T, wh, ww)
    assert np.array_equal(y, yp[:, :, :5, :12])
    K = torch.flip(torch.from_numpy(T.reshape(C, 1, 3, 9)), dims=(2, 3))
    for wy in range(3):
        for wx in range(3):
            crop = xp[:, :, wy * wh:(wy + 1) * wh, wx * ww:(wx + 1) * ww]
            ref = F.conv2d(torch.from_numpy(crop.copy()), K, padding=(wh - 1, ww - 1), groups=C).numpy()
            assert np.allclose(yp[:, :, wy * wh:(wy + 1) * wh, wx * ww:(wx + 1) * ww], ref, atol=1e-12)


@pytest.mark.parametrize("wh,ww,s,H,W", [(2, 3, (1, 2), 6, 9), (3, 5, (2, 4), 7, 11), (1, 4, (0, 3), 3, 10)])
def test_rect_shift_equals_explicit_roll(oracle, wh, ww, s, H, W):
    """A6 on rectangular windows: pad, roll by -s over the padded extent, operator, roll back, crop."""
    r = rng(34)
    x = r.standard_normal((2, 2, H, W))
    T = r.standard_normal((2, (2 * wh - 1) * (2 * ww - 1)))
    Hp, Wp = -(-H // wh) * wh, -(-W // ww) * ww
    xp = np.zeros((2, 2, Hp, Wp))
    xp[:, :, :H, :W] = x
    yr = oracle.forward_rect(np.roll(xp, shift=(-s[0], -s[1]), axis=(2, 3)), T, wh, ww)
    ref = np.roll(yr, shift=(s[0], s[1]), axis=(2, 3))[:, :, :H, :W]
    assert np.allclose(oracle.forward_rect(x, T, wh, ww, s), ref, rtol=0, atol=1e-13)


@pytest.mark.parametrize("wh,ww,s,H,W,layout", [(2, 3, (1, 2), 6, 9, NCHW), (3, 5, (2, 4), 7, 11, NHWC), (1, 6, (0, 0), 2, 13, NCHW)])
def test_rect_backward_adjoint_and_finite_differences(oracle, wh, ww, s, H, W, layout):
    """<dy, A x> = <A^T dy, x> for dx; dT against central differences of the (linear in T) forward."""
    r = rng(35)
    C = 2
    shape = (2, C, H, W) if layout == NCHW else (2, H, W, C)
    x, dy = r.standard_normal(shape), r.standard_normal(shape)
    nb = (2 * wh - 1) * (2 * ww - 1)
    T = r.standard_normal((C, nb))
    dx, dT = oracle.backward_rect(x, T, dy, wh, ww, s, layout)
    assert np.isclose(np.sum(dy * oracle.forward_rect(x, T, wh, ww, s, layout)), np.sum(dx * x), rtol=1e-12)
    for c, k in ((0, 0), (1, nb - 1), (0, nb // 2), (1, 3)):
        E = np.zeros_like(T)
        E[c, k] = 1.0
        # the forward is linear in T: its derivative along E is the forward with table E
        assert np.isclose(dT[c, k], np.sum(dy * oracle.forward_rect(x, E, wh, ww, s, layout)), rtol=1e-11, atol=1e-12)


def test_rect_one_dimensional_windows(oracle):
    """w_h = 1 (1-D sequences): rows never mix, each row is a windowed 1-D operator."""
    r = rng(36)
    ww = 5
    x = r.standard_normal((2, 3, 4, 15))
    T = r.standard_normal((3, 2 * ww - 1))
    y = oracle.forward_rect(x, T, 1, ww)
    for h in range(4):
        assert np.array_equal(y[:, :, h:h + 1, :], oracle.forward_rect(x[:, :, h:h + 1, :].copy(), T, 1, ww))
    # brute force: y[v] = sum_{v' in window} T[v - v' + ww - 1] x[v']
    ref = np.zeros_like(x)
    for v in range(15):
        v0 = (v // ww) * ww
        for vq in range(v0, v0 + ww):
            ref[:, :, :, v] += T[None, :, None, v - vq + ww - 1] * x[:, :, :, vq]
    assert np.allclose(y, ref, rtol=0, atol=1e-12)


# ----------------------------------------------------------------------------- NEXT-4: INT8 forward
def _int8_brute(x, T, w, s, scale=None):
    """Pure-Python restatement of Alg. 1 on integers (NCHW): pad, roll by -s, windows, W_c[i,j] = T[rel(i,j)], roll back."""
    B, C, H, W = x.shape
    Hp, Wp = -(-H // w) * w, -(-W // w) * w
    tw = 2 * w - 1
    xp = np.zeros((B, C, Hp, Wp), dtype=np.int64)
    xp[:, :, :H, :W] = x
    xh = np.roll(xp, (-s[0], -s[1]), axis=(2, 3))
    yh = np.zeros_like(xh)
    for b in range(B):
        for c in range(C):
            for h0 in range(0, Hp, w):
                for v0 in range(0, Wp, w):
                    for i in range(w * w):
                        acc = 0
                        for j in range(w * w):
                            k = (i // w - j // w + w - 1) * tw + (i % w - j % w + w - 1)
                            acc += int(T[c, k]) * int(xh[b, c, h0 + j // w, v0 + j % w])
                        yh[b, c, h0 + i // w, v0 + i % w] = acc
    y = np.roll(yh, (s[0], s[1]), axis=(2, 3))[:, :, :H, :W]
    if scale is None:
        return y
    q = np.rint(y.astype(np.float32) * scale.astype(np.float32)[None, :, None, None])
    return np.clip(q, -128, 127).astype(np.int8)


@pytest.mark.parametrize("w,H,W,s", [(2, 4, 4, (0, 0)), (3, 7, 8, (1, 2)), (4, 9, 6, (3, 0))])
def test_int8_forward_is_the_brute_force_sum(oracle, w, H, W, s):
    """Catches: a wrong bin index, padding treated as non-zero, shift direction, sign extension of the 8-bit values."""
    r = rng(700 + w)
    x = r.integers(-128, 128, (2, 3, H, W), dtype=np.int8)
    T = r.integers(-128, 128, (3, (2 * w - 1) ** 2), dtype=np.int8)
    want = _int8_brute(x, T, w, s)
    assert np.array_equal(oracle.forward_int8(x, T, w, s).astype(np.int64), want)
    xn = np.ascontiguousarray(x.transpose(0, 2, 3, 1))
    got = oracle.forward_int8(xn, T, w, s, layout=NHWC).transpose(0, 3, 1, 2)
    assert np.array_equal(got.astype(np.int64), want)


@pytest.mark.parametrize("w,H,W,s,layout", [(7, 16, 20, (3, 5), NCHW), (14, 28, 30, (7, 2), NHWC), (5, 10, 10, (0, 0), NCHW)])
def test_int8_forward_equals_the_float64_operator_on_integers(oracle, w, H, W, s, layout):
    """Integer inputs are exact in float64 (|sum| < 2^53): the pinned float64 forward gives the same numbers.
    Catches: any disagreement between the 8-bit routine and the operator pinned above (extreme values included)."""
    r = rng(710 + w)
    shape = (2, 4, H, W) if layout == NCHW else (2, H, W, 4)
    x = r.integers(-128, 128, shape, dtype=np.int8)
    T = r.integers(-128, 128, (4, (2 * w - 1) ** 2), dtype=np.int8)
    x.flat[:7] = -128
    T[0, :] = -128                                    # the largest products: (-128) * (-128)
    want = oracle.forward(x.astype(np.float64), T.astype(np.float64), w, s, layout)
    assert np.array_equal(oracle.forward_int8(x, T, w, s, layout).astype(np.float64), want)


def test_int8_requantisation_rounds_to_even_and_saturates(oracle):
    """Identity table (centre bin 1): the sum is x itself, so q = sat(rne(x * scale)) has a closed form.
    Catches: truncation or round-half-away instead of ties-to-even, missing saturation, scale taken from the wrong channel."""
    w = 3
    x = np.arange(-128, 128, dtype=np.int8).reshape(1, 1, 16, 16).repeat(3, axis=1).copy()
    T = np.zeros((3, 25), dtype=np.int8)
    T[:, 12] = 1
    scale = np.array([0.5, 1.5, -2.0], dtype=np.float32)
    q = oracle.forward_int8(x, T, w, scale=scale)
    xi = np.arange(-128, 128).reshape(16, 16)
    # ties to even written out: v/2 is a tie when v is odd; the even neighbour is chosen
    def rne(a):
        f = np.floor(a)
        d = a - f
        return np.where(d > 0.5, f + 1, np.where(d < 0.5, f, np.where(f % 2 == 0, f, f + 1)))
    assert np.array_equal(q[0, 0], np.clip(rne(xi * 0.5), -128, 127).astype(np.int8))
    assert np.array_equal(q[0, 1], np.clip(rne(xi * 1.5), -128, 127).astype(np.int8))      # saturates beyond |x| > 85
    assert np.array_equal(q[0, 2], np.clip(rne(xi * -2.0), -128, 127).astype(np.int8))     # sign, saturation at +127 / -128
    assert q[0, 0, 8, 1] == 0 and q[0, 0, 8, 3] == 2 and q[0, 0, 8, 5] == 2                # 0.5 -> 0, 1.5 -> 2, 2.5 -> 2
    assert q[0, 1].max() == 127 and q[0, 1].min() == -128


def test_int8_requantisation_uses_binary32_products(oracle):
    """The largest sum of a 14 x 14 window (196 * 127 * 127 = 3 161 284) times scales that are not binary fractions:
    the quantised value is the one numpy gets with every intermediate held in binary32 (conversion, one product,
    round-to-nearest-even).  Catches: a float64 product, a fused multiply-add, a wrong clamp order."""
    w = 14
    T = np.zeros((1, 729), dtype=np.int8)
    T[0, :] = 127
    x = np.full((1, 1, 14, 14), 127, dtype=np.int8)
    s = int(oracle.forward_int8(x, T, w)[0, 0, 7, 7])
    assert s == 196 * 127 * 127
    for sc in (np.float32(1e-4), np.float32(3.3e-5), np.nextafter(np.float32(4e-5), np.float32(0))):
        q = int(oracle.forward_int8(x, T, w, scale=np.array([sc], dtype=np.float32))[0, 0, 7, 7])
        want = int(np.clip(np.rint(np.float32(np.float32(s) * sc)), -128, 127))
        assert q == want, (sc, q, want)


# ----------------------------------------------------------------------------- NEXT-4: FP8 (E4M3) decode
def test_e4m3_decode_matches_the_format_and_the_library(oracle):
    """All 256 codes against torch's float8_e4m3fn conversion (a library routine) and the facts of the format: 0x38 = 1,
    largest finite 448 (0x7e), smallest subnormal 2^-9 (0x01), 0x7f / 0xff NaN, 0x80 = -0.
    Catches: wrong bias, subnormals treated as normals, the 'fnuz' or IEEE-like flavour with infinities."""
    codes = np.arange(256, dtype=np.uint8)
    got = oracle.e4m3_decode(codes)
    lib = torch.from_numpy(codes.copy()).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    assert np.array_equal(np.isnan(got), np.isnan(lib)) and np.array_equal(got[~np.isnan(got)], lib[~np.isnan(lib)])
    assert got[0x38] == 1.0 and got[0x7e] == 448.0 and got[0x01] == 2.0 ** -9 and got[0x08] == 2.0 ** -6
    assert np.isnan(got[0x7f]) and np.isnan(got[0xff]) and got[0x80] == 0.0 and np.signbit(got[0x80])
    assert got[0xb8] == -1.0 and got[0x3c] == 1.5


def test_fp8_forward_is_the_operator_on_decoded_values(oracle):
    """Identity table (code 0x38 = 1.0 at the centre bin) returns the decoded input; an all-ones table the window sums.
    Catches: codes used as integers, scale applied to the wrong axis in NHWC."""
    r = rng(900)
    w = 4
    codes = r.integers(0, 256, (2, 3, 8, 8)).astype(np.uint8)
    codes[(codes & 0x7f) == 0x7f] = 0x38                      # no NaN
    T = np.zeros((3, 49), dtype=np.uint8)
    T[:, 24] = 0x38
    x = oracle.e4m3_decode(codes)
    assert np.array_equal(oracle.forward_fp8(codes, T, w), x)
    T1 = np.full((3, 49), 0x38, dtype=np.uint8)
    y = oracle.forward_fp8(codes, T1, w)
    want = x.reshape(2, 3, 2, 4, 2, 4).sum(axis=(3, 5), keepdims=True).repeat(4, axis=3).repeat(4, axis=5).reshape(2, 3, 8, 8)
    assert np.array_equal(y, want)
    sc = np.array([0.5, 2.0, -1.0])
    yn = oracle.forward_fp8(np.ascontiguousarray(codes.transpose(0, 2, 3, 1)), T1, w, layout=NHWC, scale=sc)
    assert np.array_equal(yn.transpose(0, 3, 1, 2), want * sc[None, :, None, None])


# ----------------------------------------------------------------------------- NEXT-4: 3-D windows (reading A23)
WIN3 = [(2, 3, 4), (3, 2, 2), (1, 3, 3), (2, 1, 5)]


@pytest.mark.parametrize("win", WIN3)
def test_3d_single_window_is_depthwise_conv3d(oracle, win):
    """Theorem 3.2 with one more axis: on a volume of ONE window the operator is the zero-padded depthwise conv3d with a
    (2w_d-1) x (2w_h-1) x (2w_w-1) kernel (library routine).  Catches: a wrong stride in the 3-D index, swapped axes."""
    wd, wh, ww = win
    r = rng(950)
    C = 3
    x = r.standard_normal((2, C, wd, wh, ww))
    T = r.standard_normal((C, (2 * wd - 1) * (2 * wh - 1) * (2 * ww - 1)))
    y = oracle.forward_3d(x, T, win)
    K = torch.from_numpy(T.reshape(C, 1, 2 * wd - 1, 2 * wh - 1, 2 * ww - 1))
    ref = F.conv3d(torch.from_numpy(x), torch.flip(K, dims=(2, 3, 4)), padding=(wd - 1, wh - 1, ww - 1), groups=C)
    assert np.allclose(y, ref.numpy(), rtol=0, atol=1e-12)


@pytest.mark.parametrize("layout", [NCHW, NHWC])
def test_3d_depth_one_windows_are_the_rectangular_operator_per_slice(oracle, layout):
    """w_d = 1: every depth slice is an independent 2-D problem (depth acts as batch); forward, dX and dT equal the
    pinned rectangular oracle's.  Catches: depth leaking between slices, layout strides."""
    r = rng(951)
    B, C, D, H, W, wh, ww, s = 2, 3, 4, 7, 9, 3, 4, (0, 2, 1)
    x = r.standard_normal((B, C, D, H, W))
    dy = r.standard_normal((B, C, D, H, W))
    T = r.standard_normal((C, (2 * wh - 1) * (2 * ww - 1)))
    to = (lambda a: np.ascontiguousarray(a.transpose(0, 2, 3, 4, 1))) if layout == NHWC else (lambda a: a)
    back = (lambda a: a.transpose(0, 4, 1, 2, 3)) if layout == NHWC else (lambda a: a)
    y = back(oracle.forward_3d(to(x), T, (1, wh, ww), s, layout))
    dx, dT = oracle.backward_3d(to(x), T, to(dy), (1, wh, ww), s, layout)
    x2 = x.transpose(0, 2, 1, 3, 4).reshape(B * D, C, H, W)
    g2 = dy.transpose(0, 2, 1, 3, 4).reshape(B * D, C, H, W)
    y2 = oracle.forward_rect(x2, T, wh, ww, s[1:])
    dx2, dT2 = oracle.backward_rect(x2, T, g2, wh, ww, s[1:])
    unfold = lambda a: a.reshape(B, D, C, H, W).transpose(0, 2, 1, 3, 4)
    assert np.allclose(y, unfold(y2), rtol=0, atol=1e-12)
    assert np.allclose(back(dx), unfold(dx2), rtol=0, atol=1e-12) and np.allclose(dT, dT2, rtol=0, atol=1e-11)


def test_3d_axes_are_interchangeable(oracle):
    """Transposing the volume's depth and height axes together with the window and the table's axes transposes the
    result.  Catches: an axis handled differently from the others (padding, shift, index stride)."""
    r = rng(952)
    win, s = (2, 3, 2), (1, 2, 0)
    x = r.standard_normal((2, 2, 5, 7, 4))
    T = r.standard_normal((2, 3 * 5 * 3))
    y = oracle.forward_3d(x, T, win, s)
    xt = np.ascontiguousarray(x.transpose(0, 1, 3, 2, 4))
    Tt = np.ascontiguousarray(T.reshape(2, 3, 5, 3).transpose(0, 2, 1, 3)).reshape(2, -1)
    yt = oracle.forward_3d(xt, Tt, (3, 2, 2), (2, 1, 0))
    assert np.allclose(y, yt.transpose(0, 1, 3, 2, 4), rtol=0, atol=1e-12)


def test_3d_padding_shift_and_window_independence(oracle):
    """Explicit zero padding + roll + per-window conv3d + roll back + crop (library pieces) equals the operator."""
    r = rng(953)
    win, s = (2, 3, 2), (1, 1, 1)
    B, C, D, H, W = 1, 2, 3, 7, 5
    x = r.standard_normal((B, C, D, H, W))
    T = r.standard_normal((C, 3 * 5 * 3))
    Dp, Hp, Wp = 4, 9, 6
    xp = np.zeros((B, C, Dp, Hp, Wp))
    xp[:, :, :D, :H, :W] = x
    xh = np.roll(xp, (-s[0], -s[1], -s[2]), axis=(2, 3, 4))
    yh = np.zeros_like(xh)
    K = torch.flip(torch.from_numpy(T.reshape(C, 1, 3, 5, 3)), dims=(2, 3, 4))
    for z0 in range(0, Dp, 2):
        for h0 in range(0, Hp, 3):
            for v0 in range(0, Wp, 2):
                blk = torch.from_numpy(np.ascontiguousarray(xh[:, :, z0:z0 + 2, h0:h0 + 3, v0:v0 + 2]))
                yh[:, :, z0:z0 + 2, h0:h0 + 3, v0:v0 + 2] = F.conv3d(blk, K, padding=(1, 2, 1), groups=C).numpy()
    want = np.roll(yh, s, axis=(2, 3, 4))[:, :, :D, :H, :W]
    assert np.allclose(oracle.forward_3d(x, T, win, s), want, rtol=0, atol=1e-12)


@pytest.mark.parametrize("layout", [NCHW, NHWC])
def test_3d_backward_adjoint_and_one_hot_derivative(oracle, layout):
    """<dy, WBMM(x2;T)> = <dX, x2>, <dT, T2> = <dy, WBMM(x;T2)> (the operator is bilinear), and dT along a one-hot
    table direction is the derivative of the pinned forward.  Catches: dX built from W instead of W^T, a bin offset."""
    r = rng(954)
    win, s = (2, 2, 3), (1, 0, 2)
    shape = (2, 3, 3, 5, 7) if layout == NCHW else (2, 3, 5, 7, 3)
    x, x2, dy = (r.standard_normal(shape) for _ in range(3))
    nb = 3 * 3 * 5
    T, T2 = r.standard_normal((3, nb)), r.standard_normal((3, nb))
    dx, dT = oracle.backward_3d(x, T, dy, win, s, layout)
    assert np.isclose(np.sum(dy * oracle.forward_3d(x2, T, win, s, layout)), np.sum(dx * x2), rtol=1e-12)
    assert np.isclose(np.sum(dT * T2), np.sum(dy * oracle.forward_3d(x, T2, win, s, layout)), rtol=1e-12)
    for (c, k) in [(0, 0), (1, nb // 2), (2, nb - 1), (1, 7)]:
        E = np.zeros((3, nb))
        E[c, k] = 1.0
        assert np.isclose(dT[c, k], np.sum(dy * oracle.forward_3d(x, E, win, s, layout)), rtol=1e-12, atol=1e-12)
