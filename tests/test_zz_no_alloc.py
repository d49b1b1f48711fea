"""wbmm_forward_static_scratch: the NHWC transposition route with its temporaries in a file-scope device array
(no allocation in the call).  Checked against the existing path (wbmm_forward) on calls made back to back.
This file sorts last on purpose: it is collected after every other test."""
import pytest
import torch

import synth_inputs as si
from parity import TOL, max_err_over_tol, widen

pytestmark = pytest.mark.gpu

NHWC = si.NHWC


@pytest.fixture(scope="module")
def wb():
    import paper_2607_02097_b200 as wb
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    wb.wbmm_version()          # loads libwbmm.so or raises: no silent fallback
    return wb


CASES = [
    si.Case("ss_w14_shift", 6, 16, 28, 56, 14, shift=(7, 3), layout=NHWC, seed=601),
    si.Case("ss_w14_ragged_small", 3, 24, 60, 60, 14, layout=NHWC, seed=602),        # smaller: stale bytes lie behind it
    si.Case("ss_w7_f16", 9, 32, 28, 28, 7, dtype="f16", shift=(3, 2), layout=NHWC, seed=603),
    si.Case("ss_near_limit", 16, 96, 56, 56, 14, layout=NHWC, seed=604),             # 9.6 MB of the 16 MiB
]


def test_static_scratch_matches_the_existing_path_on_calls_in_a_row(wb):
    """Several calls in a row on one stream, different shapes, then the first shape again: each result equals what
    wbmm_forward gives for the same inputs (same kernels on the w = 14 shapes: bitwise; w = 7 takes the one-pass
    kernel in wbmm_forward: within the 16-bit tolerance of the parity tests)."""
    data = [si.make(c, device="cuda") for c in CASES]
    refs, ref_paths = [], []
    for c, d in zip(CASES, data):
        refs.append(wb.wbmm_forward(d["x"], d["T"], c.w, c.shift, c.layout))
        ref_paths.append(wb.wbmm_last_path())
    outs = [torch.full_like(d["x"], 7.0) for d in data]
    torch.cuda.synchronize()
    order = [0, 1, 2, 3, 0, 0, 1]
    for k, i in enumerate(order):
        c, d = CASES[i], data[i]
        outs[i].fill_(7.0)
        y = wb.wbmm_forward_static_scratch(d["x"], d["T"], c.w, c.shift, out=outs[i])
        assert wb.wbmm_last_path() == wb.PATH_TC_TRANSPOSED
        torch.cuda.synchronize()
        assert max_err_over_tol(y, widen(refs[i]), TOL[c.dtype]) <= 1.0, (k, c.name)
        if ref_paths[i] == wb.PATH_TC_TRANSPOSED:
            assert torch.equal(y, refs[i]), (k, c.name)


def test_static_scratch_call_allocates_no_device_memory(wb):
    """Free device memory does not drop across a call (the kernels' modules are loaded by a first call)."""
    c = CASES[0]
    d = si.make(c, device="cuda")
    out = torch.empty_like(d["x"])
    wb.wbmm_forward_static_scratch(d["x"], d["T"], c.w, c.shift, out=out)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        wb.wbmm_forward_static_scratch(d["x"], d["T"], c.w, c.shift, out=out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, (free0, free1)


def test_static_scratch_rejects_what_it_cannot_hold(wb):
    big = si.Case("ss_too_large", 32, 96, 56, 56, 14, layout=NHWC, seed=605)         # 19.3 MB > 16 MiB
    d = si.make(big, device="cuda")
    out = torch.full_like(d["x"], 7.0)
    n0 = wb.wbmm_launch_count()
    with pytest.raises(wb.WbmmError) as ei:
        wb.wbmm_forward_static_scratch(d["x"], d["T"], big.w, big.shift, out=out)
    assert ei.value.status == wb.STATUS_TOO_LARGE and "static scratch" in str(ei.value)
    torch.cuda.synchronize()
    assert wb.wbmm_launch_count() == n0 and bool((out == 7.0).all())                 # nothing launched, nothing written
    # not a problem of the transposition route (fp32; C not a multiple of 8): unsupported, nothing launched
    x = torch.zeros((2, 14, 14, 8), dtype=torch.float32, device="cuda")
    with pytest.raises(wb.WbmmError) as ei:
        wb.wbmm_forward_static_scratch(x, torch.zeros((8, 729), dtype=torch.float32, device="cuda"), 14)
    assert ei.value.status == 2
    x = torch.zeros((2, 28, 28, 12), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(wb.WbmmError) as ei:
        wb.wbmm_forward_static_scratch(x, torch.zeros((12, 729), dtype=torch.bfloat16, device="cuda"), 14)
    assert ei.value.status == 2
    assert wb.wbmm_launch_count() == n0
