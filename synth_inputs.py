"""Seeded synthetic inputs for the WBMM operator (shared by tests and bench.py).

This module holds NONE of the method's arithmetic: it only draws random tensors
of the shapes, distributions and seeds DESIGN.md ("Input recipe") states, which stand
in for the paper's operator benchmark (batch 4-256, maps >= 28x28,
windows 7x7 and 14x14; BASELINE.json configs 1-5).  Neither oracle/ nor the CUDA
path imports the other; both are fed from here.

Recipe: torch.Generator(device="cpu").manual_seed(seed); draw order x, T, dy (fp32,
logical NCHW); x ~ N(0,1), T ~ N(0, 0.02^2), dy ~ N(0,1); cast (RNE) to the case dtype;
NHWC cases are permute(0,2,3,1).contiguous() of the same logical NCHW draw.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Iterator, Tuple

import torch

NCHW, NHWC = 0, 1
TORCH_DTYPES = {"f32": torch.float32, "bf16": torch.bfloat16, "f16": torch.float16}


@dataclass(frozen=True)
class Case:
    name: str
    B: int
    C: int
    H: int
    W: int
    w: int
    dtype: str = "bf16"            # "f32" | "bf16" | "f16"
    layout: int = NCHW
    shift: Tuple[int, int] = (0, 0)
    seed: int = 0
    backward: bool = False
    table: str = "normal"          # "normal" | "structured" (diagonal-dominant, fast decay)

    @property
    def n_elem(self) -> int:
        return self.B * self.C * self.H * self.W

    @property
    def bins(self) -> int:
        return (2 * self.w - 1) ** 2

    def shape(self):
        if self.layout == NCHW:
            return (self.B, self.C, self.H, self.W)
        return (self.B, self.H, self.W, self.C)


# BASELINE.json "configs" (1-based numbering as in SURVEY.md section 8(d)).
CFG1 = Case("cfg1_tiny_f32", 1, 4, 14, 14, 7, dtype="f32", seed=0)
CFG2 = Case("cfg2_w7_bf16", 64, 96, 56, 56, 7, seed=1)
CFG3 = Case("cfg3_w14_bf16_headline", 128, 96, 56, 56, 14, seed=2)
CFG5 = Case("cfg5_train_shift", 128, 192, 28, 28, 14, shift=(7, 7), seed=9, backward=True)


def sweep_cases() -> Iterator[Case]:
    """Config 4: layout x B x (C,H) x w = 80 cases, then the ragged 60x60 pair; seed 3+index."""
    idx = 0
    for layout in (NCHW, NHWC):
        for B in (4, 16, 64, 128, 256):
            for (C, H) in ((96, 56), (192, 28), (384, 28), (96, 112)):
                for w in (7, 14):
                    lay = "nchw" if layout == NCHW else "nhwc"
                    yield Case(f"cfg4_{lay}_B{B}_C{C}_H{H}_w{w}", B, C, H, H, w,
                               layout=layout, seed=3 + idx)
                    idx += 1
    for layout in (NCHW, NHWC):
        lay = "nchw" if layout == NCHW else "nhwc"
        yield Case(f"cfg4_{lay}_ragged_B64_C96_H60_w14", 64, 96, 60, 60, 14,
                   layout=layout, seed=3 + idx)
        idx += 1


def with_(case: Case, **kw) -> Case:
    return replace(case, **kw)


def make(case: Case, device: str = "cpu", pin: bool = False):
    """Returns dict(x=, T=, dy= or None) of torch tensors in the case dtype and layout."""
    g = torch.Generator(device="cpu").manual_seed(case.seed)
    dt = TORCH_DTYPES[case.dtype]
    x = torch.randn((case.B, case.C, case.H, case.W), generator=g, dtype=torch.float32)
    if case.table == "normal":
        T = torch.randn((case.C, case.bins), generator=g, dtype=torch.float32) * 0.02
    else:
        # diagonal-dominant, fast spatial decay (the shape PAPER.md:559 reports for learned M)
        tw = 2 * case.w - 1
        r = torch.arange(tw, dtype=torch.float32) - (case.w - 1)
        dist = (r[:, None] ** 2 + r[None, :] ** 2).sqrt()
        amp = 0.5 + torch.rand((case.C, 1, 1), generator=g)
        T = (amp * torch.exp(-dist / 1.5)[None] +
             0.002 * torch.randn((case.C, tw, tw), generator=g)).reshape(case.C, case.bins)
    dy = torch.randn((case.B, case.C, case.H, case.W), generator=g,
                     dtype=torch.float32) if case.backward else None

    def fin(t, act):
        if t is None:
            return None
        t = t.to(dt)
        if act and case.layout == NHWC:
            t = t.permute(0, 2, 3, 1).contiguous()
        if pin:
            t = t.pin_memory()
        return t.to(device) if device != "cpu" else t

    return {"x": fin(x, True), "T": fin(T, False), "dy": fin(dy, True)}


def make_int8(case: Case, device: str = "cpu", extreme: bool = False):
    """dict(x=, T=, scale=) for the INT8 forward: activations as symmetric 8-bit quantisation of a normal map
    (round(x / 3 sigma * 127), clipped), the table likewise from the case's table recipe, per-channel float32
    requantisation scales that put the sums' spread at about a third of the int8 range.  extreme: a few -128 / 127
    runs and one all -128 table row (the largest products)."""
    f = make(with_(case, dtype="f32", layout=NCHW), device="cpu")
    x = torch.clamp(torch.round(f["x"] / 3.0 * 127.0), -128, 127).to(torch.int8)
    T = f["T"]
    T = torch.clamp(torch.round(T / T.abs().amax(dim=1, keepdim=True) * 127.0), -128, 127).to(torch.int8)
    if extreme:
        x.view(-1)[: min(x.numel(), 3 * case.w * case.w)] = -128
        x.view(-1)[-min(x.numel(), 2 * case.w * case.w):] = 127
        T[0, :] = -128
        if case.C > 1:
            T[1, :] = 127
    g = torch.Generator(device="cpu").manual_seed(case.seed + 77)
    sigma = 42.0 * 42.0 * case.w                       # ~ std of a sum of w*w products of such values
    scale = (40.0 / sigma) * (0.5 + torch.rand((case.C,), generator=g, dtype=torch.float32))
    if case.layout == NHWC:
        x = x.permute(0, 2, 3, 1).contiguous()
    if device != "cpu":
        x, T, scale = x.to(device), T.to(device), scale.to(device)
    return {"x": x, "T": T, "scale": scale}


def make_fp8(case: Case, device: str = "cpu"):
    """dict(x=, T=, scale=) for the FP8 forward: the case's normal activations and table recipe (table scaled to unit
    row maximum) rounded to E4M3 by torch's conversion, per-channel float32 scales that put sum * scale at O(1-100)."""
    f = make(with_(case, dtype="f32", layout=NCHW), device="cpu")
    x = f["x"].to(torch.float8_e4m3fn)
    T = f["T"]
    T = (T / T.abs().amax(dim=1, keepdim=True)).to(torch.float8_e4m3fn)
    g = torch.Generator(device="cpu").manual_seed(case.seed + 78)
    scale = (32.0 / case.w) * (0.5 + torch.rand((case.C,), generator=g, dtype=torch.float32))
    if case.layout == NHWC:
        x = x.permute(0, 2, 3, 1).contiguous()
    if device != "cpu":
        x, T, scale = x.to(device), T.to(device), scale.to(device)
    return {"x": x, "T": T, "scale": scale}
