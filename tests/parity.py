"""Helpers for the GPU-vs-oracle parity tests (tests only; imports oracle/ and the binding)."""
from __future__ import annotations

import numpy as np
import torch

import synth_inputs as si

# Tolerances (BASELINE.json north_star): |y - y_ref| <= tol * (1 + |y_ref|)
TOL = {"f32": 1e-4, "bf16": 1e-2, "f16": 1e-2}


def widen(t: torch.Tensor) -> np.ndarray:
    """Case-dtype tensor -> float64 numpy (the oracle sees exactly the rounded values)."""
    return t.detach().cpu().to(torch.float64).numpy()


def max_err_over_tol(got: torch.Tensor, ref: np.ndarray, tol: float) -> float:
    g = widen(got)
    assert g.shape == ref.shape, (g.shape, ref.shape)
    if g.size == 0:
        return 0.0
    assert np.isfinite(g).all(), "non-finite output"
    return float(np.max(np.abs(g - ref) / (tol * (1.0 + np.abs(ref)))))


def plane_subset(case: si.Case, nb: int, nc: int, seed: int = 1234):
    """Seeded sample of images and channels (full planes) for full-size cases."""
    r = np.random.default_rng(seed)
    bs = np.sort(r.choice(case.B, size=min(nb, case.B), replace=False))
    cs = np.sort(r.choice(case.C, size=min(nc, case.C), replace=False))
    return torch.from_numpy(bs), torch.from_numpy(cs)


def take_planes(t: torch.Tensor, layout: int, bs, cs) -> torch.Tensor:
    t = t.cpu()
    if bs is not None:
        t = t.index_select(0, bs)
    if cs is not None:
        t = t.index_select(1 if layout == si.NCHW else 3, cs)
    return t.contiguous()
