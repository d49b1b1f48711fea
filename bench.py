#!/usr/bin/env python
"""bench.py -- WBMM forward on the headline workload (BASELINE.json config 3:
B=128, C=96, 56x56, w=14, bf16 in / fp32 accumulate / bf16 out, NCHW), one B200 per rank.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl wbmm|reference]

A "step" is one pass of the whole hot path (relative index -> W_c in shared memory -> window
loads -> contraction -> un-partition/store) over one batch, i.e. one
wbmm_forward call through the C ABI.  Prints ONE JSON line (rank 0).

  value      TFLOP/s = algorithmic FLOPs (2*N per activation element, N=w*w=196, unpadded) of all
             ranks / max-over-ranks device time, inputs resident in HBM.
  e2e        the same metric through wbmm_forward_host (pinned HOST buffers; H2D + kernels + D2H
             inside the timed region).
  roofline   HBM-bound: algorithmic bytes (read x once + write y once + the table) / kernel time,
             against MEASURED_PEAKS.json (else the profiling guide's fallback 6650 GB/s).
  cpu_baseline  the CPU oracle (oracle/wbmm_ref.c, direct form, fp64, OpenMP) on a bounded sample
             of the same workload, on this box's host cores.  A baseline, not the target.
  train_step    config 5 (B=128, C=192, 28x28, w=14, shift 7: forward + dX + dT) ms, as context.

`--impl reference` times the oracle itself (there is no reference code).
Multi-GPU: the operator shards by batch with no exchange in the forward pass -> weak scaling,
each rank runs the full config-3 batch on its own GPU.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

import synth_inputs as si  # noqa: E402

METRIC = "wbmm_fwd_tflops_B128_C96_56x56_w14_bf16"
UNIT = "TFLOP/s"
FALLBACK_HBM_GBS = 6650.0      # /opt/skills/guides/B200_PROFILING.md fallback
L2_BYTES = 126e6


def flops_of(case: si.Case) -> float:
    Hp = -(-case.H // case.w) * case.w
    Wp = -(-case.W // case.w) * case.w
    return 2.0 * case.w * case.w * case.B * case.C * Hp * Wp


def bytes_of(case: si.Case) -> float:
    es = 4 if case.dtype == "f32" else 2
    return 2.0 * es * case.n_elem + es * case.C * case.bins


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), float(d.get("bf16_tflops", 1590.0)), "measured"
    return FALLBACK_HBM_GBS, 1590.0, "fallback"


def ncu_traffic_bytes():
    """dram bytes per launch of the headline kernel from the committed ncu capture, or None."""
    p = os.path.join(ROOT, "profiles", "headline_traffic.txt")
    if not os.path.exists(p):
        return None
    for line in open(p):
        line = line.split("#")[0].strip()
        if line.startswith("dram_bytes_per_launch"):
            return float(line.split("=")[1])
        if line.isdigit():  # a bare number is the same figure
            return float(line)
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons, sampled while the GPU is under load."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        for ts, line in self.rows:
            if ts < t0 or ts > t1 + 0.06:
                continue
            f = [s.strip() for s in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def dist_setup(n_gpus: int):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl" if torch.cuda.is_available() else "gloo")
    return rank, world, local


def barrier(world):
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(v: float, world: int, device) -> float:
    if world == 1:
        return v
    import torch.distributed as dist
    t = torch.tensor([v], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


# ------------------------------------------------------------------------------- oracle timing
def oracle_probe(case: si.Case):
    """Seconds per image of the oracle (direct form) on this box, measured on 2 images."""
    from oracle import wbmm_ref
    d = si.make(si.with_(case, B=2))
    x2, T = d["x"].double().numpy(), d["T"].double().numpy()
    wbmm_ref.forward(x2[:1], T, case.w, case.shift, case.layout, "direct")     # page-in, thread pool
    t0 = time.perf_counter()
    wbmm_ref.forward(x2, T, case.w, case.shift, case.layout, "direct")
    return (time.perf_counter() - t0) / 2, T


def oracle_sample(case: si.Case, target_s: float, per_image: float):
    nb = int(max(1, min(case.B, target_s / max(per_image, 1e-6))))
    sub = si.with_(case, B=nb)
    return sub, si.make(sub)["x"].double().numpy(), \
        f"first {nb} of {case.B} images, all {case.C} channels, direct form fp64"


def time_oracle(case: si.Case, target_s: float = 12.0):
    """The oracle as it stands (direct form, fp64, OpenMP over (b,c) planes) on a bounded sample
    of `case`.  Returns (TFLOP/s, cores, sample, seconds)."""
    from oracle import wbmm_ref
    per_image, T = oracle_probe(case)
    sub, xs, sample = oracle_sample(case, target_s, per_image)
    t0 = time.perf_counter()
    wbmm_ref.forward(xs, T, case.w, case.shift, case.layout, "direct")
    dt = time.perf_counter() - t0
    return flops_of(sub) / dt / 1e12, wbmm_ref.num_threads(), sample, dt


def oracle_legs(case3: si.Case, case5: si.Case, budget_s: float = 4.0):
    """BASELINE.md section 3 context rows, each on a bounded sample: the oracle on ONE core, the matrix form
    (Alg. 1 with a materialised M) on config 3, and the config-5 training step (forward + dX + dT)."""
    from oracle import wbmm_ref
    out = {}
    ncores = wbmm_ref.num_threads()
    per_image, T = oracle_probe(case3)           # all cores
    # one core
    nb1 = int(max(1, min(case3.B, budget_s / max(per_image * ncores, 1e-6))))
    sub = si.with_(case3, B=nb1)
    xs = si.make(sub)["x"].double().numpy()
    wbmm_ref.set_threads(1)
    t0 = time.perf_counter()
    wbmm_ref.forward(xs, T, case3.w, case3.shift, case3.layout, "direct")
    dt = time.perf_counter() - t0
    wbmm_ref.set_threads(ncores)
    out["cfg3_direct_1core"] = {"value": flops_of(sub) / dt / 1e12, "unit": UNIT, "cores": 1, "seconds": dt,
                                "sample": f"first {nb1} of {case3.B} images, all {case3.C} channels"}
    # matrix form, all cores
    nbm = int(max(1, min(case3.B, budget_s / max(per_image, 1e-6))))
    sub = si.with_(case3, B=nbm)
    xs = si.make(sub)["x"].double().numpy()
    t0 = time.perf_counter()
    wbmm_ref.forward(xs, T, case3.w, case3.shift, case3.layout, "matrix")
    dt = time.perf_counter() - t0
    out["cfg3_matrix_form"] = {"value": flops_of(sub) / dt / 1e12, "unit": UNIT, "cores": ncores, "seconds": dt,
                               "sample": f"first {nbm} of {case3.B} images, all {case3.C} channels"}
    # config 5: forward + backward (dX, dT), all cores
    per5, T5 = oracle_probe(case5)
    nb5 = int(max(1, min(case5.B, budget_s / max(3 * per5, 1e-6))))
    sub = si.with_(case5, B=nb5)
    d = si.make(sub)
    x5, g5 = d["x"].double().numpy(), d["dy"].double().numpy()
    t0 = time.perf_counter()
    wbmm_ref.forward(x5, T5, case5.w, case5.shift, case5.layout, "direct")
    wbmm_ref.backward(x5, T5, g5, case5.w, case5.shift, case5.layout)
    dt = time.perf_counter() - t0
    out["cfg5_fwd_bwd"] = {"ms": dt * 1e3, "value": 3 * flops_of(sub) / dt / 1e12, "unit": UNIT, "cores": ncores,
                           "sample": f"first {nb5} of {case5.B} images, all {case5.C} channels, forward + dX + dT"}
    return out


def run_reference(args, rank, world):
    """--impl reference: the paper ships no code, so the reference arm is the CPU oracle, timed as
    it stands on this box's host cores; each step is a bounded sample of config 3."""
    if rank != 0:
        return
    from oracle import wbmm_ref
    case = si.CFG3
    per_image, T = oracle_probe(case)
    per_step = max(0.05, min(15.0, args.ref_seconds / max(1, args.steps + args.warmup)))
    sub, xs, sample = oracle_sample(case, per_step, per_image)
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        wbmm_ref.forward(xs, T, case.w, case.shift, case.layout, "direct")
        if i >= args.warmup:
            times.append(time.perf_counter() - t0)
    dt = sum(times) / len(times)
    value = flops_of(sub) / dt / 1e12
    cores = wbmm_ref.num_threads()
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "cfg3: B=128 C=96 H=W=56 w=14 NCHW (bounded sample per step)", "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)


# ------------------------------------------------------------------------------- GPU timing
def time_steps(fn, n, stream):
    """n calls of fn(i), each bracketed by CUDA events on `stream`; returns per-step ms list."""
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
    for i in range(n):
        evs[i][0].record(stream)
        fn(i)
        evs[i][1].record(stream)
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in evs]


def conv_context(case: si.Case, x):
    """Same-run torch depthwise conv (cuDNN as shipped) at k=5/7/13: context only."""
    out = {}
    try:
        for k in (5, 7, 13):
            wgt = torch.randn(case.C, 1, k, k, device=x.device, dtype=x.dtype) * 0.02
            f = lambda: torch.nn.functional.conv2d(x, wgt, padding=k // 2, groups=case.C)
            for _ in range(3):
                f()
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(5):
                f()
            b.record()
            torch.cuda.synchronize()
            out[f"torch_dwconv_k{k}_ms"] = round(a.elapsed_time(b) / 5, 4)
    except Exception as e:  # context only
        out["error"] = str(e)[:100]
    return out


def region_ms_rot(fn, n, stream, warm=3):
    """Average device ms of n back-to-back calls fn(i) (i rotates the buffer set), CUDA events on `stream`."""
    for i in range(warm):
        fn(i)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for i in range(n):
        fn(warm + i)
    b.record(stream)
    torch.cuda.synchronize()
    return a.elapsed_time(b) / n


def buffer_sets(per_set_bytes: float, cap: int = 8) -> int:
    """Enough buffer sets that the rotating footprint exceeds 2 x L2 (cold-L2 numbers)."""
    return int(max(2, min(cap, -(-2 * L2_BYTES // per_set_bytes) + 1)))


def other_rooflines(wb, dev, stream, hbm_peak):
    """Roofline fractions of the other kernels / configs, measured in the same run with rotating buffers (cold L2):
    algorithmic bytes (read the inputs once, write the outputs once, + the table) / average launch duration."""
    out = {}

    def fwd_row(name, case, n=30):
        d = si.make(case, device=dev)
        es = 4 if case.dtype == "f32" else 2
        ns = buffer_sets(2.0 * case.n_elem * es)
        xs = [d["x"]] + [d["x"].clone() for _ in range(ns - 1)]
        ys = [torch.empty_like(d["x"]) for _ in range(ns)]
        ms = region_ms_rot(lambda i: wb.wbmm_forward(xs[i % ns], d["T"], case.w, case.shift, case.layout, out=ys[i % ns]), n, stream)
        by = bytes_of(case)
        out[name] = {"ms": round(ms, 5), "gbs": round(by / ms / 1e6, 1), "frac": round(by / (hbm_peak * 1e9) * 1e3 / ms, 4),
                     "path": wb.wbmm_path_string(wb.wbmm_last_path()), "buffer_sets": ns}
        del xs, ys, d
        torch.cuda.empty_cache()

    fwd_row("cfg2_fwd_w7", si.CFG2)
    fwd_row("cfg5_fwd_shift7", si.with_(si.CFG5, backward=False))
    fwd_row("ragged_B64_C96_60x60_w14_fwd", si.Case("ragged", 64, 96, 60, 60, 14, seed=85))
    fwd_row("nhwc_cfg3_shape_fwd", si.with_(si.CFG3, layout=si.NHWC))
    fwd_row("nhwc_cfg2_shape_fwd_w7", si.with_(si.CFG2, layout=si.NHWC))
    fwd_row("fp32_B128_C96_56x56_w14_fwd", si.with_(si.CFG3, dtype="f32"), n=10)
    fwd_row("fp32_B128_C96_56x56_w7_fwd", si.Case("f32w7", 128, 96, 56, 56, 7, dtype="f32", seed=86), n=10)
    # small planes (the paper's S3 / S4 stages and a 30 x 30 map): plane boxes; launch-latency-bound
    fwd_row("s3_B128_C256_14x14_w14_fwd", si.Case("s3w14", 128, 256, 14, 14, 14, seed=88))
    fwd_row("s4_B128_C256_7x7_w7_fwd", si.Case("s4w7", 128, 256, 7, 7, 7, seed=90))
    fwd_row("B64_C96_30x30_w14_fwd", si.Case("r30", 64, 96, 30, 30, 14, seed=92))

    # backward of config 5, each kernel alone, rotating (x, dy, dx) sets
    c5 = si.CFG5
    d = si.make(c5, device=dev)
    ns = buffer_sets(3.0 * c5.n_elem * 2)
    xs = [d["x"]] + [d["x"].clone() for _ in range(ns - 1)]
    gs = [d["dy"]] + [d["dy"].clone() for _ in range(ns - 1)]
    dxs = [torch.empty_like(d["x"]) for _ in range(ns)]
    dT = torch.empty((c5.C, c5.bins), dtype=torch.float32, device=dev)
    by = bytes_of(c5)
    ms = region_ms_rot(lambda i: wb.wbmm_backward(None, d["T"], gs[i % ns], c5.w, c5.shift, need_dT=False, dx=dxs[i % ns]), 30, stream)
    out["cfg5_dX"] = {"ms": round(ms, 5), "frac": round(by / (hbm_peak * 1e9) * 1e3 / ms, 4), "buffer_sets": ns}
    ms = region_ms_rot(lambda i: wb.wbmm_backward(xs[i % ns], None, gs[i % ns], c5.w, c5.shift, need_dx=False, dT=dT), 30, stream)
    out["cfg5_dT"] = {"ms": round(ms, 5), "frac": round(by / (hbm_peak * 1e9) * 1e3 / ms, 4), "buffer_sets": ns,
                      "note": "includes the dT zeroing launch"}
    del xs, gs, dxs, d
    torch.cuda.empty_cache()

    fwd_row("fp32_nhwc_B128_C96_56x56_w14_fwd", si.with_(si.CFG3, dtype="f32", layout=si.NHWC), n=5)

    # rectangular windows 7 x 14 (FFMA kernels, section 7.10 of DESIGN.md) on the config-2 shape: context
    cr = si.CFG2
    dr = si.make(cr, device=dev)
    Tr = (torch.randn((cr.C, 13 * 27), generator=torch.Generator().manual_seed(93)) * 0.02).to(dr["x"].dtype).to(dev)
    yr = torch.empty_like(dr["x"])
    ms = region_ms_rot(lambda i: wb.wbmm_forward_rect(dr["x"], Tr, 7, 14, out=yr), 5, stream)
    out["rect_7x14_B64_C96_56x56_fwd"] = {"ms": round(ms, 5), "tflops": round(2.0 * 98 * cr.n_elem / ms / 1e9, 2),
                                         "frac": round(bytes_of(cr) / (hbm_peak * 1e9) * 1e3 / ms, 4),
                                         "path": wb.wbmm_path_string(wb.wbmm_last_path())}
    del dr, Tr, yr
    torch.cuda.empty_cache()

    # 3-D windows 2 x 7 x 7 (the FFMA kernels with a depth axis, section 7.10 of DESIGN.md) on a video-shaped volume: context
    g3 = torch.Generator().manual_seed(94)
    x3 = torch.randn((16, 96, 8, 56, 56), generator=g3).to(torch.bfloat16).to(dev)
    T3 = (torch.randn((96, 3 * 13 * 13), generator=g3) * 0.02).to(torch.bfloat16).to(dev)
    y3 = torch.empty_like(x3)
    ms = region_ms_rot(lambda i: wb.wbmm_forward_win3d(x3, T3, (2, 7, 7), out=y3), 5, stream)
    out["win3d_2x7x7_B16_C96_8x56x56_fwd"] = {"ms": round(ms, 5), "tflops": round(2.0 * 98 * x3.numel() / ms / 1e9, 2),
                                             "frac": round(4.0 * x3.numel() / (hbm_peak * 1e9) * 1e3 / ms, 4),
                                             "path": wb.wbmm_path_string(wb.wbmm_last_path())}
    del x3, T3, y3
    torch.cuda.empty_cache()

    # INT8 forward (tcgen05 kind::i8, section 7.11 of DESIGN.md) on the shapes of configs 3 and 2: int8 in, int8 out
    # (requantised): 2 bytes per element of algorithmic traffic; int32 out: 5 bytes
    for ci in (si.with_(si.CFG3, backward=False), si.with_(si.CFG2, backward=False)):
        name = f"int8_B{ci.B}_C{ci.C}_{ci.H}x{ci.W}_w{ci.w}_fwd"
        d8 = si.make_int8(ci, device=dev)
        ns = buffer_sets(2.0 * ci.n_elem)
        xs = [d8["x"]] + [d8["x"].clone() for _ in range(ns - 1)]
        y8 = [torch.empty_like(d8["x"]) for _ in range(ns)]
        ms = region_ms_rot(lambda i: wb.wbmm_forward_int8(xs[i % ns], d8["T"], ci.w, scale=d8["scale"], out=y8[i % ns]), 30, stream)
        by8 = 2.0 * ci.n_elem + ci.C * ci.bins + 4 * ci.C
        out[name] = {"ms": round(ms, 5), "gbs": round(by8 / ms / 1e6, 1), "frac": round(by8 / (hbm_peak * 1e9) * 1e3 / ms, 4),
                     "tops": round(2.0 * ci.w * ci.w * ci.n_elem / ms / 1e9, 2), "path": wb.wbmm_path_string(wb.wbmm_last_path()),
                     "buffer_sets": ns}
        y32 = [torch.empty(d8["x"].shape, dtype=torch.int32, device=dev) for _ in range(2)]
        ms = region_ms_rot(lambda i: wb.wbmm_forward_int8(xs[i % ns], d8["T"], ci.w, out=y32[i % 2]), 10, stream)
        out[name.replace("_fwd", "_fwd_int32_out")] = {"ms": round(ms, 5), "frac": round((5.0 * ci.n_elem) / (hbm_peak * 1e9) * 1e3 / ms, 4)}
        del xs, y8, y32, d8
        torch.cuda.empty_cache()
        # FP8 (E4M3 in, E4M3 out with per-channel scale) on the same kernels (kind::f8f6f4)
        f8 = si.make_fp8(ci, device=dev)
        xs = [f8["x"]] + [f8["x"].clone() for _ in range(ns - 1)]
        yf = [torch.empty_like(f8["x"]) for _ in range(ns)]
        ms = region_ms_rot(lambda i: wb.wbmm_forward_fp8(xs[i % ns], f8["T"], ci.w, scale=f8["scale"], out=yf[i % ns]), 30, stream)
        out[name.replace("int8_", "fp8_")] = {"ms": round(ms, 5), "gbs": round(by8 / ms / 1e6, 1), "frac": round(by8 / (hbm_peak * 1e9) * 1e3 / ms, 4),
                                              "tflops": round(2.0 * ci.w * ci.w * ci.n_elem / ms / 1e9, 2),
                                              "path": wb.wbmm_path_string(wb.wbmm_last_path()), "buffer_sets": ns}
        del xs, yf, f8
        torch.cuda.empty_cache()

    # INT8 on config 5's shape with its shift (7, 7): the gather kernel's rotated-window form
    c5i = si.with_(si.CFG5, backward=False)
    d8 = si.make_int8(c5i, device=dev)
    ns = buffer_sets(2.0 * c5i.n_elem)
    xs = [d8["x"]] + [d8["x"].clone() for _ in range(ns - 1)]
    y8 = [torch.empty_like(d8["x"]) for _ in range(ns)]
    ms = region_ms_rot(lambda i: wb.wbmm_forward_int8(xs[i % ns], d8["T"], c5i.w, c5i.shift, scale=d8["scale"], out=y8[i % ns]), 20, stream)
    out["int8_cfg5_shape_shift7_fwd"] = {"ms": round(ms, 5), "frac": round(2.0 * c5i.n_elem / (hbm_peak * 1e9) * 1e3 / ms, 4),
                                        "path": wb.wbmm_path_string(wb.wbmm_last_path()), "buffer_sets": ns}
    del xs, y8, d8
    torch.cuda.empty_cache()

    # table gradient at w = 7 (two CTAs per SM) on the config-2 shape
    c2 = si.with_(si.CFG2, backward=True)
    d = si.make(c2, device=dev)
    ns = buffer_sets(2.0 * c2.n_elem * 2)
    xs = [d["x"]] + [d["x"].clone() for _ in range(ns - 1)]
    gs = [d["dy"]] + [d["dy"].clone() for _ in range(ns - 1)]
    dT = torch.empty((c2.C, c2.bins), dtype=torch.float32, device=dev)
    ms = region_ms_rot(lambda i: wb.wbmm_backward(xs[i % ns], None, gs[i % ns], c2.w, c2.shift, need_dx=False, dT=dT), 30, stream)
    out["cfg2_shape_dT_w7"] = {"ms": round(ms, 5), "frac": round(bytes_of(c2) / (hbm_peak * 1e9) * 1e3 / ms, 4), "buffer_sets": ns,
                               "path": wb.wbmm_path_string(wb.wbmm_last_path()), "note": "includes the dT zeroing launch"}
    del xs, gs, d
    torch.cuda.empty_cache()

    # float32 table gradient (3-way / 2-way bf16 split on the tensor cores): reads x and dy once
    for name, cf in (("fp32_B128_C96_56x56_w14_dT", si.with_(si.CFG3, dtype="f32", backward=True)),
                     ("fp32_B128_C96_56x56_w7_dT", si.Case("f32w7", 128, 96, 56, 56, 7, dtype="f32", backward=True, seed=86))):
        d = si.make(cf, device=dev)
        ns = buffer_sets(2.0 * cf.n_elem * 4)
        xs = [d["x"]] + [d["x"].clone() for _ in range(ns - 1)]
        gs = [d["dy"]] + [d["dy"].clone() for _ in range(ns - 1)]
        dT = torch.empty((cf.C, cf.bins), dtype=torch.float32, device=dev)
        ms = region_ms_rot(lambda i: wb.wbmm_backward(xs[i % ns], None, gs[i % ns], cf.w, cf.shift, need_dx=False, dT=dT), 10, stream)
        by = 2 * cf.n_elem * 4 + cf.C * cf.bins * 4
        out[name] = {"ms": round(ms, 5), "gbs": round(by / ms / 1e6, 1), "frac": round(by / (hbm_peak * 1e9) * 1e3 / ms, 4),
                     "path": wb.wbmm_path_string(wb.wbmm_last_path()), "buffer_sets": ns, "note": "includes the dT zeroing launch"}
        del xs, gs, d
        torch.cuda.empty_cache()
    return out


def run_wbmm(args, rank, world, local):
    import paper_2607_02097_b200 as wb

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libwbmm has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream()
    case = si.CFG3
    fl, by = flops_of(case), bytes_of(case)

    # rotating buffer sets so that consecutive steps never find their inputs in L2
    nsets = 3
    d0 = si.make(case, device=dev)
    xs = [d0["x"]] + [d0["x"].roll(i + 1, 0).contiguous() for i in range(nsets - 1)]
    ys = [torch.empty_like(d0["x"]) for _ in range(nsets)]
    T = d0["T"]
    footprint = nsets * 2 * d0["x"].numel() * 2

    def step(i):
        wb.wbmm_forward(xs[i % nsets], T, case.w, case.shift, case.layout, out=ys[i % nsets])

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    warm = max(3, args.warmup)
    for i in range(warm):
        step(i)
    torch.cuda.synchronize()
    path = wb.wbmm_path_string(wb.wbmm_last_path())
    # keep the GPU under load long enough for nvidia-smi to sample clocks under this kernel
    t_load0 = time.time()
    i = 0
    while time.time() - t_load0 < 0.6:
        for _ in range(50):
            step(i); i += 1
        torch.cuda.synchronize()

    barrier(world)
    torch.cuda.synchronize()
    n0 = wb.wbmm_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(args.steps):
        step(i)
    e1.record(stream)
    torch.cuda.synchronize()
    barrier(world)
    t_load1 = time.time()
    launches = wb.wbmm_launch_count() - n0
    ms_total = max_over_ranks(e0.elapsed_time(e1), world, dev)
    ms_step = ms_total / args.steps
    clocks = sampler.stop(t_load0, t_load1) if rank == 0 else None

    # per-launch statistics (same kernel, each launch bracketed by events on its stream)
    per = time_steps(step, max(args.steps, 20), stream)
    ms_med, ms_min = statistics.median(per), min(per)
    # hot-L2 number for contrast: same buffers every step
    hot = time_steps(lambda i: wb.wbmm_forward(xs[0], T, case.w, out=ys[0]), 20, stream)

    value = world * fl / (ms_step * 1e-3) / 1e12

    # end to end through the C ABI with pinned host buffers
    e2e = None
    if True:
        h = si.make(case, pin=True)
        yh = torch.empty_like(h["x"]).pin_memory()
        for _ in range(2):
            wb.wbmm_forward_host(h["x"], h["T"], case.w, out=yh)
        barrier(world)
        n_e2e = max(3, min(args.steps, 10))
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            wb.wbmm_forward_host(h["x"], h["T"], case.w, out=yh)
        dt = (time.perf_counter() - t0) / n_e2e
        dt = max_over_ranks(dt, world, dev)
        e2e = {"value": world * fl / dt / 1e12, "unit": UNIT, "ms_per_step": dt * 1e3,
               "h2d_bytes_per_step": h["x"].numel() * 2 + h["T"].numel() * 2,
               "d2h_bytes_per_step": yh.numel() * 2, "steps": n_e2e,
               "api": "wbmm_forward_host (pinned host buffers)"}

    if rank != 0:
        return

    hbm_peak, tc_peak, peak_kind = measured_peaks()
    # one launch per step and nothing else on the stream: the average launch duration over the timed
    # region (CUDA events on the launching stream) is ms_step
    achieved = by / (ms_step * 1e-3) / 1e9
    t_roof = max(fl / (tc_peak * 1e12), by / (hbm_peak * 1e9))
    roofline = {"bound": "hbm", "achieved": achieved, "peak": hbm_peak, "unit": "GB/s",
                "frac": achieved / hbm_peak, "traffic": ncu_traffic_bytes(),
                "peak_kind": f"{peak_kind} (MEASURED_PEAKS.json hbm_gbs)" if peak_kind == "measured" else "fallback (B200_PROFILING.md)",
                "kernel": path, "kernel_ms_avg_timed_region": ms_step,
                "kernel_ms_median_event_pair_per_launch": ms_med, "kernel_ms_min_event_pair_per_launch": ms_min,
                "algorithmic_bytes_per_launch": by, "algorithmic_flops_per_launch": fl,
                "t_roof_ms": t_roof * 1e3, "frac_of_roofline_time": t_roof * 1e3 / ms_step,
                "tensor_tflops": fl / (ms_step * 1e-3) / 1e12,
                "hot_l2_ms_median_event_pair": statistics.median(hot)}

    # training step (config 5) as context: forward + dX + dT on rotating buffer sets (x, y, dy, dx of one set are
    # 154 MB; three sets never find their inputs in the 126 MB L2)
    c5 = si.CFG5
    d5 = si.make(c5, device=dev)
    ns5 = 3
    x5 = [d5["x"]] + [d5["x"].clone() for _ in range(ns5 - 1)]
    g5s = [d5["dy"]] + [d5["dy"].clone() for _ in range(ns5 - 1)]
    y5s = [torch.empty_like(d5["x"]) for _ in range(ns5)]
    dx5 = [torch.empty_like(d5["x"]) for _ in range(ns5)]
    dT5r = torch.empty((c5.C, c5.bins), dtype=torch.float32, device=dev)
    y5 = y5s[0]

    def train(i):
        j = i % ns5
        wb.wbmm_forward(x5[j], d5["T"], c5.w, c5.shift, out=y5s[j])
        wb.wbmm_backward(x5[j], d5["T"], g5s[j], c5.w, c5.shift, dT=dT5r, dx=dx5[j])

    def region_ms(fn, n=20):
        return region_ms_rot(lambda i: fn(), n, stream)

    for i in range(3):
        train(i)
    t5 = time_steps(train, 12, stream)
    train_path = wb.wbmm_path_string(wb.wbmm_last_path())
    parts = {
        "fwd_ms": region_ms_rot(lambda i: wb.wbmm_forward(x5[i % ns5], d5["T"], c5.w, c5.shift, out=y5s[i % ns5]), 30, stream),
        "dX_ms": region_ms_rot(lambda i: wb.wbmm_backward(None, d5["T"], g5s[i % ns5], c5.w, c5.shift, need_dT=False, dx=dx5[i % ns5]), 30, stream),
        "dT_ms": region_ms_rot(lambda i: wb.wbmm_backward(x5[i % ns5], None, g5s[i % ns5], c5.w, c5.shift, need_dx=False, dT=dT5r), 30, stream),
    }
    by5 = 2 * c5.n_elem * 2 * 2 + 2 * c5.n_elem * 2 + c5.C * c5.bins * 4   # x,y; dy,dx; x,dy; dT
    train_step = {"workload": "cfg5 B128 C192 28x28 w14 shift7 fwd+dX+dT", "ms_median": statistics.median(t5),
                  "ms_min": min(t5), "back_to_back": parts, "last_path": train_path, "flops": 3 * flops_of(c5),
                  "hbm_frac_at_median": by5 / (statistics.median(t5) * 1e-3) / 1e9 / hbm_peak,
                  "note": f"rotating {ns5} buffer sets of (x, y, dy, dx) = 462 MB: cold-L2 numbers; back_to_back = each kernel alone"}

    # the same step (forward, dX, dT zeroing, dT) replayed from one CUDA graph: device-side time, no host gaps
    try:
        dT5 = torch.empty((c5.C, c5.bins), dtype=torch.float32, device=dev)
        torch.cuda.synchronize()
        g5 = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g5):
            for j in range(ns5):
                wb.wbmm_forward(x5[j], d5["T"], c5.w, c5.shift, out=y5s[j])
                wb.wbmm_backward(x5[j], d5["T"], g5s[j], c5.w, c5.shift, dT=dT5, dx=dx5[j])
        train_step["ms_graph"] = region_ms(g5.replay) / ns5       # the graph holds one step per buffer set
        del g5
    except Exception as e:  # capture not possible: the eager numbers stand
        sys.stderr.write(f"train-step graph capture failed: {str(e)[:80]}\n")
        torch.cuda.synchronize()
        train_step["ms_graph"] = None

    # hierarchical reparameterisation, fused forward on the headline shape: context
    g_l = torch.Generator(device="cpu").manual_seed(77)
    Tl = (torch.randn((case.C, (case.w - 1) ** 2), generator=g_l) * 0.02).to(T.dtype).to(dev)
    hier_ms = region_ms(lambda: wb.wbmm_hier_forward(xs[0], T, Tl, case.w, out=ys[0]))
    train_step["hier_forward_cfg3_ms"] = hier_ms
    # cached-M mode (WBMM-C) on the headline shape: given matrices through the gather kernel -- context
    Mc = wb.wbmm_materialize_weight(T, case.w)
    train_step["cached_matrix_forward_cfg3_ms"] = region_ms(lambda: wb.wbmm_forward_matrix(xs[0], Mc, case.w, out=ys[0]))
    del Mc
    # ... and its backward on the config-5 shape: dX (transposed fused operator) + both table gradients in one pass
    g_l5 = torch.Generator(device="cpu").manual_seed(78)
    Tl5 = (torch.randn((c5.C, (c5.w - 1) ** 2), generator=g_l5) * 0.02).to(d5["T"].dtype).to(dev)
    train_step["hier_cfg5_ms"] = {
        "fwd": region_ms(lambda: wb.wbmm_hier_forward(d5["x"], d5["T"], Tl5, c5.w, c5.shift, out=y5)),
        "dX": region_ms(lambda: wb.wbmm_hier_backward(None, d5["T"], Tl5, d5["dy"], c5.w, c5.shift, need_dT=False)),
        "dTg_dTl": region_ms(lambda: wb.wbmm_hier_backward(d5["x"], None, None, d5["dy"], c5.w, c5.shift, need_dx=False)),
    }

    del x5, g5s, y5s, dx5
    torch.cuda.empty_cache()
    others = other_rooflines(wb, dev, stream, hbm_peak)

    tfl_cpu, cores, sample, dt_cpu = time_oracle(case)
    cpu = {"value": tfl_cpu, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
           "seconds": dt_cpu, "legs": oracle_legs(case, c5)}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": warm, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": {"workload": "cfg3: B=128 C=96 H=W=56 w=14 NCHW bf16 in/fp32 acc/bf16 out (BASELINE.json configs[2], the headline)",
                   "per_gpu_batch": case.B, "path": path,
                   "l2": f"rotating {nsets} buffer sets, footprint {footprint / 1e6:.0f} MB > 2x L2 (cold-L2 numbers)"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
        "roofline": roofline, "other_rooflines": others, "cpu_baseline": cpu, "train_step": train_step,
        "context": conv_context(case, d0["x"]),
    }
    print(json.dumps(out), flush=True)


def run_sweep(args):
    """--sweep: BASELINE.json config 4 (82 forward cases) + configs 2 and 5, one JSON line per case.
    Not the bench line; a table for profiles/ and BASELINE.md context."""
    import paper_2607_02097_b200 as wb
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream()
    hbm_peak, tc_peak, _ = measured_peaks()
    cases = [si.CFG2, si.CFG3, si.with_(si.CFG5, backward=False)] + list(si.sweep_cases())
    for case in cases:
        d = si.make(case, device="cuda")
        tensor_bytes = d["x"].numel() * 2
        nsets = int(min(4, max(2, -(-2 * L2_BYTES // (2 * tensor_bytes)) + 1)))
        xs = [d["x"]] + [d["x"].clone() for _ in range(nsets - 1)]
        ys = [torch.empty_like(d["x"]) for _ in range(nsets)]
        f = lambda i: wb.wbmm_forward(xs[i % nsets], d["T"], case.w, case.shift, case.layout, out=ys[i % nsets])
        n = 30 if case.n_elem < 2e8 else 10
        for i in range(3):
            f(i)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for i in range(n):
            f(i)
        b.record(stream)
        torch.cuda.synchronize()
        ms = a.elapsed_time(b) / n
        # the same launches replayed from a CUDA graph: device-side time without the per-call host cost
        # of the Python binding (which bounds the small shapes at ~14 us per call)
        ms_graph = None
        try:
            gr = torch.cuda.CUDAGraph()
            with torch.cuda.graph(gr):
                for i in range(n):
                    f(i)
            gr.replay()
            torch.cuda.synchronize()
            a.record()
            gr.replay()
            b.record()
            torch.cuda.synchronize()
            ms_graph = a.elapsed_time(b) / n
        except Exception as e:  # capture not possible: keep the eager number only
            sys.stderr.write(f"graph capture failed for {case.name}: {str(e)[:80]}\n")
            torch.cuda.synchronize()
        fl, by = flops_of(case), bytes_of(case)
        t_roof = max(fl / (tc_peak * 1e12), by / (hbm_peak * 1e9))
        print(json.dumps({"sweep_case": case.name, "layout": "NHWC" if case.layout else "NCHW", "B": case.B, "C": case.C,
                          "H": case.H, "w": case.w, "shift": list(case.shift), "ms": round(ms, 5),
                          "ms_graph": None if ms_graph is None else round(ms_graph, 5),
                          "frac_of_roofline_graph": None if ms_graph is None else round(t_roof * 1e3 / ms_graph, 4),
                          "tflops": round(fl / ms / 1e9, 2), "gbs": round(by / ms / 1e6, 1),
                          "frac_of_roofline": round(t_roof * 1e3 / ms, 4),
                          "path": wb.wbmm_path_string(wb.wbmm_last_path()), "buffer_sets": nsets}), flush=True)
        del xs, ys, d

    # backward (rows a7, a8 of SURVEY.md 8(a)) on the named configs and the large sweep shapes: dX and dT timed
    # apart, back to back on rotating buffer sets
    bwd = [si.with_(si.CFG2, backward=True), si.with_(si.CFG3, backward=True), si.CFG5,
           si.with_(si.CFG5, shift=(0, 0), name="cfg5_shape_no_shift")]
    for (C, H) in ((96, 56), (192, 28), (384, 28), (96, 112)):
        for w in (7, 14):
            bwd.append(si.Case(f"bwd_B128_C{C}_H{H}_w{w}", 128, C, H, H, w, backward=True, seed=200 + C + H + w))
    bwd.append(si.Case("bwd_ragged_B64_C96_H60_w14", 64, 96, 60, 60, 14, backward=True, seed=299))
    for case in bwd:
        d = si.make(case, device="cuda")
        ns = buffer_sets(3.0 * case.n_elem * 2, cap=6)       # rotating (x, dy, dx) sets: cold-L2 numbers
        xs = [d["x"]] + [d["x"].clone() for _ in range(ns - 1)]
        gs = [d["dy"]] + [d["dy"].clone() for _ in range(ns - 1)]
        dxs = [torch.empty_like(d["x"]) for _ in range(ns)]
        dT = torch.empty((case.C, case.bins), dtype=torch.float32, device="cuda")
        out = {}
        for key, fn in (("dX", lambda i: wb.wbmm_backward(None, d["T"], gs[i % ns], case.w, case.shift, case.layout, need_dT=False, dx=dxs[i % ns])),
                        ("dT", lambda i: wb.wbmm_backward(xs[i % ns], None, gs[i % ns], case.w, case.shift, case.layout, need_dx=False, dT=dT))):
            out[key] = (region_ms_rot(fn, 20, stream), wb.wbmm_path_string(wb.wbmm_last_path()))
        by = bytes_of(case)          # dX: dy in, dx out; dT: x and dy in -- the same 2 x tensor bytes (+ table)
        print(json.dumps({"sweep_case": "backward_" + case.name, "layout": "NCHW", "B": case.B, "C": case.C, "H": case.H,
                          "w": case.w, "shift": list(case.shift), "dX_ms": round(out["dX"][0], 5), "dT_ms": round(out["dT"][0], 5),
                          "dX_frac_of_hbm_roofline": round(by / (hbm_peak * 1e9) * 1e3 / out["dX"][0], 4),
                          "dT_frac_of_hbm_roofline": round(by / (hbm_peak * 1e9) * 1e3 / out["dT"][0], 4),
                          "dX_path": out["dX"][1], "dT_path": out["dT"][1], "buffer_sets": ns}), flush=True)
        del d, xs, gs, dxs, dT
        torch.cuda.empty_cache()


# The paper's operator benchmark, Table 13 B=128 block: single A800, FP32,
# 256 channels, kFPS read as 10^3 [256,H,W] maps per second.  Context, not the target: another machine, another
# precision for the bf16 rows.  {w: {map side: (WBMM-C kFPS, WBMM-NC kFPS)}}
PAPER_TABLE13_B128 = {
    7: {7: (2016, 1582), 14: (566, 525), 28: (165, 161), 56: (42, 42), 112: (10.5, 10.5), 224: (2.66, 2.67)},
    14: {14: (1276, 641), 28: (242, 199), 56: (63, 60), 112: (15.1, 14.9), 224: (3.83, 3.84)},
}


def run_paper_shapes(args):
    """--paper-shapes: wbmm_forward on the shapes of the paper's own operator benchmark (B=128, C=256, maps 7^2 ..
    224^2, windows 7 and 14), in bf16 and in fp32, one JSON line per case with kFPS = B / ms next to the paper's
    A800 FP32 figures.  Values are drawn on the device (timing only; parity lives in tests/)."""
    import paper_2607_02097_b200 as wb
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream()
    hbm_peak, tc_peak, _ = measured_peaks()
    B, C = 128, 256
    gen = torch.Generator(device="cuda").manual_seed(1313)
    for dtype, tdt in (("bf16", torch.bfloat16), ("f32", torch.float32)):
        for w, maps in PAPER_TABLE13_B128.items():
            for H, (kfps_c, kfps_nc) in maps.items():
                x = torch.randn((B, C, H, H), generator=gen, device="cuda", dtype=torch.float32).to(tdt)
                T = (torch.randn((C, (2 * w - 1) ** 2), generator=gen, device="cuda") * 0.02).to(tdt)
                y = torch.empty_like(x)
                f = lambda: wb.wbmm_forward(x, T, w, (0, 0), si.NCHW, out=y)
                for _ in range(2):
                    f()
                torch.cuda.synchronize()
                n = 3 if dtype == "f32" and H >= 112 else 10
                ms = None
                try:        # from a CUDA graph: device-side time (the small maps are host-bound when called eagerly)
                    gr = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(gr):
                        for _ in range(n):
                            f()
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(stream)
                    gr.replay()
                    b.record(stream)
                    torch.cuda.synchronize()
                    ms = a.elapsed_time(b) / n
                    del gr
                except Exception as e:
                    sys.stderr.write(f"graph capture failed for H={H} w={w} {dtype}: {str(e)[:80]}\n")
                    torch.cuda.synchronize()
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(stream)
                    for _ in range(n):
                        f()
                    b.record(stream)
                    torch.cuda.synchronize()
                    ms = a.elapsed_time(b) / n
                es = 2 if dtype == "bf16" else 4
                by = 2.0 * x.numel() * es + T.numel() * es
                fl = 2.0 * w * w * x.numel()
                print(json.dumps({"paper_case": f"B{B}_C{C}_H{H}_w{w}_{dtype}", "B": B, "C": C, "H": H, "w": w, "dtype": dtype,
                                  "ms": round(ms, 5), "kfps": round(B / ms, 2), "tflops": round(fl / ms / 1e9, 2),
                                  "gbs": round(by / ms / 1e6, 1), "frac_of_hbm_roofline": round(by / (hbm_peak * 1e9) * 1e3 / ms, 4),
                                  "path": wb.wbmm_path_string(wb.wbmm_last_path()),
                                  "paper_A800_fp32_kfps_cached": kfps_c, "paper_A800_fp32_kfps_not_cached": kfps_nc}), flush=True)
                del x, y, T
                torch.cuda.empty_cache()


PROFILE_CASES = {
    "cfg3_fwd": (si.CFG3, "fwd"), "cfg2_fwd": (si.CFG2, "fwd"),
    "cfg5_fwd": (si.with_(si.CFG5, backward=False), "fwd"), "cfg5_dX": (si.CFG5, "dX"), "cfg5_dT": (si.CFG5, "dT"),
    "cfg3_shape_dT": (si.with_(si.CFG3, backward=True), "dT"),
    "fp32_w14_fwd": (si.with_(si.CFG3, dtype="f32"), "fwd"),
    "fp32_w7_fwd": (si.Case("f32w7", 128, 96, 56, 56, 7, dtype="f32", seed=86), "fwd"),
    "fp32_w14_dT": (si.with_(si.CFG3, dtype="f32", backward=True), "dT"),
    "fp32_w7_dT": (si.Case("f32w7", 128, 96, 56, 56, 7, dtype="f32", backward=True, seed=86), "dT"),
    "nhwc_cfg3_fwd": (si.with_(si.CFG3, layout=si.NHWC), "fwd"),
    "s3_B128_C256_14x14_w14_fwd": (si.Case("s3w14", 128, 256, 14, 14, 14, seed=88), "fwd"),
    "s3_B128_C256_14x14_w7_fwd": (si.Case("s3w7", 128, 256, 14, 14, 7, seed=89), "fwd"),
    "s4_B128_C256_7x7_w7_fwd": (si.Case("s4w7", 128, 256, 7, 7, 7, seed=90), "fwd"),
    "s3_B128_C592_14x14_w14_fwd": (si.Case("s3w14big", 128, 592, 14, 14, 14, seed=91), "fwd"),
    "B64_C96_30x30_w14_fwd": (si.Case("r30", 64, 96, 30, 30, 14, seed=92), "fwd"),
    "cfg2_shape_dT": (si.with_(si.CFG2, backward=True), "dT"),
    "nhwc_cfg2_shape_B128_fwd": (si.Case("nhwc_w7", 128, 96, 56, 56, 7, layout=si.NHWC, seed=87), "fwd"),
    "int8_w14_fwd": (si.with_(si.CFG3, backward=False), "int8"), "int8_w7_fwd": (si.with_(si.CFG2, backward=False), "int8"),
}


def run_profile_case(name: str):
    """--profile-case NAME: five launches of one kernel on one named workload and nothing else -- the command the
    `ncu --set full` captures under profiles/ are taken with (a number printed under a profiler is never a result)."""
    import paper_2607_02097_b200 as wb
    case, op = PROFILE_CASES[name]
    torch.cuda.set_device(0)
    if op == "int8":
        d = si.make_int8(case, device="cuda")
        y = torch.empty_like(d["x"])
        for _ in range(5):
            wb.wbmm_forward_int8(d["x"], d["T"], case.w, scale=d["scale"], out=y)
        torch.cuda.synchronize()
        print(json.dumps({"profile_case": name, "op": op, "path": wb.wbmm_path_string(wb.wbmm_last_path())}))
        return
    d = si.make(case, device="cuda")
    y = torch.empty_like(d["x"])
    dT = torch.empty((case.C, case.bins), dtype=torch.float32, device="cuda")
    for _ in range(5):
        if op == "fwd":
            wb.wbmm_forward(d["x"], d["T"], case.w, case.shift, case.layout, out=y)
        elif op == "dX":
            wb.wbmm_backward(None, d["T"], d["dy"], case.w, case.shift, case.layout, need_dT=False, dx=y)
        else:
            wb.wbmm_backward(d["x"], None, d["dy"], case.w, case.shift, case.layout, need_dx=False, dT=dT)
    torch.cuda.synchronize()
    print(json.dumps({"profile_case": name, "op": op, "path": wb.wbmm_path_string(wb.wbmm_last_path())}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="wbmm", choices=["wbmm", "reference"])
    ap.add_argument("--sweep", action="store_true", help="time the config-4 operator sweep instead (one JSON line per case)")
    ap.add_argument("--ref-seconds", type=float, default=100.0, help="--impl reference: CPU seconds for the whole run")
    ap.add_argument("--paper-shapes", action="store_true",
                    help="time the shapes of the paper's Table 13 (B=128, C=256) in bf16 and fp32 (one JSON line per case)")
    ap.add_argument("--profile-case", choices=sorted(PROFILE_CASES), help="five launches of one kernel on one workload (for ncu)")
    args = ap.parse_args()
    if args.profile_case:
        run_profile_case(args.profile_case)
        return
    if args.sweep:
        run_sweep(args)
        return
    if args.paper_shapes:
        run_paper_shapes(args)
        return
    if args.impl == "reference":
        rank = int(os.environ.get("RANK", "0"))
        run_reference(args, rank, int(os.environ.get("WORLD_SIZE", "1")))
        return
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        # plain `python bench.py --gpus N`: launch the N ranks ourselves (one process per GPU, replicas only)
        if torch.cuda.device_count() < args.gpus:
            sys.stderr.write(f"bench.py: --gpus {args.gpus} but {torch.cuda.device_count()} CUDA device(s) visible\n")
            raise SystemExit(2)
        import socket
        with socket.socket() as sock:
            sock.bind(("127.0.0.1", 0))
            port = sock.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
        raise SystemExit(subprocess.call(cmd))
    if int(os.environ.get("WORLD_SIZE", "1")) != args.gpus:
        sys.stderr.write(f"bench.py: --gpus {args.gpus} does not match WORLD_SIZE={os.environ.get('WORLD_SIZE')}\n")
        raise SystemExit(2)
    rank, world, local = dist_setup(args.gpus)
    try:
        run_wbmm(args, rank, world, local)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
