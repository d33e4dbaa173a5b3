#!/usr/bin/env python
"""bench.py -- Spense FP8 GLU-MLP decode step on B200 (BASELINE.json metric: us/layer + HBM GB/s vs peak,
speedup vs the library's own all-dense FP8 kernel).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--M 64] [--no-sweep] [--no-cpu] [--report]

Workload (BASELINE.json configs[1]): Qwen3-32B-shaped MLP layer, H=5120, I=25600, p=25 % dense
intermediate indices, FP8 E4M3 weights/activations, seeded synthetic inputs (spense_inputs).  One
STEP = one pass of the whole hot path (spense_mlp = gate_up -> SiLU*up -> requant -> down) over
LAYERS distinct packed layers (8 x 283 MB = 2.26 GB >> the 126 MB L2, so every weight byte streams from
HBM), launched back to back on one stream and replayed as one CUDA graph.  value = us per layer.
N > 1 (torchrun): the path does not shard at bar level ("replicas only"): every rank runs
the same step; value = step time / (N * LAYERS).
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

H, I, P_DENSE = 5120, 25600, 0.25
SEED_H, SEED_I = 5120, 27648
LAYERS = 8
# dram__bytes_read.sum + dram__bytes_write.sum of the GEMM launches of a real step, from the committed ncu
# application-replay capture of THIS kernel version (profiles/, with the command that made it); keyed by M
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r03_traffic_app_replay_M64.csv")
TRAFFIC_M = 64


def algorithmic_bytes(M: int, h: int, i: int, i_d: int) -> int:
    """SURVEY.md 8(d) / DESIGN.md section 5: weights streamed once + activations the method must move."""
    w = 3 * h * (i_d + (i - i_d) * 0.625)
    act = M * h + 4 * M + 2 * M * i + 2 * M * h          # X, s_x, Hq written + read, Y bf16
    return int(w + act)


NOMINAL_HBM_GBS = 8000.0     # north_star: "against the ~8 TB/s peak"


def blob_bytes_of(h: int, i: int, i_d: int) -> int:
    return 1024 + int(3 * h * (i_d + (i - i_d) * 0.625))


def config_of(M: int, i_d: int, world: int) -> dict:
    """The workload both arms report (the reference arm times a bounded sample of it, named in its cpu_baseline.sample)."""
    return {"workload": f"qwen3_32b_mlp_layer H={H} I={I} p=25% (I_dense={i_d}) M={M}",
            "layers_per_step": LAYERS, "launch": "CUDA graph of LAYERS x spense_mlp (2 PDL-chained kernels each)",
            "l2": f"inputs larger than L2: {LAYERS} distinct packed layers = {LAYERS * blob_bytes_of(H, I, i_d) / 1e9:.2f} GB rotate",
            "parallelism": "replicas only" if world > 1 else "single GPU"}


def read_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), float(d.get("bf16_tflops", 0.0)), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, 1590.0, "fallback (B200_PROFILING.md)"


def traffic_from_profile(M: int):
    """traffic per layer = (sum of dram read + write bytes over the captured GEMM launches) / layers captured; None
    unless the committed capture is for this M (it goes stale with the kernel: re-capture, do not edit)."""
    if M != TRAFFIC_M or not os.path.exists(TRAFFIC_CSV):
        return None
    tot, launches = 0.0, set()
    with open(TRAFFIC_CSV) as f:
        for row in csv.DictReader(l for l in f if not l.startswith("==")):
            name, val, unit = row.get("Metric Name", ""), row.get("Metric Value", ""), row.get("Metric Unit", "")
            if name in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                v = float(val.replace(",", ""))
                tot += v * {"byte": 1, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(unit, 1)
                launches.add(row.get("ID"))
    if not launches:
        return None
    return int(tot / (len(launches) / 2))                # two GEMM launches per layer


class ClockSampler:
    """nvidia-smi polled every 20 ms in the background; every line is stamped with the host time it arrived, so
    the samples that fall inside a timed region can be picked out afterwards."""
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, idx: int):
        self.p = None
        self.idx = idx
        self.lines = []

    def start(self):
        import threading
        try:
            self.p = subprocess.Popen(
                ["nvidia-smi", f"--id={self.idx}",
                 "--query-gpu=clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
                 "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
                 "clocks_event_reasons.sw_power_cap", "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True, bufsize=1)
        except Exception:
            self.p = None
            return

        def pump():
            for line in self.p.stdout:
                self.lines.append((time.time(), line))
        self.t = threading.Thread(target=pump, daemon=True)
        self.t.start()

    def n_samples(self):
        return len(self.lines)

    def window(self, t0=None, t1=None, fallback_all=True):
        inside = [l for (t, l) in self.lines if t0 is None or (t0 <= t <= t1 + 0.02)]
        where = "timed region"
        if not inside and fallback_all:                  # region shorter than the polling period: the load around it
            inside = [l for (t, l) in self.lines]
            where = "warm-up + timed region (timed region shorter than the 20 ms polling period)"
        sm, mx, reasons = [], [], set()
        for line in inside:
            t = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(t[0])); mx.append(float(t[1]))
            except Exception:
                continue
            for n, v in zip(self.NAMES, t[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "sampled_over": where}

    def stop(self):
        if self.p is not None:
            self.p.terminate()
            self.t.join(timeout=2)


def oracle_layer(M: int):
    """One FULL-SIZE layer for the oracle: generated by the seeded generator (on the GPU when there is one: the bytes are
    what counts), packed and reconstructed by the oracle itself.  Set-up, not timed."""
    import numpy as np
    import torch
    import spense_inputs as si
    from oracle import spense_oracle as o
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    L = si.make_layer(H, I, P_DENSE, seed=2000, device=dev)
    x, sx = si.make_activations(M, H, seed=1000 + M)
    c = o.pack_canonical(L.wgate.cpu().numpy(), L.wup.cpu().numpy(), L.wdown.cpu().numpy(), L.perm.cpu().numpy(), L.I_dense)
    wg, wu, wd = o.unpack_canonical(c)
    w_scale, i_d = L.w_scale, int(L.I_dense)
    del L, c
    if dev == "cuda":
        torch.cuda.empty_cache()
    return dict(o=o, x=x.numpy(), sx=sx.numpy(), wg=wg, wu=wu, wd=wd, w_scale=w_scale, s_h=np.full(M, 0.05, np.float32), I_dense=i_d)


def oracle_time_layer(ol, reps: int):
    """seconds per full layer: oracle.mlp (decode E4M3 -> float64 GEMMs -> SiLU*up -> requant -> down), as it stands"""
    t0 = time.perf_counter()
    for _ in range(reps):
        ol["o"].mlp(ol["x"], ol["sx"], ol["wg"], ol["wu"], ol["wd"], ol["w_scale"], ol["s_h"])
    return (time.perf_counter() - t0) / reps


def cpu_baseline(M: int, reps: int = 4):
    import torch
    ol = oracle_layer(M)
    oracle_time_layer(ol, 1)                              # first touch
    dt = oracle_time_layer(ol, reps)
    return {"value": dt * 1e6, "unit": "us/layer", "cores": int(torch.get_num_threads() or os.cpu_count()), "kind": "oracle",
            "sample": f"oracle.mlp on ONE full-size layer (H={H}, I={I}, p=25 %, M={M}; the bench step is {LAYERS} such layers), "
                      f"mean of {reps} runs after one warm-up; numpy float64 GEMMs on the host cores"}


def run_reference(args):
    """--impl reference: for this tier the reference arm is the oracle on the host cores.  One step = the oracle on ONE
    full-size layer (a bounded sample of the 8-layer step: the layers are statistically identical)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import torch
    ol = oracle_layer(args.M)
    t_start = time.perf_counter()
    n_warm = 0
    for _ in range(args.warmup):                          # the requested warm-up (each step is ~2 s of host work)
        oracle_time_layer(ol, 1)
        n_warm += 1
        if time.perf_counter() - t_start > 60:
            break
    steps = []
    for _ in range(args.steps):
        steps.append(oracle_time_layer(ol, 1))
        if time.perf_counter() - t_start > 200:
            break
    v = sum(steps) / len(steps) * 1e6
    sample = (f"oracle.mlp on ONE full-size layer per step (H={H}, I={I}, p=25 %, M={args.M}), {len(steps)} timed steps; "
              f"ms_per_step is that one layer, not {LAYERS}")
    line = {"impl": "reference", "metric": "spense_fp8_mlp_us_per_layer", "value": v, "unit": "us/layer",
            "n_gpus": args.gpus, "steps": len(steps), "warmup": n_warm, "ms_per_step": v / 1e3,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_of(args.M, ol["I_dense"], 1 if args.gpus <= 1 else args.gpus),
            "cpu_baseline": {"value": v, "unit": "us/layer", "cores": int(torch.get_num_threads() or os.cpu_count()), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": v, "unit": "us/layer", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------- GPU helpers
def make_blobs(sp, si, dev, h, i, p, n, seed0, i_dense=None):
    import torch
    out = []
    for k in range(n):
        L = si.make_layer(h, i, p, seed0 + k, device=dev, I_dense=i_dense)
        out.append(sp.spense_pack(L.wgate, L.wup, L.wdown, L.w_scale, L.perm, L.I_dense))
        del L
    torch.cuda.empty_cache()
    return out


def graph_of(fn):
    """capture fn (a sequence of library calls on the current stream) into a CUDA graph; no eager call first: the
    library neither synchronises nor reads device memory on the host"""
    import torch
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):
            fn()
    torch.cuda.current_stream().wait_stream(s)
    return g


def event_time_ms(replay, steps, warmup, dist=None, replicas=None, dev=None, host_window=None):
    import torch
    for _ in range(warmup):
        replay()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_host0 = time.time()
    e0.record()
    for _ in range(steps):
        replay()
    e1.record()
    torch.cuda.synchronize()
    if host_window is not None:
        host_window[:] = [t_host0, time.time()]
    ms = e0.elapsed_time(e1)
    if dist is not None:
        ms = replicas.max_over_ranks(ms, dist, dev)
        dist.barrier()
    return ms / steps


def hbm_probes(sp, dev, timed, sustained_s: float):
    """SURVEY.md 8d "time floors", measured in THIS run on THIS box: (a) the read-only stream ceiling (spense_probe_read: the
    GEMM's own bulk-copy producer with nothing behind it, 4 GiB per call >> L2), best of 10 single calls (burst, like
    MEASURED_PEAKS.json's copy figure) and back to back for sustained_s seconds; (b) torch's b.copy_(a) over 2 x 2 GiB
    (read + write bytes) back to back for sustained_s seconds, the sustained twin of MEASURED_PEAKS.json's hbm_gbs."""
    import torch
    n = 4 << 30
    buf = torch.empty(n, dtype=torch.uint8, device=dev)
    buf.view(torch.int64).random_()
    sink = torch.zeros(256, dtype=torch.int32, device=dev)
    call = lambda: sp.spense_probe_read(buf, sink)
    best = min(timed(call, 1, 2 if k == 0 else 0) for k in range(10))
    out = {"read_probe_gbs": round(n / best / 1e6, 1), "read_probe_bytes": n}
    if sustained_s > 0:
        reps = max(10, int(sustained_s / (best * 1e-3)))
        out["read_probe_sustained_gbs"] = round(n / timed(call, reps, 2) / 1e6, 1)
        a, b = buf[: n // 2], buf[n // 2:]
        t_copy = min(timed(lambda: b.copy_(a), 1, 2 if k == 0 else 0) for k in range(10))
        out["copy_gbs"] = round(n / t_copy / 1e6, 1)                     # n/2 read + n/2 written
        reps = max(10, int(sustained_s / (t_copy * 1e-3)))
        out["copy_sustained_gbs"] = round(n / timed(lambda: b.copy_(a), reps, 2) / 1e6, 1)
    del buf
    torch.cuda.empty_cache()
    return out


def fp8_dense_peak(sp, si, dev, dense_blobs, ws):
    """The FP8 dense tensor peak of THIS box, measured: torch._scaled_mm on 8192^3 (cuBLASLt, burst) and the
    library's own all-dense kernel at M = 8192 (gate_up of the Qwen shape).  TFLOP/s."""
    import torch
    out = {}
    try:
        n = 8192
        a = torch.randn(n, n, device=dev).to(torch.float8_e4m3fn)
        b = torch.randn(n, n, device=dev).to(torch.float8_e4m3fn).t()
        one = torch.ones((), device=dev)
        f = lambda: torch._scaled_mm(a, b, scale_a=one, scale_b=one, out_dtype=torch.bfloat16)
        for _ in range(3):
            f()
        best = 1e9
        for _ in range(10):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); f(); e1.record(); torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        out["scaled_mm_8192_tflops"] = round(2 * n ** 3 / best / 1e9, 1)
        del a, b
    except Exception as ex:                               # not fatal: the library's own kernel still gives a number
        out["scaled_mm_error"] = str(ex)[:120]
    m = 8192
    x, sx = si.make_activations(m, H, 1000 + m, device=dev)
    sh = torch.full((m,), 0.05, device=dev)
    hq = torch.empty(m, I, dtype=torch.uint8, device=dev)
    t = event_time_ms(graph_of(lambda: sp.spense_gate_up(dense_blobs[0], x, sx, sh, ws, hq=hq)).replay, 3, 2)
    out["own_dense_gate_up_M8192_tflops"] = round(2 * m * 2 * H * I / t / 1e9, 1)
    torch.cuda.empty_cache()
    return out


def prefill_rows(sp, si, dev, blobs, ws, fp8_peak_tflops):
    """BASELINE.json configs[4]: gate_up and down separately at M = 2048 / 8192, executed and dense-equivalent TFLOP/s"""
    import torch
    rows = []
    i_d = blobs[0].I_dense
    four = blobs[:4]
    for m in (2048, 8192):
        x, sx = si.make_activations(m, H, 1000 + m, device=dev)
        sh = torch.full((m,), 0.05, device=dev)
        hq = torch.empty(m, I, dtype=torch.uint8, device=dev)
        y = torch.empty(m, H, dtype=torch.bfloat16, device=dev)
        t_gu = event_time_ms(graph_of(lambda: [sp.spense_gate_up(b, x, sx, sh, ws, hq=hq) for b in four]).replay, 3, 2) * 1e3 / 4
        t_dn = event_time_ms(graph_of(lambda: [sp.spense_down(b, hq, sh, ws, y=y) for b in four]).replay, 3, 2) * 1e3 / 4
        ex_gu = 2 * m * 2 * H * (i_d + (I - i_d) / 2)       # executed flops (2:4 tiles do half)
        ex_dn = 2 * m * H * (i_d + (I - i_d) / 2)
        rows.append({"M": m, "gate_up_us": round(t_gu, 1), "down_us": round(t_dn, 1),
                     "gate_up_executed_tflops": round(ex_gu / t_gu / 1e6, 1), "down_executed_tflops": round(ex_dn / t_dn / 1e6, 1),
                     "gate_up_dense_equiv_tflops": round(2 * m * 2 * H * I / t_gu / 1e6, 1),
                     "down_dense_equiv_tflops": round(2 * m * H * I / t_dn / 1e6, 1),
                     "gate_up_frac_of_fp8_peak": round(ex_gu / t_gu / 1e6 / fp8_peak_tflops, 3),
                     "down_frac_of_fp8_peak": round(ex_dn / t_dn / 1e6 / fp8_peak_tflops, 3)})
        del x, hq, y
        torch.cuda.empty_cache()
    return rows


def w_bytes(h, i, i_d):
    return 3 * h * (i_d + (i - i_d) * 0.625)


def seed_sweep_rows(sp, si, dev, peak, ps=(1.0, 0.0, 0.10, 0.25, 0.50), ms=(1, 16, 64, 256), nl=5):
    """BASELINE.json configs[2]: Seed-OSS-36B-shaped layer, dense fraction x token count, speedup vs the all-dense kernel
    (p = 1.0 must come first: its times are the denominators)."""
    import torch
    rows, dense_t = [], {}
    for p in ps:
        bl = make_blobs(sp, si, dev, SEED_H, SEED_I, p, nl, 4000 + int(p * 100) * 10)
        i_d = bl[0].I_dense
        ws = sp.spense_workspace(bl[0], 256)
        for m in ms:
            x, sx = si.make_activations(m, SEED_H, 1000 + m, device=dev)
            sh = torch.full((m,), 0.05, device=dev)
            hq = torch.empty(m, SEED_I, dtype=torch.uint8, device=dev)
            y = torch.empty(m, SEED_H, dtype=torch.bfloat16, device=dev)
            t = event_time_ms(graph_of(lambda: [sp.spense_mlp(b, x, sx, sh, ws, hq_scratch=hq, y=y, next_layer=bl[(k + 1) % nl])
                                                for k, b in enumerate(bl)]).replay, 20, 5) * 1e3 / nl
            if p == 1.0:
                dense_t[m] = t
            algo = algorithmic_bytes(m, SEED_H, SEED_I, i_d)
            rows.append({"p": p, "I_dense": i_d, "M": m, "us_per_layer": round(t, 2), "gbs": round(algo / t / 1e3, 1),
                         "frac_of_hbm_peak": round(algo / t / 1e3 / peak, 3), "speedup_vs_dense": round(dense_t[m] / t, 3),
                         "byte_ratio_bound": round(w_bytes(SEED_H, SEED_I, SEED_I) / w_bytes(SEED_H, SEED_I, i_d), 3)})
        del bl, ws
        torch.cuda.empty_cache()
    return rows


def stack_rows(sp, si, dev, peak, bl, ws, ms=(32, 128)):
    """BASELINE.json configs[3]: 64 consecutive Qwen3-32B-shaped layers (18 GB of blobs) in one CUDA graph, tokens/s.
    Every layer reads the same x (the layers are chained through the stream, not through data: the paper's method has
    nothing between two MLPs; the data-chained variant with a normalise-and-quantise kernel is not built)."""
    import torch
    nl = len(bl)
    stack = []
    for m in ms:
        x, sx = si.make_activations(m, H, 1000 + m, device=dev)
        sh = torch.full((m,), 0.05, device=dev)
        hq = torch.empty(m, I, dtype=torch.uint8, device=dev)
        y = torch.empty(m, H, dtype=torch.bfloat16, device=dev)
        t = event_time_ms(graph_of(lambda: [sp.spense_mlp(b, x, sx, sh, ws, hq_scratch=hq, y=y, next_layer=bl[(k + 1) % nl])
                                            for k, b in enumerate(bl)]).replay, 10, 3) * 1e3
        algo = nl * algorithmic_bytes(m, H, I, bl[0].I_dense)
        stack.append({"M": m, "layers": nl, "ms_per_stack": round(t / 1e3, 4), "us_per_layer": round(t / nl, 2),
                      "tokens_per_s": round(m / (t * 1e-6), 1), "gbs": round(algo / t / 1e3, 1),
                      "frac_of_hbm_peak": round(algo / t / 1e3 / peak, 3)})
    return stack


def obs_rows(sp, dev):
    """NEXT-4, spense_prune_obs_2to4 on the two Qwen3-32B shapes (the sparse rows of gate / up along H; down along the
    permuted intermediate dimension with the 6400 dense columns as buffer): ms per sweep (best of 3, events) and the
    trailing update's flops (2 N 128 (K - j1) per 128-column block) over that time.  Synthetic weights N(0, 0.02^2);
    U = upper Cholesky factor of the inverse of a damped Gram matrix of K / 2 random samples (float64 library routines)."""
    import torch
    rows = []
    for name, n, k, ks in (("gate_or_up_sparse_rows", I - int(I * P_DENSE), H, H), ("down", H, I, I - int(I * P_DENSE))):
        g = torch.Generator(device=dev).manual_seed(k)
        xs = torch.randn(k // 2, k, device=dev, generator=g)
        hm = (xs.t() @ xs).double()
        del xs
        hm += 0.01 * hm.diagonal().mean() * torch.eye(k, device=dev, dtype=torch.float64)
        hinv = torch.cholesky_inverse(torch.linalg.cholesky(hm))
        del hm
        u = torch.linalg.cholesky(hinv, upper=True).float().contiguous()
        del hinv
        w0 = torch.randn(n, k, device=dev, generator=g) * 0.02
        w = torch.empty_like(w0)
        best = None
        for _ in range(3):
            w.copy_(w0)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            sp.spense_prune_obs_2to4(w, u, ks)                       # in place on w
            e1.record()
            torch.cuda.synchronize()
            best = e0.elapsed_time(e1) if best is None else min(best, e0.elapsed_time(e1))
        ok = bool(((w[:, :ks].view(n, ks // 4, 4) == 0).sum(dim=2) == 2).all())
        flops = sum(2.0 * n * min(128, ks - j0) * (k - min(j0 + 128, ks)) for j0 in range(0, ks, 128))
        rows.append({"matrix": name, "N": n, "K": k, "K_sparse": ks, "ms": round(best, 2), "two_of_four_holds": ok,
                     "trailing_update_tflops": round(flops / best / 1e9, 2), "arithmetic": "fp32 CUDA cores"})
        del u, w, w0
        torch.cuda.empty_cache()
    return rows


def run_report(args):
    """--report: the other BASELINE.json configs in full (context rows, not the bench line): Seed-OSS-36B shape
    dense-fraction sweep, the 64-layer Qwen3-32B-shaped stack, prefill-shaped GEMMs, the SparseGPT sweep's timing.
    Writes one JSON object to stdout and to gpurun_out/report.json.  Same timing rules as the bench line."""
    import torch
    import spense_inputs as si
    from paper_2606_10445_b200 import build, spense as sp
    build.build()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    peak, bf16_peak, _ = read_peaks()
    out = {"hbm_peak_gbs": peak}
    out["seed_oss_36b_sweep"] = seed_sweep_rows(sp, si, dev, peak)
    bl = make_blobs(sp, si, dev, H, I, P_DENSE, 64, 6000)
    ws = sp.spense_workspace(bl[0], 8192)
    out["qwen3_32b_stack"] = stack_rows(sp, si, dev, peak, bl, ws)

    # ---- config 5: prefill-shaped GEMMs against the measured FP8 dense peak
    dense = make_blobs(sp, si, dev, H, I, 1.0, 1, 3000)
    out["fp8_peak"] = fp8_dense_peak(sp, si, dev, dense, ws)
    del dense
    fp8 = out["fp8_peak"].get("scaled_mm_8192_tflops") or 2 * bf16_peak
    out["prefill_shaped"] = prefill_rows(sp, si, dev, bl, ws, fp8)
    del bl, ws
    torch.cuda.empty_cache()
    out["obs_sweep"] = obs_rows(sp, dev)
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    with open(os.path.join(ROOT, "gpurun_out", "report.json"), "w") as f:
        json.dump(out, f, indent=1)
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--report", action="store_true")
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="spense")
    ap.add_argument("--M", type=int, default=64)
    ap.add_argument("--no-sweep", action="store_true", help="skip the extras (M sweep vs the dense kernel, Seed-OSS row, prefill rows)")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--sustained-s", type=float, default=2.0)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.report:
        return run_report(args)

    import torch
    import spense_inputs as si
    from paper_2606_10445_b200 import build, replicas, spense as sp

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    build.build()                       # no-op when libspense.so is current; raises if it cannot be built
    dev = torch.device("cuda", local)
    M = args.M
    warmup = max(args.warmup, 3)

    blobs = make_blobs(sp, si, dev, H, I, P_DENSE, LAYERS, 2000)
    I_d = blobs[0].I_dense
    x, sx = si.make_activations(M, H, 1000 + M, device=dev)
    sh = torch.full((M,), 0.05, device=dev)
    ws = sp.spense_workspace(blobs[0], 8192)
    hq = torch.empty(M, I, dtype=torch.uint8, device=dev)
    y = torch.empty(M, H, dtype=torch.bfloat16, device=dev)

    def step_eager(layers, xx, ssx, ssh, hqq, yy, wsp=None):
        wsp = ws if wsp is None else wsp
        for i, b in enumerate(layers):                   # the layer that runs next is named as an L2 prefetch hint
            sp.spense_mlp(b, xx, ssx, ssh, wsp, hq_scratch=hqq, y=yy, next_layer=layers[(i + 1) % len(layers)])

    timed = lambda replay, steps, wu, hw=None: event_time_ms(replay, steps, wu, dist, replicas, dev, hw)
    timed_local = lambda replay, steps, wu: event_time_ms(replay, steps, wu)     # rank-0-only extras: no barrier, no all-reduce

    g_main = graph_of(lambda: step_eager(blobs, x, sx, sh, hq, y))
    sampler = ClockSampler(local)
    sampler.start()
    t_pre = time.time()
    while sampler.p is not None and sampler.n_samples() == 0 and time.time() - t_pre < 3.0:
        time.sleep(0.02)                                 # wait (idle) until nvidia-smi is polling
    window = [None, None]
    ms_step = timed(g_main.replay, args.steps, warmup, window)
    clocks = sampler.window(window[0], window[1])
    us_layer = ms_step * 1e3 / LAYERS

    # ---- end to end through the C ABI with HOST buffers (pinned; measured right after the device-timed region, before
    # the sustained leg and the extras heat the board): per STEP one H2D of x and the scales, LAYERS x
    # spense_mlp, one D2H of y, one synchronise (spense_mlp_stack_host)
    hx = x.cpu().pin_memory(); hsx = sx.cpu().pin_memory(); hsh = sh.cpu().pin_memory()
    hy = torch.empty(M, H, dtype=torch.bfloat16).pin_memory()
    staging = dict(d_x=torch.empty_like(x), d_scales=torch.empty(2 * M, device=dev), d_hq=hq, d_y=y)
    ms_e2e = timed(lambda: sp.spense_mlp_stack_host(blobs, hx, hsx, hsh, hy, staging, ws), max(5, args.steps // 5), 3)
    h2d = M * H + 4 * M + 4 * M
    d2h = M * H * 2

    # ---- sustained: the same graph replayed back to back for >= sustained_s seconds, clocks sampled INSIDE the region
    sustained = None
    if args.sustained_s > 0:
        n_sus = max(args.steps, int(args.sustained_s / (ms_step * 1e-3)) + 1)
        w2 = [None, None]
        ms_sus = timed(g_main.replay, n_sus, 3, w2)
        sustained = {"value": ms_sus * 1e3 / LAYERS / world, "unit": "us/layer", "steps": n_sus, "seconds": round(ms_sus * n_sus / 1e3, 3),
                     "clocks": sampler.window(w2[0], w2[1], fallback_all=False)}

    # ---- per-kernel view, other configs and the all-dense baseline kernel (same library, I_dense = I), rank 0 extras
    extras = {}
    peak, bf16_peak, peak_src = read_peaks()
    algo = algorithmic_bytes(M, H, I, I_d)
    if sustained is not None:
        sustained["hbm_gbs"] = algo / (sustained["value"] * world * 1e-6) / 1e9
        sustained["frac"] = sustained["hbm_gbs"] / peak
    probes = None
    if rank == 0:
        def t_us(fn, n=LAYERS):
            return timed_local(graph_of(fn).replay, 20, 5) * 1e3 / n
        extras["gate_up_us"] = t_us(lambda: [sp.spense_gate_up(b, x, sx, sh, ws, hq=hq) for b in blobs])
        extras["down_us"] = t_us(lambda: [sp.spense_down(b, hq, sh, ws, y=y) for b in blobs])
        # NEXT-1: the same layers with dynamic per-token requant (gate_up -> row requant kernel -> down)
        h32 = torch.empty(M, I, dtype=torch.float32, device=dev)
        sh_dyn = torch.empty(M, device=dev)
        extras["dynamic_requant_us"] = t_us(lambda: [sp.spense_mlp_dyn(b, x, sx, ws, s_h=sh_dyn, hq_scratch=hq, h_scratch=h32, y=y,
                                                                       next_layer=blobs[(i + 1) % len(blobs)]) for i, b in enumerate(blobs)])
        del h32
        if not args.no_sweep:
            # configs[1]: M sweep, Spense vs the all-dense kernel
            sweep = []
            dense = make_blobs(sp, si, dev, H, I, 1.0, 6, 3000)
            for Ms in (1, 8, 32, 64, 128, 160, 192, 240, 256):
                xs, sxs = si.make_activations(Ms, H, 1000 + Ms, device=dev)
                shs = torch.full((Ms,), 0.05, device=dev)
                hqs = torch.empty(Ms, I, dtype=torch.uint8, device=dev)
                ys = torch.empty(Ms, H, dtype=torch.bfloat16, device=dev)
                t_sp = t_us(lambda: step_eager(blobs[:6], xs, sxs, shs, hqs, ys), 6)
                t_dn = t_us(lambda: step_eager(dense, xs, sxs, shs, hqs, ys), 6)
                a_sp, a_dn = algorithmic_bytes(Ms, H, I, I_d), algorithmic_bytes(Ms, H, I, I)
                sweep.append({"M": Ms, "spense_us": round(t_sp, 2), "dense_us": round(t_dn, 2),
                              "speedup_vs_dense": round(t_dn / t_sp, 3),
                              "spense_gbs": round(a_sp / t_sp / 1e3, 1), "spense_frac_of_hbm_peak": round(a_sp / t_sp / 1e3 / peak, 3),
                              "dense_gbs": round(a_dn / t_dn / 1e3, 1), "dense_frac_of_hbm_peak": round(a_dn / t_dn / 1e3 / peak, 3),
                              "tokens_per_s_64_layers": round(Ms / (64 * t_sp * 1e-6), 1)})
            extras["sweep"] = sweep
            extras["byte_ratio_bound"] = round(1.0 / (P_DENSE + 0.625 * (1 - P_DENSE)), 4)
            del dense
            torch.cuda.empty_cache()
            # (measured BEFORE the prefill rows: seconds of tensor-bound work leave the board power-capped, which inflated
            # the dense row measured right after them)
            # configs[2]: one Seed-OSS-36B-shaped row, p = 50 % (the paper's "25 % sparsity" headline point, PAPER.md:226,
            # 238-240), M = 64, against the all-dense kernel on the same shape
            row = {}
            for p in (1.0, 0.5):
                bl = make_blobs(sp, si, dev, SEED_H, SEED_I, p, 4, 4000 + int(p * 100) * 10)
                xs, sxs = si.make_activations(64, SEED_H, 1064, device=dev)
                shs = torch.full((64,), 0.05, device=dev)
                hqs = torch.empty(64, SEED_I, dtype=torch.uint8, device=dev)
                ys = torch.empty(64, SEED_H, dtype=torch.bfloat16, device=dev)
                row[p] = (t_us(lambda: step_eager(bl, xs, sxs, shs, hqs, ys), 4), bl[0].I_dense)
                del bl
                torch.cuda.empty_cache()
            a50 = algorithmic_bytes(64, SEED_H, SEED_I, row[0.5][1])
            extras["seed_oss_36b_p50_M64"] = {"us_per_layer": round(row[0.5][0], 2), "dense_us_per_layer": round(row[1.0][0], 2),
                                              "speedup_vs_dense": round(row[1.0][0] / row[0.5][0], 3), "byte_ratio_bound": 1.231,
                                              "gbs": round(a50 / row[0.5][0] / 1e3, 1),
                                              "frac_of_hbm_peak": round(a50 / row[0.5][0] / 1e3 / peak, 3)}

        if not args.no_sweep:
            # configs[2] in full (dense fraction x token count) and configs[3] (the 64-layer stack), as in --report
            extras["seed_oss_36b_sweep"] = seed_sweep_rows(sp, si, dev, peak, nl=4)
            bl64 = blobs + make_blobs(sp, si, dev, H, I, P_DENSE, 64 - LAYERS, 6000)
            extras["qwen3_32b_stack"] = stack_rows(sp, si, dev, peak, bl64, ws)
            del bl64
            torch.cuda.empty_cache()

        # the HBM ceilings of this box in this run (after the decode rows, which seconds of full-rate streaming would heat;
        # before the tensor-bound prefill rows)
        probes = hbm_probes(sp, dev, timed_local, args.sustained_s)
        if sustained is not None and probes.get("copy_sustained_gbs"):
            sustained["frac_of_sustained_copy"] = sustained["hbm_gbs"] / probes["copy_sustained_gbs"]
            sustained["frac_of_sustained_read_probe"] = sustained["hbm_gbs"] / probes["read_probe_sustained_gbs"]
        if not args.no_sweep:
            # configs[4]: prefill-shaped GEMMs against the FP8 dense peak MEASURED on this box
            dense = make_blobs(sp, si, dev, H, I, 1.0, 1, 3000)
            extras["fp8_peak"] = fp8_dense_peak(sp, si, dev, dense, ws)
            del dense
            torch.cuda.empty_cache()
            fp8 = extras["fp8_peak"].get("scaled_mm_8192_tflops") or 2 * bf16_peak
            extras["prefill_shaped"] = prefill_rows(sp, si, dev, blobs, ws, fp8)
    sampler.stop()

    if rank == 0:
        achieved = algo / (us_layer * 1e-6) / 1e9
        _, info = sp.spense_schedule(H, I, I_d, M, 0)
        rounds = -(-info["blocks"] // info["blocks_per_launch"])
        line = {
            "metric": "spense_fp8_mlp_us_per_layer", "value": replicas.whole_job_us_per_layer(ms_step, LAYERS, world), "unit": "us/layer",
            "n_gpus": world, "steps": args.steps, "warmup": warmup, "ms_per_step": ms_step,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f8e4m3", "data": "synthetic",
            "config": config_of(M, I_d, world),
            "hbm_gbs": achieved,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": traffic_from_profile(M), "traffic_source": os.path.relpath(TRAFFIC_CSV, ROOT) if M == TRAFFIC_M else None,
                         "peak_source": peak_src,
                         "peak_read_gbs": probes["read_probe_gbs"], "frac_of_read_probe": achieved / probes["read_probe_gbs"],
                         "nominal_gbs": NOMINAL_HBM_GBS, "frac_of_nominal": achieved / NOMINAL_HBM_GBS,
                         "probes": probes,
                         "kernel": "spense_gemm_kernel (gate_up + down launches of one layer)",
                         "algorithmic_bytes_per_layer": algo},
            "sustained": sustained,
            "e2e": {"value": ms_e2e * 1e3 / LAYERS / world, "unit": "us/layer", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "call": "spense_mlp_stack_host: per step one H2D of x + scales, LAYERS x spense_mlp, one D2H of y, one synchronise"},
            "gpu_launches": 2 * rounds * LAYERS * args.steps,
            "clocks": clocks,
        }
        line.update(extras)
        if not args.no_cpu and world == 1:
            line["cpu_baseline"] = cpu_baseline(M)
        elif not args.no_cpu:
            line["cpu_baseline"] = None
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
