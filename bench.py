#!/usr/bin/env python
"""bench.py -- Spense FP8 GLU-MLP decode step on B200 (BASELINE.json metric: us/layer + HBM GB/s vs peak,
speedup vs the library's own all-dense FP8 kernel).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--M 64] [--no-sweep]

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
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

H, I, P_DENSE = 5120, 25600, 0.25
LAYERS = 8
# dram__bytes_read.sum + dram__bytes_write.sum of the two spense_gemm_kernel launches of one layer at
# M=64, from the committed ncu capture (profiles/); per layer, like `achieved`.
NCU_TRAFFIC_BYTES_PER_LAYER = 286584960   # r01_traffic_app_replay_M64.csv: 16 launches = 8 layers, read + write


def algorithmic_bytes(M: int, I_d: int) -> int:
    """SURVEY.md 8(d) / DESIGN.md: weights streamed once + activations the method must move."""
    I_s = I - I_d
    w = 3 * H * (I_d + I_s * 0.625)
    act = M * H + 4 * M + 2 * M * I + 2 * M * H     # X, s_x, Hq written + read, Y bf16
    return int(w + act)


def read_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi polled every 20 ms in the background; every line is stamped with the host time it arrived, so
    the samples that fall inside the timed region can be picked out afterwards."""
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

    def stop(self, t0=None, t1=None):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"], "samples": 0}
        self.p.terminate()
        self.t.join(timeout=2)
        inside = [l for (t, l) in self.lines if t0 is None or (t0 <= t <= t1 + 0.02)]
        where = "timed region"
        if not inside:                                   # region shorter than the polling period: the load around it
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


def cpu_oracle_sample(M: int, seconds_hint: float = 20.0):
    """Time the oracle, as it stands, on a bounded slice of the same workload: I_sample intermediate
    indices (same 75/25 sparse/dense split) at full H and M; scaled to one layer by I / I_sample."""
    import numpy as np
    import spense_inputs as si
    from oracle import spense_oracle as o
    I_sample = 2560
    L = si.make_layer(H, I_sample, P_DENSE, seed=1001)
    x, sx = si.make_activations(M, H, seed=1000 + M)
    c = o.pack_canonical(L.wgate.numpy(), L.wup.numpy(), L.wdown.numpy(), L.perm.numpy(), L.I_dense)
    wg, wu, wd = o.unpack_canonical(c)
    s_h = np.full(M, 0.05, np.float32)
    t0 = time.perf_counter()
    reps = 0
    while True:
        o.mlp(x.numpy(), sx.numpy(), wg, wu, wd, L.w_scale, s_h)
        reps += 1
        if time.perf_counter() - t0 > seconds_hint / 4 or reps >= 8:
            break
    dt = (time.perf_counter() - t0) / reps
    us_per_layer = dt * 1e6 * (I / I_sample)
    import torch
    cores = torch.get_num_threads()
    return {"value": us_per_layer, "unit": "us/layer", "cores": int(os.cpu_count() if cores is None else cores),
            "kind": "oracle",
            "sample": f"oracle.mlp (decode E4M3 -> float64 GEMMs -> SiLU*up -> requant -> down) on a slice of "
                      f"{I_sample}/{I} intermediate indices at full H={H}, M={M}, {reps} reps, scaled by {I // I_sample}x"}


def run_reference(args):
    """--impl reference: for this tier the reference arm is the oracle on the host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    t0 = time.perf_counter()
    steps = []
    for i in range(args.warmup + args.steps):
        r = cpu_oracle_sample(args.M, seconds_hint=6.0)
        if i >= args.warmup:
            steps.append(r)
        if time.perf_counter() - t0 > 150:
            break
    steps = steps or [r]
    v = sum(s["value"] for s in steps) / len(steps)
    base = steps[-1]
    line = {"impl": "reference", "metric": "spense_fp8_mlp_us_per_layer", "value": v, "unit": "us/layer",
            "n_gpus": args.gpus, "steps": len(steps), "warmup": args.warmup, "ms_per_step": v * LAYERS / 1e3,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"qwen3_32b_mlp_layer H={H} I={I} p=25% M={args.M} (oracle on a bounded slice)"},
            "cpu_baseline": {"value": v, "unit": "us/layer", "cores": base["cores"], "kind": "oracle", "sample": base["sample"]},
            "e2e": {"value": v, "unit": "us/layer", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_report(args):
    """--report: the other BASELINE.json configs (context rows, not the bench line): Seed-OSS-36B shape
    dense-fraction sweep, the 64-layer Qwen3-32B-shaped stack, prefill-shaped GEMMs.  Writes one JSON
    object to stdout and to gpurun_out/report.json.  Same timing rules as the bench line (CUDA graph,
    CUDA events, layers rotate so every weight byte streams from HBM)."""
    import torch
    import spense_inputs as si
    from paper_2606_10445_b200 import build, spense as sp
    build.build()
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    peak, _ = read_peaks()
    out = {"hbm_peak_gbs": peak}

    def blobs_of(h, i, p, n, seed0, i_dense=None):
        res = []
        for k in range(n):
            L = si.make_layer(h, i, p, seed0 + k, device=dev, I_dense=i_dense)
            res.append(sp.spense_pack(L.wgate, L.wup, L.wdown, L.w_scale, L.perm, L.I_dense))
            del L
        torch.cuda.empty_cache()
        return res

    def graph_time(fn, reps=20, warm=5):
        fn(); torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            with torch.cuda.graph(g, stream=s):
                fn()
        torch.cuda.current_stream().wait_stream(s)
        for _ in range(warm):
            g.replay()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            g.replay()
        e1.record(); torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e3 / reps          # us per replay

    def w_bytes(h, i, i_d):
        return 3 * h * (i_d + (i - i_d) * 0.625)

    def act_bytes(m, h, i):
        return m * h + 4 * m + 2 * m * i + 2 * m * h

    # ---- config 3: Seed-OSS-36B-shaped layer, p sweep x M sweep, speedup vs the all-dense kernel
    h, i = 5120, 27648
    rows, dense_t = [], {}
    for p in (1.0, 0.0, 0.10, 0.25, 0.50):
        nl = 5
        bl = blobs_of(h, i, p, nl, 4000 + int(p * 100) * 10)
        i_d = bl[0].I_dense
        ws = sp.spense_workspace(bl[0], 256)
        for m in (1, 16, 64, 256):
            x, sx = si.make_activations(m, h, 1000 + m, device=dev)
            sh = torch.full((m,), 0.05, device=dev)
            hq = torch.empty(m, i, dtype=torch.uint8, device=dev)
            y = torch.empty(m, h, dtype=torch.bfloat16, device=dev)
            t = graph_time(lambda: [sp.spense_mlp(b, x, sx, sh, ws, hq_scratch=hq, y=y, next_layer=bl[(k + 1) % nl])
                                    for k, b in enumerate(bl)]) / nl
            if p == 1.0:
                dense_t[m] = t
            algo = w_bytes(h, i, i_d) + act_bytes(m, h, i)
            rows.append({"p": p, "I_dense": i_d, "M": m, "us_per_layer": round(t, 2), "gbs": round(algo / t / 1e3, 1),
                         "frac_of_hbm_peak": round(algo / t / 1e3 / peak, 3),
                         "speedup_vs_dense": round(dense_t[m] / t, 3),
                         "byte_ratio_bound": round(w_bytes(h, i, i) / w_bytes(h, i, i_d), 3)})
        del bl, ws
        torch.cuda.empty_cache()
    out["seed_oss_36b_sweep"] = rows

    # ---- config 4: 64 consecutive Qwen3-32B-shaped layers (18 GB of blobs), one CUDA graph, tokens/s
    nl = 64
    bl = blobs_of(H, I, P_DENSE, nl, 6000)
    ws = sp.spense_workspace(bl[0], 256)
    stack = []
    for m in (32, 128):
        x, sx = si.make_activations(m, H, 1000 + m, device=dev)
        sh = torch.full((m,), 0.05, device=dev)
        hq = torch.empty(m, I, dtype=torch.uint8, device=dev)
        y = torch.empty(m, H, dtype=torch.bfloat16, device=dev)
        t = graph_time(lambda: [sp.spense_mlp(b, x, sx, sh, ws, hq_scratch=hq, y=y, next_layer=bl[(k + 1) % nl])
                                for k, b in enumerate(bl)], reps=10, warm=3)
        algo = nl * (w_bytes(H, I, bl[0].I_dense) + act_bytes(m, H, I))
        stack.append({"M": m, "layers": nl, "ms_per_stack": round(t / 1e3, 4), "us_per_layer": round(t / nl, 2),
                      "tokens_per_s": round(m / (t * 1e-6), 1), "gbs": round(algo / t / 1e3, 1),
                      "frac_of_hbm_peak": round(algo / t / 1e3 / peak, 3)})
    out["qwen3_32b_stack"] = stack

    # ---- config 5: prefill-shaped GEMMs, gate_up and down separately (the decode kernel run over 128-token
    # blocks: weights are re-streamed per block, so this is far from the tensor roofline -- NEXT-3)
    pre = []
    for m in (2048, 8192):
        x, sx = si.make_activations(m, H, 1000 + m, device=dev)
        sh = torch.full((m,), 0.05, device=dev)
        hq = torch.empty(m, I, dtype=torch.uint8, device=dev)
        y = torch.empty(m, H, dtype=torch.bfloat16, device=dev)
        four = bl[:4]
        t_gu = graph_time(lambda: [sp.spense_gate_up(b, x, sx, sh, ws, hq=hq) for b in four], reps=3, warm=1) / 4
        t_dn = graph_time(lambda: [sp.spense_down(b, hq, sh, ws, y=y) for b in four], reps=3, warm=1) / 4
        i_d = bl[0].I_dense
        macs_gu = m * 2 * H * (i_d + (I - i_d) / 2)          # executed MACs (2:4 tiles do half)
        macs_dn = m * H * (i_d + (I - i_d) / 2)
        pre.append({"M": m, "gate_up_us": round(t_gu, 1), "down_us": round(t_dn, 1),
                    "gate_up_executed_tflops": round(2 * macs_gu / t_gu / 1e6, 1),
                    "down_executed_tflops": round(2 * macs_dn / t_dn / 1e6, 1),
                    "gate_up_dense_equiv_tflops": round(2 * m * 2 * H * I / t_gu / 1e6, 1),
                    "down_dense_equiv_tflops": round(2 * m * H * I / t_dn / 1e6, 1),
                    "fp8_dense_peak_tflops_nominal": 4500.0})
    out["prefill_shaped"] = pre
    os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
    with open(os.path.join(ROOT, "gpurun_out", "report.json"), "w") as f:
        json.dump(out, f, indent=1)
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--report", action="store_true")
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=400)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="spense")
    ap.add_argument("--M", type=int, default=64)
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
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

    def make_blobs(p, n, seed0):
        out = []
        for i in range(n):
            L = si.make_layer(H, I, p, seed0 + i, device=dev)
            out.append(sp.spense_pack(L.wgate, L.wup, L.wdown, L.w_scale, L.perm, L.I_dense))
            del L
        torch.cuda.empty_cache()
        return out

    blobs = make_blobs(P_DENSE, LAYERS, 2000)
    I_d = blobs[0].I_dense
    x, sx = si.make_activations(M, H, 1000 + M, device=dev)
    sh = torch.full((M,), 0.05, device=dev)
    ws = sp.spense_workspace(blobs[0], max(M, 256))
    ws_dense = None                                      # the all-dense baseline has its own schedule and workspace size
    hq = torch.empty(M, I, dtype=torch.uint8, device=dev)
    y = torch.empty(M, H, dtype=torch.bfloat16, device=dev)

    def step_eager(layers, xx, ssx, ssh, hqq, yy, wsp=None):
        wsp = ws if wsp is None else wsp
        for i, b in enumerate(layers):                   # the layer that runs next is named as an L2 prefetch hint
            sp.spense_mlp(b, xx, ssx, ssh, wsp, hq_scratch=hqq, y=yy, next_layer=layers[(i + 1) % len(layers)])

    def graph_of(fn):
        fn()                                             # warm: header cache, schedules, func attributes
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            fn()
            s.synchronize()
            with torch.cuda.graph(g, stream=s):
                fn()
        torch.cuda.current_stream().wait_stream(s)
        return g

    def time_steps(replay, steps, warmup, host_window=None):
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

    g_main = graph_of(lambda: step_eager(blobs, x, sx, sh, hq, y))
    sampler = ClockSampler(local)
    sampler.start()
    t_pre = time.time()
    while sampler.p is not None and sampler.n_samples() == 0 and time.time() - t_pre < 2.0:
        g_main.replay()                                  # untimed pre-roll under load until nvidia-smi is polling
        torch.cuda.synchronize()
    window = [None, None]
    ms_step = time_steps(g_main.replay, args.steps, max(args.warmup, 3), window)
    clocks = sampler.stop(window[0], window[1])
    us_layer = ms_step * 1e3 / LAYERS

    # ---- per-kernel view and the all-dense baseline kernel (same library, I_dense = I), rank 0 extras
    extras = {}
    peak, peak_src = read_peaks()
    if rank == 0:
        def t_us(fn, n=LAYERS):
            g = graph_of(fn)
            return time_steps(g.replay, 20, 5) * 1e3 / n
        extras["gate_up_us"] = t_us(lambda: [sp.spense_gate_up(b, x, sx, sh, ws, hq=hq) for b in blobs])
        extras["down_us"] = t_us(lambda: [sp.spense_down(b, hq, sh, ws, y=y) for b in blobs])
        # NEXT-1: the same layers with dynamic per-token requant (gate_up -> row requant kernel -> down)
        h32 = torch.empty(M, I, dtype=torch.float32, device=dev)
        sh_dyn = torch.empty(M, device=dev)
        extras["dynamic_requant_us"] = t_us(lambda: [sp.spense_mlp_dyn(b, x, sx, ws, s_h=sh_dyn, hq_scratch=hq, h_scratch=h32, y=y,
                                                                       next_layer=blobs[(i + 1) % len(blobs)]) for i, b in enumerate(blobs)])
        del h32
        sweep = []
        if not args.no_sweep:
            dense = make_blobs(1.0, 6, 3000)
            ws_dense = sp.spense_workspace(dense[0], 256)
            for Ms in (1, 8, 32, 64, 128, 256):
                xs, sxs = si.make_activations(Ms, H, 1000 + Ms, device=dev)
                shs = torch.full((Ms,), 0.05, device=dev)
                hqs = torch.empty(Ms, I, dtype=torch.uint8, device=dev)
                ys = torch.empty(Ms, H, dtype=torch.bfloat16, device=dev)
                t_sp = t_us(lambda: step_eager(blobs[:6], xs, sxs, shs, hqs, ys), 6)
                t_dn = t_us(lambda: step_eager(dense, xs, sxs, shs, hqs, ys, ws_dense), 6)
                sweep.append({"M": Ms, "spense_us": round(t_sp, 2), "dense_us": round(t_dn, 2),
                              "speedup_vs_dense": round(t_dn / t_sp, 3),
                              "spense_gbs": round(algorithmic_bytes(Ms, I_d) / t_sp / 1e3, 1),
                              "dense_gbs": round(algorithmic_bytes(Ms, I) / t_dn / 1e3, 1),
                              "tokens_per_s_64_layers": round(Ms / (64 * t_sp * 1e-6), 1)})
            del dense
            torch.cuda.empty_cache()
        extras["sweep"] = sweep
        extras["byte_ratio_bound"] = round(1.0 / (P_DENSE + 0.625 * (1 - P_DENSE)), 4)

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D x, scales; D2H y, every layer
    hx = x.cpu().pin_memory(); hsx = sx.cpu().pin_memory(); hsh = sh.cpu().pin_memory()
    hy = torch.empty(M, H, dtype=torch.bfloat16).pin_memory()
    staging = dict(d_x=torch.empty_like(x), d_scales=torch.empty(2 * M, device=dev), d_hq=hq, d_y=y)

    def step_host():
        for i, b in enumerate(blobs):
            sp.spense_mlp_host(b, hx, hsx, hsh, hy, staging, ws, next_layer=blobs[(i + 1) % len(blobs)])
    ms_e2e = time_steps(step_host, max(5, args.steps // 5), 3)
    h2d = LAYERS * (M * H + 4 * M + 4 * M)
    d2h = LAYERS * (M * H * 2)

    if rank == 0:
        algo = algorithmic_bytes(M, I_d)
        achieved = algo / (us_layer * 1e-6) / 1e9
        line = {
            "metric": "spense_fp8_mlp_us_per_layer", "value": replicas.whole_job_us_per_layer(ms_step, LAYERS, world), "unit": "us/layer",
            "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f8e4m3", "data": "synthetic",
            "config": {"workload": f"qwen3_32b_mlp_layer H={H} I={I} p=25% (I_dense={I_d}) M={M}",
                       "layers_per_step": LAYERS, "launch": "CUDA graph of LAYERS x spense_mlp (2 PDL-chained kernels each)",
                       "l2": f"inputs larger than L2: {LAYERS} distinct packed layers = {LAYERS * (blobs[0].blob.numel()) / 1e9:.2f} GB rotate",
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "hbm_gbs": achieved,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": NCU_TRAFFIC_BYTES_PER_LAYER, "peak_source": peak_src,
                         "kernel": "spense_gemm_kernel (gate_up + down launches of one layer)",
                         "algorithmic_bytes_per_layer": algo},
            "e2e": {"value": ms_e2e * 1e3 / LAYERS / world, "unit": "us/layer", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": 2 * LAYERS * args.steps,
            "clocks": clocks,
        }
        line.update(extras)
        if not args.no_cpu and world == 1:
            line["cpu_baseline"] = cpu_oracle_sample(M)
        elif not args.no_cpu:
            line["cpu_baseline"] = None
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
