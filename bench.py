#!/usr/bin/env python
"""bench.py -- throughput of the protected GEMM hot path (encode A, encode B, encoded tcgen05 GEMM with fused
checksum epilogue, detect / locate / correct) on B200, through the C ABI.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--dtype bf16|f32] [--impl ours|reference]

One "step" = one pass of the whole path over one 4096^3 product (BASELINE.json configs[2], the configuration the
TFLOP/s metric is quoted on) with the faults of one of the paper's scenarios a-f injected, rotating.
Prints ONE JSON line (see DESIGN.md "Measurement" for every key).  `--impl reference` times the CPU fp64 oracle.
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
sys.path.insert(0, ROOT)

N_DEFAULT = 4096
SCENARIOS = ("a", "b", "c", "d", "e", "f")
ROTATE = 4  # resident input / output sets the steps rotate over: 4 x ~130 MB > 126 MB of L2


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1200)
    ap.add_argument("--warmup", type=int, default=24)
    ap.add_argument("--dtype", default="bf16", choices=["bf16", "f32"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--size", type=int, default=N_DEFAULT, help="n = k = m")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return {"hbm": p["hbm_gbs"], "bf16": p["bf16_tflops"], "bf16_sustained": p.get("bf16_tflops_sustained"), "src": "measured"}
    return {"hbm": 6650.0, "bf16": 1590.0, "bf16_sustained": 1400.0, "src": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md clocks line)."""

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
            "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for i, nm in enumerate(names) if any(len(r) >= 6 and r[2 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons, "samples": len(sm)}


# -------------------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands, on the host cores, on a bounded sample of the workload
# -------------------------------------------------------------------------------------------------------------
def oracle_sample_step(A_h, B_h, faults, O):
    """The oracle's whole path (encode, inject, product, decode) on a row slab of A against all of B."""
    rep = O.protected_matmul(A_h, B_h, faults=faults, level=1)
    return rep


def time_oracle(size, dtype, steps, warmup, rows):
    import numpy as np
    from oracle import gecc_oracle as O
    from paper_2508_04355_b200 import inputs as I
    A_h, B_h = I.make_operands(rows, size, size, seed=0, dtype=dtype)
    times, ok = [], 0
    for s in range(warmup + steps):
        faults = I.draw_faults(rows, size, size, I.SCENARIOS[SCENARIOS[s % 6]], seed=100 + s)
        t0 = time.perf_counter()
        rep = oracle_sample_step(A_h, B_h, faults, O)
        dt = time.perf_counter() - t0
        if s >= warmup:
            times.append(dt)
            ok += rep.verdict == O.CORRECTED
    t = sum(times) / len(times)
    try:
        from threadpoolctl import threadpool_info
        cores = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        cores = os.cpu_count() or 1
    return {"value": 2.0 * rows * size * size / t / 1e12, "unit": "TFLOP/s", "cores": int(cores), "kind": "oracle",
            "sample": f"whole oracle path (encode, inject, fp64 product, decode level X) on a {rows}-row slab of A x full B "
                      f"({rows}x{size}x{size}), mean of {len(times)} steps, scenarios a-f rotating",
            "ms_per_step": t * 1e3, "correction_rate": ok / len(times)}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    rows = 256
    r = time_oracle(args.size, args.dtype, args.steps, max(args.warmup, 1), rows)
    line = {"impl": "reference", "metric": "protected_gemm_tflops", "value": r["value"], "unit": "TFLOP/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"square GEMM n=k=m={args.size}, {args.dtype} inputs i.i.d. N(0,1), faults of scenarios a-f rotating "
                                   f"(BASELINE.json configs[2]); each reference step is a {rows}-row slab of it"},
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "correction_rate": r["correction_rate"], "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# -------------------------------------------------------------------------------------------------------------
# our arm: the CUDA path through the C ABI
# -------------------------------------------------------------------------------------------------------------
# dram__bytes_read.sum + dram__bytes_write.sum of one gecc_gemm_kernel launch from the `ncu --set full` capture summarised
# in profiles/ (per dtype at n = k = m = 4096); None until captured.
NCU_GEMM_TRAFFIC = {("bf16", 4096): 178.6e6, ("f32", 4096): 972.2e6}  # bytes per launch, profiles/r01g_kernels_full.md


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2508_04355_b200 import binding as G
    from paper_2508_04355_b200 import inputs as I

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (there is no CPU fallback for the product path)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    G.load()
    dev = torch.device("cuda", local)
    n = k = m = args.size
    tdt = torch.bfloat16 if args.dtype == "bf16" else torch.float32
    peaks = load_peaks()

    # independent products per rank (row shards of a larger A are independent codes; no collective)
    gen = torch.Generator(device=dev)
    gen.manual_seed(1234 + rank)
    sets = []
    for r in range(ROTATE):
        A = torch.randn(n, k, device=dev, generator=gen).to(tdt)
        B = torch.randn(k, m, device=dev, generator=gen).to(tdt)
        sets.append((A, B, G.Buffers(n, k, m, tdt, device=dev)))
    total = args.warmup + args.steps
    NF = 48  # distinct fault lists, cycled (scenario of list i is a-f by i % 6)
    fault_cycle = [I.draw_faults(n, k, m, I.SCENARIOS[SCENARIOS[i % 6]], seed=777 + 13 * i + 1000 * rank) for i in range(NF)]
    fault_cycle_dev = [G.faults_to_device(f, dev) for f in fault_cycle]
    fault_lists = [fault_cycle[s % NF] for s in range(total)]
    fault_devs = [fault_cycle_dev[s % NF] for s in range(total)]
    reports = torch.zeros(total, sets[0][2].report.numel(), dtype=torch.uint8, device=dev)

    def step(s):
        A, B, buf = sets[s % ROTATE]
        G.protected_matmul(A, B, buf, faults=fault_lists[s], level=1, faults_dev=fault_devs[s], report=reports[s])

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, count, first=0):
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for s in range(first, first + count):
            fn(s)
        e1.record()
        barrier()
        return e0.elapsed_time(e1)  # ms

    # ---- whole path, inputs resident in HBM ----
    for s in range(args.warmup):
        step(s)
    sampler = ClockSampler(local)
    sampler.start()
    ms_total = timed(step, args.steps, first=args.warmup)
    clocks = sampler.stop()
    t = torch.tensor([ms_total], device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_step = float(t.item()) / args.steps
    flops = 2.0 * n * k * m
    value = world * flops / (ms_step * 1e-3) / 1e12

    # correction rate over the timed steps: verdict CORRECTED and located set = injected set
    import ctypes
    ok = 0
    raw_reports = reports.cpu().numpy()
    for s in range(args.warmup, total):
        rep = G.GeccReport.from_buffer_copy(raw_reports[s].tobytes()[: ctypes.sizeof(G.GeccReport)])
        ok += int(rep.verdict == G.CORRECTED and rep.located() == sorted((f[0], f[1], f[2]) for f in fault_lists[s]))
    rate = ok / args.steps

    # ---- stage split and comparison GEMMs (same rotation, device timed) ----

    def gemm_prot(s):
        A, B, buf = sets[s % ROTATE]
        G.gecc_matmul_protected(A, buf.A_par, buf.A_lo, buf.A_par_lo, B, buf.B_par, buf.B_lo, buf.B_par_lo, buf.C, buf.P_r, buf.P_c, buf.P_g,
                                None, 0, buf.workspace, sumsq_a=buf.sumsq_a, sumsq_b=buf.sumsq_b, report=buf.report)

    def gemm_plain(s):
        A, B, buf = sets[s % ROTATE]
        G.gecc_matmul_plain(A, buf.A_lo, B, buf.B_lo, buf.C)

    def gemm_cublas(s):
        A, B, buf = sets[s % ROTATE]
        torch.matmul(A, B)

    def enc(s):
        A, B, buf = sets[s % ROTATE]
        G.gecc_encode(G.GECC_LEFT, A, buf.A_par, buf.A_par_lo, buf.A_lo, buf.A_par64, buf.sumsq_a, buf.workspace)
        G.gecc_encode(G.GECC_RIGHT, B, buf.B_par, buf.B_par_lo, buf.B_lo, buf.B_par64, buf.sumsq_b, buf.workspace)

    def dec_clean(s):
        A, B, buf = sets[s % ROTATE]
        G.gecc_decode_correct(buf.code, n, k, m, buf.C, buf.P_r, buf.P_c, None, buf.sumsq_a, buf.sumsq_b, 1, A, buf.A_lo, buf.A_par64,
                              B, buf.B_lo, buf.B_par64, buf.report, buf.workspace)

    def step_clean(s):
        A, B, buf = sets[s % ROTATE]
        G.protected_matmul(A, B, buf, faults=(), level=1)

    def enc_a(s):
        A, B, buf = sets[s % ROTATE]
        G.gecc_encode(G.GECC_LEFT, A, buf.A_par, buf.A_par_lo, buf.A_lo, buf.A_par64, buf.sumsq_a, buf.workspace)

    def enc_b(s):
        A, B, buf = sets[s % ROTATE]
        G.gecc_encode(G.GECC_RIGHT, B, buf.B_par, buf.B_par_lo, buf.B_lo, buf.B_par64, buf.sumsq_b, buf.workspace)

    def syn_unfused(s):
        A, B, buf = sets[s % ROTATE]
        G.gecc_syndrome_unfused(buf.code, k, buf.C, buf.workspace)

    def timed_graph(fn, count):
        """Device time per call with the CPU launch cost taken out: `count` calls captured in a CUDA graph, replayed."""
        side = torch.cuda.Stream(device=dev)
        with torch.cuda.stream(side):
            for s in range(ROTATE):
                fn(s)
            torch.cuda.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=side):
                for s in range(count):
                    fn(s)
        torch.cuda.synchronize()
        graph.replay()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(5):
            graph.replay()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / (5 * count)

    split = {}
    if tdt == torch.float32:
        torch.backends.cuda.matmul.allow_tf32 = False
    reps = 24
    for name, fn in (("gemm_protected", gemm_prot), ("gemm_plain", gemm_plain), ("cublas", gemm_cublas), ("encode", enc),
                     ("encode_a", enc_a), ("encode_b", enc_b), ("step_fault_free", step_clean), ("decode_fault_free", dec_clean),
                     ("syndrome_unfused", syn_unfused)):
        split[name] = timed_graph(fn, reps)
    ms_gemm = split["gemm_protected"]

    # ---- end to end: host buffers in, corrected product and report out, copies inside the timed region ----
    A0, B0, buf0 = sets[0]
    hA = torch.empty(A0.shape, dtype=tdt, pin_memory=True).copy_(A0)
    hB = torch.empty(B0.shape, dtype=tdt, pin_memory=True).copy_(B0)
    hC = torch.empty(n, m, dtype=torch.float32, pin_memory=True)
    hR = torch.empty(reports.shape[1], dtype=torch.uint8, pin_memory=True)

    def step_e2e(s):
        A, B, buf = sets[s % ROTATE]
        A.copy_(hA, non_blocking=True)
        B.copy_(hB, non_blocking=True)
        G.protected_matmul(A, B, buf, faults=fault_lists[s], level=1, faults_dev=fault_devs[s], report=reports[s])
        hC.copy_(buf.C, non_blocking=True)
        hR.copy_(reports[s], non_blocking=True)

    for s in range(2):
        step_e2e(s)
    e2e_steps = min(args.steps, 12)
    t2 = torch.tensor([timed(step_e2e, e2e_steps, first=args.warmup)], device=dev)
    if world > 1:
        dist.all_reduce(t2, op=dist.ReduceOp.MAX)
    ms_e2e = float(t2.item()) / e2e_steps
    h2d = hA.numel() * hA.element_size() + hB.numel() * hB.element_size()
    d2h = hC.numel() * 4 + hR.numel()

    if rank == 0:
        if args.dtype == "bf16":
            peak, exec_flops, peak_note = peaks["bf16"], flops, f"bf16 dense, {peaks['src']} (burst)"
        else:  # 3xTF32 executes three tf32 MMAs per product; tf32 peak = measured bf16 peak x nominal ratio 1.1 / 2.25
            peak, exec_flops, peak_note = peaks["bf16"] * 1.1 / 2.25, 3.0 * flops, f"tf32 dense = bf16 {peaks['src']} x 1.1/2.25; achieved counts the 3 tf32 passes"
        achieved = exec_flops / (ms_gemm * 1e-3) / 1e12
        n_launch = sum(G.launches_per_call(len(fault_lists[s]), 1) for s in range(args.warmup, total))
        line = {
            "metric": "protected_gemm_tflops", "value": value, "unit": "TFLOP/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
            "config": {"workload": f"square GEMM n=k=m={n}, {args.dtype} inputs i.i.d. N(0,1) with fp32 accumulation, faults of scenarios a-f "
                                   f"(PAPER.md:241) rotating, decoder level X (BASELINE.json configs[2])",
                       "l2": f"steps rotate over {ROTATE} resident operand/output sets (> 126 MB L2 in total)", "parallelism": f"independent products x{world}"},
            "roofline": {"bound": "tensor", "kernel": "gecc_gemm_kernel (protected)", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                         "frac": achieved / peak, "traffic": NCU_GEMM_TRAFFIC.get((args.dtype, n)), "peak_note": peak_note,
                         "ms_per_launch": ms_gemm,
                         # the launches are timed back to back (graph replay), i.e. under the sustained clocks: for context
                         "frac_of_sustained_peak": (achieved / peaks["bf16_sustained"]) if (args.dtype == "bf16" and peaks.get("bf16_sustained")) else None},
            "e2e": {"value": world * flops / (ms_e2e * 1e-3) / 1e12, "unit": "TFLOP/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": ms_e2e},
            "gpu_launches": n_launch,
            "clocks": clocks,
            "correction_rate": rate,
            "split_ms": split, "split_note": "device time per call, CUDA-graph replay of 24 calls over the rotating buffer sets",
            "overhead_pct": {"vs_own_plain_gemm": 100.0 * (ms_step / split["gemm_plain"] - 1.0), "vs_cublas": 100.0 * (ms_step / split["cublas"] - 1.0),
                             "fault_free_vs_own_plain_gemm": 100.0 * (split["step_fault_free"] / split["gemm_plain"] - 1.0),
                             "gemm_only_vs_own_plain_gemm": 100.0 * (ms_gemm / split["gemm_plain"] - 1.0)},
            "encode_hbm": {"achieved_gbs": (n * k + k * m) * (2 if args.dtype == "bf16" else 8) / (split["encode"] * 1e-3) / 1e9, "peak_gbs": peaks["hbm"],
                           "frac": (n * k + k * m) * (2 if args.dtype == "bf16" else 8) / (split["encode"] * 1e-3) / 1e9 / peaks["hbm"],
                           "bytes": "operand bytes read once (+ the fp32 lo planes written)"},
            "syndrome_hbm": {"achieved_gbs": 4.0 * n * m / (split["syndrome_unfused"] * 1e-3) / 1e9, "peak_gbs": peaks["hbm"],
                             "frac": 4.0 * n * m / (split["syndrome_unfused"] * 1e-3) / 1e9 / peaks["hbm"],
                             "bytes": "stored C (fp32) read once by gecc_syndrome_unfused (the detection sums of a C at rest)"},
        }
        if world == 1 and not args.no_cpu_baseline:
            cb = time_oracle(n, args.dtype, steps=4, warmup=1, rows=1024)
            line["cpu_baseline"] = {kk: cb[kk] for kk in ("value", "unit", "cores", "kind", "sample")}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
