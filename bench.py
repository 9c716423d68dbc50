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
    ap.add_argument("--steps", type=int, default=24)
    ap.add_argument("--warmup", type=int, default=6)
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
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "50"],
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
