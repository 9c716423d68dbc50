#!/usr/bin/env python
"""bench.py -- throughput of the protected GEMM hot path (encode A and B, encoded tcgen05 GEMM with fused checksum
epilogue and in-product detection, locate / correct) on B200, through the C ABI.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--dtype bf16|f32] [--impl ours|reference]
                    [--size S | --shape n,k,m] [--trans-a] [--trans-b] [--std-b X] [--no-split] [--no-cpu-baseline]

One "step" = one pass of the whole path over one product (default 4096^3: BASELINE.json configs[2], the configuration
the TFLOP/s metric is quoted on) with the faults of one of the paper's scenarios a-f injected, rotating.
`--shape` / `--trans-*` time the transformer-shaped products of configs[3] (Y = X W, dX = dY W^T, dW = X^T dY).
Prints ONE JSON line (see DESIGN.md "Measurement" for every key).  `--impl reference` times the CPU fp64 oracle.
"""
from __future__ import annotations

import argparse
import ctypes
import json
import os
import statistics

import numpy as np
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

N_DEFAULT = 4096
SCENARIOS = ("a", "b", "c", "d", "e", "f")
ORACLE_ROWS = 512  # rows of A in one oracle sample step (cpu_baseline and --impl reference use the same slab)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1200)
    ap.add_argument("--warmup", type=int, default=24)
    ap.add_argument("--dtype", default="bf16", choices=["bf16", "f32"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--size", type=int, default=N_DEFAULT, help="n = k = m")
    ap.add_argument("--shape", default=None, help="n,k,m of the product C[n x m] = A[n x k] B[k x m] (overrides --size)")
    ap.add_argument("--trans-a", action="store_true", help="A is stored transposed (k x n): dW = X^T dY")
    ap.add_argument("--trans-b", action="store_true", help="B is stored transposed (m x k): dX = dY W^T")
    ap.add_argument("--std-b", type=float, default=1.0, help="standard deviation of B's entries (0.02 for config-3 weights)")
    ap.add_argument("--no-split", action="store_true", help="timed steps only: no stage split, no end-to-end leg (for ncu launch lists)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    a = ap.parse_args()
    a.n, a.k, a.m = (int(x) for x in a.shape.split(",")) if a.shape else (a.size, a.size, a.size)
    return a


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return {"hbm": p["hbm_gbs"], "bf16": p["bf16_tflops"], "bf16_sustained": p.get("bf16_tflops_sustained"), "src": "measured"}
    return {"hbm": 6650.0, "bf16": 1590.0, "bf16_sustained": 1400.0, "src": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled while the GPU section runs (B200_PROFILING.md clocks line)."""

    def __init__(self, index):
        self.index, self.rows, self.proc, self.marks = index, [], None, []

    def start(self):
        q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
            "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "10"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [x.strip() for x in line.split(",")]))

    def mark(self):
        self.marks.append(time.perf_counter())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"], "samples": 0}
        self.proc.terminate()
        self.thread.join(timeout=2)
        rows = [r for _, r in self.rows if len(r) >= 6]
        timed = [r for t, r in self.rows if len(r) >= 6 and len(self.marks) >= 2 and self.marks[0] <= t <= self.marks[1]]

        def col(rs, i):
            return [float(r[i]) for r in rs if r[i].replace(".", "").isdigit()]

        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for i, nm in enumerate(names) if any(r[2 + i].lower().startswith("active") for r in rows)]
        sm, mx, smt = col(rows, 0), col(rows, 1), col(timed, 0)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None, "reasons": reasons,
                "samples": len(sm), "samples_in_timed_loop": len(smt), "sm_mhz_timed_loop": statistics.median(smt) if smt else None,
                "note": "sampled every 10 ms over the whole GPU section (timed loop, stage split, end-to-end leg)"}


# -------------------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands, on the host cores, on a bounded sample of the workload
# -------------------------------------------------------------------------------------------------------------
def time_oracle(n, k, m, dtype, steps, warmup, rows, std_b=1.0):
    from oracle import gecc_oracle as O
    from paper_2508_04355_b200 import inputs as I
    rows = min(rows, n)
    A_h, B_h = I.make_operands(rows, k, m, seed=0, dtype=dtype, std_b=std_b)
    times, ok = [], 0
    for s in range(warmup + steps):
        faults = I.draw_faults(rows, k, m, I.SCENARIOS[SCENARIOS[s % 6]], seed=100 + s)
        t0 = time.perf_counter()
        rep = O.protected_matmul(A_h, B_h, faults=faults, level=1)   # encode, inject, fp64 product, decode level X
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
    return {"value": 2.0 * rows * k * m / t / 1e12, "unit": "TFLOP/s", "cores": int(cores), "kind": "oracle",
            "sample": f"whole oracle path (numpy fp64: encode, inject, product by BLAS dgemm, decode level X) on a {rows}-row slab of A x full B "
                      f"({rows}x{k}x{m}), mean of {len(times)} steps, scenarios a-f rotating",
            "ms_per_step": t * 1e3, "correction_rate": ok / len(times)}


def workload_text(a):
    lay = ("A^T stored, " if a.trans_a else "") + ("B^T stored, " if a.trans_b else "")
    cfg = "BASELINE.json configs[2]" if (a.n == a.k == a.m == 4096 and not a.trans_a and not a.trans_b) else \
          ("BASELINE.json configs[3] shapes" if a.shape else "BASELINE.json configs[4] sweep")
    return (f"GEMM n={a.n} k={a.k} m={a.m}, {lay}{a.dtype} inputs i.i.d. N(0,1)" + (f" (B: std {a.std_b})" if a.std_b != 1.0 else "") +
            f" with fp32 accumulation, faults of scenarios a-f (PAPER.md:241) rotating, decoder level X ({cfg})")


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    r = time_oracle(args.n, args.k, args.m, args.dtype, args.steps, max(args.warmup, 1), ORACLE_ROWS, args.std_b)
    line = {"impl": "reference", "metric": "protected_gemm_tflops", "value": r["value"], "unit": "TFLOP/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_text(args) + f"; each reference step is a {min(ORACLE_ROWS, args.n)}-row slab of it"},
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": "TFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "correction_rate": r["correction_rate"], "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# -------------------------------------------------------------------------------------------------------------
# our arm: the CUDA path through the C ABI
# -------------------------------------------------------------------------------------------------------------
# dram__bytes_read.sum + dram__bytes_write.sum of one gecc_gemm_kernel launch from the `ncu --set full` capture summarised
# in profiles/ (per dtype at n = k = m = 4096); None where not captured.
# dram__bytes_read.sum + dram__bytes_write.sum of gecc_gemm_kernel per launch, from `ncu --set full` captures: bf16 4096^3 mean of the six
# launches in profiles/r02_kernels_full.md (119.9 MB read + 53.1 MB written); fp32 4096^3 from profiles/r01g_kernels_full.md (not re-captured)
NCU_GEMM_TRAFFIC = {("bf16", 4096): 173.0e6, ("f32", 4096): 972.2e6}


def run_ours(args):
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
    n, k, m = args.n, args.k, args.m
    ta, tb = int(args.trans_a), int(args.trans_b)
    tdt = torch.bfloat16 if args.dtype == "bf16" else torch.float32
    es = 2 if args.dtype == "bf16" else 4
    peaks = load_peaks()
    sampler = ClockSampler(local)
    sampler.start()

    # resident operand / output sets the steps rotate over: together larger than the 126 MB L2
    per_set = (n * k + k * m) * es * (1 if args.dtype == "bf16" else 2) + 4 * n * m
    rotate = max(2, min(4, int(3.0e8 // per_set) + 1))
    # independent products per rank (row shards of a larger A are independent codes; no collective)
    gen = torch.Generator(device=dev)
    gen.manual_seed(1234 + rank)
    sets = []
    for r in range(rotate):
        A = torch.randn((k, n) if ta else (n, k), device=dev, generator=gen).to(tdt)
        B = (torch.randn((m, k) if tb else (k, m), device=dev, generator=gen) * args.std_b).to(tdt)
        sets.append((A, B, G.Buffers(n, k, m, tdt, device=dev, trans_a=ta, trans_b=tb)))
    oa, ob = sets[0][0].clone(), sets[0][1].clone()
    total = args.warmup + args.steps
    NF = 48  # distinct fault lists, cycled (scenario of list i is a-f by i % 6)
    fault_cycle = [I.draw_faults(n, k, m, I.SCENARIOS[SCENARIOS[i % 6]], seed=777 + 13 * i + 1000 * rank) for i in range(NF)]
    fault_cycle_dev = [G.faults_to_device(f, dev) for f in fault_cycle]
    fault_lists = [fault_cycle[s % NF] for s in range(total)]
    fault_devs = [fault_cycle_dev[s % NF] for s in range(total)]
    reports = torch.zeros(total, sets[0][2].report.numel(), dtype=torch.uint8, device=dev)

    def step(s):
        A, B, buf = sets[s % rotate]
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
    torch.cuda.synchronize()
    sampler.mark()
    ms_total = timed(step, args.steps, first=args.warmup)
    sampler.mark()
    t = torch.tensor([ms_total], device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_step = float(t.item()) / args.steps
    flops = 2.0 * n * k * m
    value = world * flops / (ms_step * 1e-3) / 1e12

    # correction rate over the timed steps: verdict CORRECTED and located set = injected set
    ok = 0
    raw_reports = reports.cpu().numpy()
    for s in range(args.warmup, total):
        rep = G.GeccReport.from_buffer_copy(raw_reports[s].tobytes()[: ctypes.sizeof(G.GeccReport)])
        ok += int(rep.verdict == G.CORRECTED and rep.located() == sorted((f[0], f[1], f[2]) for f in fault_lists[s]))
    rate = ok / args.steps

    # value check: one more step of every scenario on set 0, the corrected product against an untouched product of the
    # same operands (library GEMM on the fp32-widened originals, no TF32) and the operands against their originals (they are
    # patched in place and reused by every step: a decoder that located correctly but patched wrongly would show here)
    torch.backends.cuda.matmul.allow_tf32 = False
    A0, B0, buf0 = sets[0]
    ref = torch.matmul((oa.t() if ta else oa).float(), (ob.t() if tb else ob).float()) if float(n) * k * m <= 5e12 else None
    worst, restored = 0.0, True
    for i in range(6):
        G.protected_matmul(A0, B0, buf0, faults=fault_cycle[i], level=1, faults_dev=fault_cycle_dev[i])
        torch.cuda.synchronize()
        if ref is not None:
            worst = max(worst, float((buf0.C - ref).abs().max() / ref.abs().max()))
        if args.dtype == "bf16":
            restored = restored and bool(torch.equal(A0, oa)) and bool(torch.equal(B0, ob))
        else:
            restored = restored and float((A0 - oa).abs().max()) <= 2e-4 and float((B0 - ob).abs().max()) <= 2e-4
    value_check = {"max_rel_err_corrected_C": worst if ref is not None else None, "operands_restored": restored,
                   "vs": "torch.matmul of the fp32-widened original operands (TF32 off): max |c - ref| / max |ref| over one step of each scenario a-f; "
                         "operands compared with their originals after the decoder patched them back"}
    del ref

    line = {
        "metric": "protected_gemm_tflops", "value": value, "unit": "TFLOP/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
        "config": {"workload": workload_text(args),
                   "l2": f"steps rotate over {rotate} resident operand/output sets ({rotate * per_set / 1e6:.0f} MB in total, L2 is 126 MB)",
                   "parallelism": f"independent products x{world}"},
        "gpu_launches": sum(G.launches_per_call(len(fault_lists[s]), 1) for s in range(args.warmup, total)),
        "correction_rate": rate, "value_check": value_check,
    }

    if not args.no_split:
        # ---- stage split and comparison GEMMs (same rotation, device timed, CPU launch cost taken out by graph replay) ----
        def gemm_prot(s):
            A, B, buf = sets[s % rotate]
            G.gecc_matmul_protected(A, buf.A_par, buf.A_lo, buf.A_par_lo, B, buf.B_par, buf.B_lo, buf.B_par_lo, buf.C, buf.P_r, buf.P_c, buf.P_g,
                                    None, 0, buf.workspace, trans_a=ta, trans_b=tb, sumsq_a=buf.sumsq_a, sumsq_b=buf.sumsq_b, report=buf.report)

        def gemm_prot_nodetect(s):
            A, B, buf = sets[s % rotate]
            G.gecc_matmul_protected(A, buf.A_par, buf.A_lo, buf.A_par_lo, B, buf.B_par, buf.B_lo, buf.B_par_lo, buf.C, buf.P_r, buf.P_c, buf.P_g,
                                    None, 0, buf.workspace, trans_a=ta, trans_b=tb)

        def gemm_plain(s):
            A, B, buf = sets[s % rotate]
            G.gecc_matmul_plain(A, buf.A_lo, B, buf.B_lo, buf.C, trans_a=ta, trans_b=tb)

        def gemm_cublas(s):
            A, B, buf = sets[s % rotate]
            torch.matmul(A.t() if ta else A, B.t() if tb else B)

        def enc(s):
            A, B, buf = sets[s % rotate]
            G.gecc_encode_both(A, B, buf)

        def enc_a(s):
            A, B, buf = sets[s % rotate]
            G.gecc_encode(G.GECC_LEFT, A, buf.A_par, buf.A_par_lo, buf.A_lo, buf.A_par64, buf.sumsq_a, buf.workspace, trans=ta)

        def enc_b(s):
            A, B, buf = sets[s % rotate]
            G.gecc_encode(G.GECC_RIGHT, B, buf.B_par, buf.B_par_lo, buf.B_lo, buf.B_par64, buf.sumsq_b, buf.workspace, trans=tb)

        def step_clean(s):
            A, B, buf = sets[s % rotate]
            G.protected_matmul(A, B, buf, faults=(), level=1)

        def syn_unfused(s):
            A, B, buf = sets[s % rotate]
            G.gecc_syndrome_unfused(buf.code, k, buf.C, buf.workspace)

        def timed_graph(fn, count):
            """Device time per call with the CPU launch cost taken out: `count` calls captured in a CUDA graph, replayed."""
            side = torch.cuda.Stream(device=dev)
            with torch.cuda.stream(side):
                for s in range(rotate):
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
        reps = 24 if flops <= 3e11 else 8
        tests = [("gemm_protected", gemm_prot), ("gemm_protected_no_detection", gemm_prot_nodetect), ("gemm_plain", gemm_plain), ("cublas", gemm_cublas),
                 ("encode", enc), ("encode_a", enc_a), ("encode_b", enc_b), ("step_fault_free", step_clean), ("syndrome_unfused", syn_unfused)]
        for name, fn in tests:
            split[name] = timed_graph(fn, reps)
        ms_gemm = split["gemm_protected"]
        tf32_tflops = None
        if args.dtype == "f32":  # the TF32 peak of this box, measured: cuBLAS TF32 product of the same shape
            torch.backends.cuda.matmul.allow_tf32 = True
            split["cublas_tf32"] = timed_graph(gemm_cublas, reps)
            torch.backends.cuda.matmul.allow_tf32 = False
            tf32_tflops = flops / (split["cublas_tf32"] * 1e-3) / 1e12

        # decoder alone, per scenario class: in-kernel time between its first and last phase stamp (%globaltimer)
        dec_us = {}
        for i, scen in enumerate(SCENARIOS):
            vals = []
            for j in list(range(i, NF, 6))[:4]:
                G.protected_matmul(A0, B0, buf0, faults=fault_cycle[j], level=1, faults_dev=fault_cycle_dev[j])
                torch.cuda.synchronize()
                vals.append(sum(G.gecc_decode_phase_ns(buf0.code, n, k, m, buf0.workspace)) / 1e3)
            dec_us[scen] = statistics.median(vals)

        # ---- tile-local grid (one code per 128 x 128 block of C; include/gecc.h gecc_tl_*), same operands ----
        tile_local = None
        if not ta and not tb:
            tlb = G.TlBuffers(n, k, m, tdt, device=dev)
            rng = np.random.default_rng(99)
            tl_faults = []
            for b in range(min(16, (m + 127) // 128)):     # two errors in each of up to 16 blocks: far beyond the global code's budget
                r0, c0 = int(rng.integers(0, (n + 127) // 128)) * 128, b * 128
                i1, i2 = rng.choice(min(128, n - r0), 2, replace=False)
                j1, j2 = rng.choice(min(128, m - c0), 2, replace=False)
                tl_faults += [(I.KIND_C, r0 + int(i1), c0 + int(j1), 50.0), (I.KIND_C, r0 + int(i2), c0 + int(j2), -75.0)]
            tl_fdev = G.faults_to_device(tl_faults, dev)

            def tl_enc(s):
                A, B, _ = sets[s % rotate]
                G.gecc_tl_encode(A, B, tlb)

            def tl_mm(s):
                A, B, _ = sets[s % rotate]
                G.gecc_tl_matmul(A, B, tlb)

            def tl_dec(s):
                G.gecc_tl_decode(tlb)

            def tl_step_clean(s):
                A, B, _ = sets[s % rotate]
                G.tl_protected_matmul(A, B, tlb)

            def tl_step_faults(s):
                A, B, _ = sets[s % rotate]
                G.tl_protected_matmul(A, B, tlb, faults=tl_faults, faults_dev=tl_fdev)

            def tl_mm_faults(s):
                A, B, _ = sets[0]
                G.gecc_tl_matmul(A, B, tlb, tl_fdev, len(tl_faults))

            tl_split = {name: timed_graph(fn, reps) for name, fn in (("encode", tl_enc), ("gemm", tl_mm), ("decode_clean", tl_dec), ("step_fault_free", tl_step_clean),
                                                                   ("step_32_errors_in_16_blocks", tl_step_faults), ("gemm_with_the_32_faults_injected", tl_mm_faults))}
            tl_mm_faults(0)   # leaves the sums of a faulted product in the workspace: the decoder alone on 16 flagged blocks
            torch.cuda.synchronize()   # (timed_graph works on a side stream: the workspace serves one call at a time)
            tl_split["decode_16_flagged_blocks"] = timed_graph(tl_dec, reps)
            tl_step_faults(0)
            torch.cuda.synchronize()
            trep = G.read_tl_report(tlb.report)
            tl_ok = trep.verdict == G.CORRECTED and trep.located() == sorted((f[0], f[1], f[2]) for f in tl_faults)
            tl_err = float((tlb.C - torch.matmul(oa.float(), ob.float())).abs().max() / tlb.C.abs().max()) if float(n) * k * m <= 5e12 else None
            tile_local = {"split_ms": tl_split, "tflops_fault_free": flops / (tl_split["step_fault_free"] * 1e-3) / 1e12,
                          "tflops_32_errors": flops / (tl_split["step_32_errors_in_16_blocks"] * 1e-3) / 1e12,
                          "overhead_pct_fault_free_vs_own_plain_gemm": 100.0 * (tl_split["step_fault_free"] / split["gemm_plain"] - 1.0),
                          "all_32_errors_located_and_corrected": bool(tl_ok), "max_rel_err_corrected_C": tl_err,
                          "tau_block": [trep.tau[q] for q in range(4)],
                          "note": "one code per 128 x 128 block (weights 1..128, thresholds of a 128-line block); 3 launches: encode (both operands), product, decode; "
                                  "the step with 32 errors pays for the E3 injection hook in the product's epilogue (every chunk compares with all 32 faults), "
                                  "not for the decoder: compare decode_16_flagged_blocks with decode_clean"}
            del tlb

        # ---- end to end: host buffers in, corrected product and report out, copies inside the timed region; the copies of
        # step s + 1 (host to device) and of step s - 1 (device to host) overlap the compute of step s on their own streams ----
        hA = torch.empty(A0.shape, dtype=tdt, pin_memory=True).copy_(oa)
        hB = torch.empty(B0.shape, dtype=tdt, pin_memory=True).copy_(ob)
        hC = [torch.empty(n, m, dtype=torch.float32, pin_memory=True) for _ in range(2)]
        hR = [torch.empty(reports.shape[1], dtype=torch.uint8, pin_memory=True) for _ in range(2)]
        s_in, s_out, s_cmp = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev), torch.cuda.current_stream()
        ev_in = [torch.cuda.Event() for _ in range(rotate)]
        ev_done = [torch.cuda.Event() for _ in range(rotate)]
        ev_out = [torch.cuda.Event() for _ in range(rotate)]

        def e2e_step(s):
            A, B, buf = sets[s % rotate]
            with torch.cuda.stream(s_in):            # operands of step s: host -> device (after the set's last result has left)
                s_in.wait_event(ev_out[s % rotate])
                A.copy_(hA, non_blocking=True)
                B.copy_(hB, non_blocking=True)
                ev_in[s % rotate].record(s_in)
            s_cmp.wait_event(ev_in[s % rotate])
            G.protected_matmul(A, B, buf, faults=fault_lists[s % total], level=1, faults_dev=fault_devs[s % total], report=reports[s % total])
            ev_done[s % rotate].record(s_cmp)
            with torch.cuda.stream(s_out):           # corrected product and report: device -> host
                s_out.wait_event(ev_done[s % rotate])
                hC[s % 2].copy_(buf.C, non_blocking=True)
                hR[s % 2].copy_(reports[s % total], non_blocking=True)
                ev_out[s % rotate].record(s_out)

        def e2e_timed(count, first):
            barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for s in range(first, first + count):
                e2e_step(s)
            s_cmp.wait_stream(s_out)
            e1.record()
            barrier()
            return e0.elapsed_time(e1)

        e2e_timed(3, 0)
        e2e_steps = max(3, min(args.steps, 16))
        t2 = torch.tensor([e2e_timed(e2e_steps, args.warmup)], device=dev)
        if world > 1:
            dist.all_reduce(t2, op=dist.ReduceOp.MAX)
        ms_e2e = float(t2.item()) / e2e_steps
        h2d = hA.numel() * hA.element_size() + hB.numel() * hB.element_size()
        d2h = hC[0].numel() * 4 + hR[0].numel()

        if args.dtype == "bf16":
            peak, exec_flops, peak_note = peaks["bf16"], flops, f"bf16 dense, {peaks['src']} (burst: the kernel is timed alone)"
        else:  # 3xTF32 executes three tf32 MMAs per product
            nominal = peaks["bf16"] * 1.1 / 2.25
            peak = tf32_tflops if tf32_tflops and tf32_tflops > 0.5 * nominal else nominal
            exec_flops = 3.0 * flops
            peak_note = (f"tf32 dense: cuBLAS TF32 product of the same shape measured in this run = {tf32_tflops:.0f} TFLOP/s "
                         f"(bf16 {peaks['src']} x 1.1/2.25 would be {nominal:.0f}); achieved counts the 3 tf32 passes")
        achieved = exec_flops / (ms_gemm * 1e-3) / 1e12
        enc_bytes = (n * k + k * m) * (2 if args.dtype == "bf16" else 8)
        line.update({
            "roofline": {"bound": "tensor", "kernel": "gecc_gemm_kernel (protected, detection inside)", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                         "frac": achieved / peak, "traffic": NCU_GEMM_TRAFFIC.get((args.dtype, n)) if n == k == m else None, "peak_note": peak_note,
                         "ms_per_launch": ms_gemm,
                         "frac_of_sustained_peak": (achieved / peaks["bf16_sustained"]) if (args.dtype == "bf16" and peaks.get("bf16_sustained")) else None},
            "e2e": {"value": world * flops / (ms_e2e * 1e-3) / 1e12, "unit": "TFLOP/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": ms_e2e, "note": "pinned host buffers; the copies of neighbouring steps overlap the compute on their own streams"},
            "split_ms": split, "split_note": f"device time per call, CUDA-graph replay of {reps} calls over the rotating buffer sets",
            "decode_us_by_scenario": dec_us, "tile_local": tile_local,
            "overhead_pct": {"vs_own_plain_gemm": 100.0 * (ms_step / split["gemm_plain"] - 1.0), "vs_cublas": 100.0 * (ms_step / split["cublas"] - 1.0),
                             "fault_free_vs_own_plain_gemm": 100.0 * (split["step_fault_free"] / split["gemm_plain"] - 1.0),
                             "gemm_only_vs_own_plain_gemm": 100.0 * (ms_gemm / split["gemm_plain"] - 1.0)},
            "encode_hbm": {"achieved_gbs": enc_bytes / (split["encode"] * 1e-3) / 1e9, "peak_gbs": peaks["hbm"],
                           "frac": enc_bytes / (split["encode"] * 1e-3) / 1e9 / peaks["hbm"],
                           "bytes": "both operands read once by gecc_encode_both (+ the fp32 lo planes written)"},
            "syndrome_hbm": {"achieved_gbs": 4.0 * n * m / (split["syndrome_unfused"] * 1e-3) / 1e9, "peak_gbs": peaks["hbm"],
                             "frac": 4.0 * n * m / (split["syndrome_unfused"] * 1e-3) / 1e9 / peaks["hbm"],
                             "bytes": "stored C (fp32) read once by gecc_syndrome_unfused (the detection sums of a C at rest)"},
        })
    else:
        line.update({"roofline": None, "e2e": None})
    line["clocks"] = sampler.stop()

    if rank == 0:
        if world == 1 and not args.no_cpu_baseline and not args.no_split:
            cb = time_oracle(n, k, m, args.dtype, steps=4, warmup=1, rows=ORACLE_ROWS, std_b=args.std_b)
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
