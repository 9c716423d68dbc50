"""Injection campaigns of BASELINE.json's configs at their stated trial counts (too long for the pytest suite):

    python tests/campaign.py --config 1 --trials 10000 --out gpurun_out/campaign_cfg1.md

Every trial runs through the C ABI and through the CPU fp64 oracle on the same operand bits (tests/gpu_harness.py) and is
counted, never asserted, so that one table shows the whole population:

  corrected   oracle and library both CORRECTED, located set = injected set (bit-exact), values within tolerance
  refused     both report the same UNCORRECTABLE* verdict
  sub         both CLEAN although a fault was injected: its footprint is below the thresholds (tolerable noise, Eq. 1)
  guard       the oracle's own answer changes when tau moves by 2x: outside the bit-exact requirement;
              `guard_same` of them still agreed
  mismatch    outside the guard band and different verdict, located set or values: a parity failure

Test infrastructure: imports oracle/.
"""
from __future__ import annotations

import argparse
import collections
import sys
import time
from pathlib import Path

import numpy as np

sys.path.insert(0, str(Path(__file__).resolve().parent))
sys.path.insert(0, str(Path(__file__).resolve().parent.parent))

from oracle import gecc_oracle as O  # noqa: E402
from paper_2508_04355_b200 import inputs as I  # noqa: E402
from gpu_harness import TOL_C, Case, SampledCase, operands_as_the_oracle_leaves_them  # noqa: E402

CLASSES = ("a", "b", "c", "d", "e", "f", "aa", "bb", "ab")


def trial(case: Case, faults, level: int, stats: dict, check_values: bool = True):
    real = case.realise(faults)
    if any(f[3] == 0.0 for f in real):
        stats["null"] += 1  # the fault vanished when the symbol was rounded to the operand dtype
        return
    orc = case.run_oracle(real, level)
    guard = case.in_guard_band(real, level)
    rep, C_gpu, A_gpu, B_gpu = case.run_gpu(faults, level)
    same = rep.verdict == orc.verdict and rep.located() == orc.located()
    err = 0.0
    if same and check_values and orc.verdict in (O.CLEAN, O.CORRECTED):
        err = float(np.abs(C_gpu - orc.C).max() / np.abs(case.Cbar[: case.n, : case.m]).max())
        same = err <= TOL_C[case.dtype]
        if level == 1 and orc.verdict == O.CORRECTED:
            try:    # operands as the oracle's decode leaves them (located faults patched back, sub-threshold ones left in place)
                operands_as_the_oracle_leaves_them(case.dtype, real, orc, A_gpu, B_gpu, case.A_h, case.B_h, "")
            except AssertionError:
                same = False
    if guard:
        stats["guard"] += 1
        stats["guard_same"] += int(same)
        return
    if not same:
        stats["mismatch"] += 1
        stats.setdefault("examples", []).append((faults, rep.verdict, rep.located(), orc.verdict, orc.located(), err))
        return
    stats["max_err"] = max(stats.get("max_err", 0.0), err)
    if orc.verdict == O.CLEAN:
        stats["sub"] += 1
    elif orc.verdict == O.CORRECTED:
        injected = sorted((kd, r, c) for kd, r, c, _ in real)
        stats["corrected" if [tuple(x) for x in orc.located()] == injected else "corrected_other"] += 1
    else:
        stats["refused"] += 1


def new_stats():
    return collections.defaultdict(int)


def run_config(cfg: int, trials: int, dtypes, log):
    """Returns {(dtype, class): stats}.  `trials` is the total of the config (split as its recipe says)."""
    out = {}
    if cfg == 0:   # 64^3, N(0,1), |e| in [1, 100], every class incl. forced sub-cases, both levels
        seeds = range(32)
        per = max(1, trials // (len(CLASSES) * len(seeds)))
        for dt in dtypes:
            for seed in seeds:
                case = Case(64, 64, 64, dt, seed=seed)
                for scen in CLASSES:
                    st = out.setdefault((dt, scen), new_stats())
                    for t in range(per):
                        force = (None, "same_row", "same_col", "same_l")[t % 4]
                        faults = I.draw_faults(64, 64, 64, I.SCENARIOS[scen], seed=100000 * seed + 97 * t + len(scen) + ord(scen[0]), force=force)
                        trial(case, faults, 1, st)
                        trial(case, faults, 0, out.setdefault((dt + "/level0", scen), new_stats()))
                log(f"cfg0 {dt} seed {seed}")
    elif cfg == 1:  # 1024^3 fp32 U(-1,1): 8 matrix seeds, 1 or 2 errors, site classes uniform, |e| log-uniform [1e-2, 1e3]
        per = max(1, trials // 8)
        for seed in range(8):
            case = Case(1024, 1024, 1024, "f32", seed=seed, dist="uniform")
            rng = np.random.default_rng([seed, 2024])
            for t in range(per):
                kinds = tuple(int(x) for x in rng.integers(0, 3, size=1 + int(rng.integers(2))))
                scen = {(0,): "a", (1,): "b", (2,): "c", (0, 2): "d", (1, 2): "e", (2, 2): "f", (0, 0): "aa", (1, 1): "bb", (0, 1): "ab"}[tuple(sorted(kinds))]
                faults = I.draw_faults(1024, 1024, 1024, I.SCENARIOS[scen], seed=1000003 * seed + t, lo=1e-2, hi=1e3, law="log")
                trial(case, faults, 1, out.setdefault(("f32", scen), new_stats()), check_values=(t % 4 == 0))
            log(f"cfg1 seed {seed}")
    elif cfg in (2, 21):  # 4096^3 (21: the paper's own shape 1024 x 4096 x 1024), N(0,1), |e| in [1, 100]
        shape = (4096, 4096, 4096) if cfg == 2 else (1024, 4096, 1024)
        per = max(1, trials // len(CLASSES))
        for dt in dtypes:
            case = Case(*shape, dt, seed=0)
            for scen in CLASSES:
                st = out.setdefault((dt, scen), new_stats())
                for t in range(per):
                    faults = I.draw_faults(*shape, I.SCENARIOS[scen], seed=7000 + 131 * t + len(scen) + ord(scen[0]))
                    trial(case, faults, 1, st, check_values=(t % 8 == 0 or cfg == 21))
                log(f"cfg{cfg} {dt} {scen}")
    elif cfg == 4:  # error-free runs over the size sweep: false positives of the automatic thresholds (reading R4)
        import torch
        from paper_2508_04355_b200 import binding as G
        per = max(1, trials)
        for dt in dtypes:
            tdt = torch.bfloat16 if dt == "bf16" else torch.float32
            for size in (512, 1024, 2048, 4096, 8192, 16384):
                buf = G.Buffers(size, size, size, tdt)
                gen = torch.Generator(device="cuda")
                st = out.setdefault((dt, str(size)), new_stats())
                worst = [0.0] * 4
                for seed in range(per):
                    gen.manual_seed(900000 + seed)
                    A = torch.randn(size, size, device="cuda", generator=gen).to(tdt)
                    B = torch.randn(size, size, device="cuda", generator=gen).to(tdt)
                    G.protected_matmul(A, B, buf, faults=(), level=1)
                    torch.cuda.synchronize()
                    rep = G.read_report(buf.report)
                    st["runs"] += 1
                    st["runs_with_flag"] += int(rep.verdict != O.CLEAN or rep.n_row_flags + rep.n_col_flags > 0)
                    st["flagged_syndromes"] += rep.n_row_flags + rep.n_col_flags
                    worst = [max(w, rep.max_abs_syndrome[q] / rep.tau[q]) for q, w in enumerate(worst)]
                st["worst_over_tau"] = " ".join(f"{w:.3f}" for w in worst)
                del buf
                torch.cuda.empty_cache()
                log(f"cfg4 {dt} {size}: {dict(st)}")
    elif cfg == 5:  # error patterns over the size sweep (BASELINE.json config 4): both errors in C, both in inputs, one of each;
        # |e| log-uniform [1e-3, 1e3].  The oracle runs in error space (gpu_harness.SampledCase): verdict and located set at every
        # size, values on sampled symbols and touched lines.  `trials` = trials per class at sizes <= 4096 (a sixth of it above).
        patterns = (("cc", "f"), ("aa", "aa"), ("bb", "bb"), ("ab", "ab"), ("ac", "d"), ("bc", "e"))
        for dt in dtypes:
            for size in (512, 1024, 2048, 4096, 8192, 16384):
                case = SampledCase(size, size, size, dt, seed=70 + size % 97, samples=20_000)
                per = trials if size <= 4096 else max(2, trials // 6)
                for name, scen in patterns:
                    st = out.setdefault((dt, f"{size} {name}"), new_stats())
                    for t in range(per):
                        faults = I.draw_faults(size, size, size, I.SCENARIOS[scen], seed=555000 + 1009 * t + size + len(name) + ord(name[0]), lo=1e-3, hi=1e3, law="log")
                        real = case.realise(faults)
                        if any(f[3] == 0.0 for f in real):
                            st["null"] += 1
                            continue
                        orc = case.run_oracle(real, 1)
                        guard = case.in_guard_band(real, 1)
                        rep = case.run_gpu(faults, 1)
                        same = rep.verdict == orc.verdict and rep.located() == orc.located()
                        if guard:
                            st["guard"] += 1
                            st["guard_same"] += int(same)
                            continue
                        if same and orc.verdict in (O.CLEAN, O.CORRECTED):
                            try:
                                case.check(faults, 1)   # values on the sampled symbols and the touched lines
                            except AssertionError as e:
                                same = False
                                st.setdefault("examples", []).append((faults, "values", str(e)[:200]))
                        if not same:
                            st["mismatch"] += 1
                            st.setdefault("examples", []).append((faults, rep.verdict, rep.located(), orc.verdict, orc.located()))
                        elif orc.verdict == O.CLEAN:
                            st["sub"] += 1
                        elif orc.verdict == O.CORRECTED:
                            injected = sorted((kd, r, c) for kd, r, c, _ in real)
                            st["corrected" if [tuple(x) for x in orc.located()] == injected else "corrected_other"] += 1
                        else:
                            st["refused"] += 1
                    log(f"cfg5 {dt} {size} {name}: {dict((k2, v) for k2, v in st.items() if k2 != 'examples')}")
                del case
    else:
        raise SystemExit("config must be 0, 1, 2, 21, 4 or 5")
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--trials", type=int, default=900)
    ap.add_argument("--dtypes", default="f32,bf16")
    ap.add_argument("--out", default="")
    args = ap.parse_args()
    t0 = time.time()
    res = run_config(args.config, args.trials, args.dtypes.split(","), lambda s: print(f"[{time.time() - t0:7.1f}s] {s}", flush=True))
    cols = ("corrected", "corrected_other", "refused", "sub", "guard", "guard_same", "null", "mismatch")
    if args.config == 4:
        cols = ("runs", "runs_with_flag", "flagged_syndromes", "worst_over_tau")
    lines = [f"config {args.config}, {args.trials} trials requested, {time.time() - t0:.0f} s", "",
             "| dtype | class | " + " | ".join(cols) + " | max rel err of corrected C |", "|---|---|" + "---|" * (len(cols) + 1)]
    bad = []
    for (dt, scen), st in sorted(res.items()):
        lines.append(f"| {dt} | {scen} | " + " | ".join(str(st.get(c, 0)) for c in cols) + f" | {st.get('max_err', 0.0):.2e} |")
        bad += [(dt, scen) + ex for ex in st.get("examples", [])[:5]]
    lines += ["", "mismatches (first five per class):"] + [repr(b) for b in bad]
    text = "\n".join(lines)
    print(text)
    if args.out:
        Path(args.out).parent.mkdir(parents=True, exist_ok=True)
        Path(args.out).write_text(text + "\n")


if __name__ == "__main__":
    main()
