"""`-m gpu` parity tests: the CUDA path, called through the C ABI, against the CPU fp64 oracle on the same seeded inputs.

Bar (BASELINE.json north_star): verdict and located positions bit-exact; corrected values within max relative error
1e-4 (fp32 / 3xTF32) and 2e-2 (bf16 inputs, fp32 accumulation), measured as reading R15 of DESIGN.md states.
"""
import numpy as np
import pytest
import torch

from oracle import gecc_oracle as O
from paper_2508_04355_b200 import binding as G
from paper_2508_04355_b200 import inputs as I
from gpu_harness import TOL_C, Case, compare
from threshold_spec import stated_global_tolerances

pytestmark = pytest.mark.gpu

TWO = ("d", "e", "f", "aa", "bb", "ab")
FORCES = {"d": (None, "same_row"), "e": (None, "same_col"), "f": (None, "same_row", "same_col"),
          "aa": (None, "same_row", "same_l"), "bb": (None, "same_col", "same_l"), "ab": (None, "same_l")}


def scenario_trials(case, scen, trials, seed0, lo=1.0, hi=100.0, law="uniform"):
    n, k, m = case.n, case.k, case.m
    for fi, force in enumerate(FORCES.get(scen, (None,))):
        for t in range(trials):
            yield I.draw_faults(n, k, m, I.SCENARIOS[scen], seed=seed0 + 7919 * t + 131 * fi, lo=lo, hi=hi, law=law, force=force)


# ---------------------------------------------------------------------------------------------------------------
# encoder and product against their plain definitions
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["bf16", "f32"])
@pytest.mark.parametrize("shape", [(64, 64, 64), (200, 136, 328), (520, 72, 136), (1024, 1024, 1024)])
def test_encoder_and_product_match_the_oracle(dtype, shape):
    n, k, m = shape
    case = Case(n, k, m, dtype, seed=3)
    rep, C, _, _ = case.run_gpu([], level=0)
    buf = case.buf
    # A_P, B_P (fp64 side copy): sums of exact inputs; error bounded by fp32 partial sums of 8 (bf16) / fp64 (fp32)
    scaleA, scaleB = np.abs(case.Abar[n:]).max(), np.abs(case.Bbar[:, m:]).max()
    assert np.abs(buf.A_par64.cpu().numpy() - case.Abar[n:]).max() <= 1e-6 * scaleA
    assert np.abs(buf.B_par64.cpu().numpy() - case.Bbar[:, m:].T).max() <= 1e-6 * scaleB
    # the parity operand handed to the tensor cores: limbs (bf16) / hi + lo (fp32) sum back to the check to ~2^-24
    if dtype == "bf16":
        Ap = buf.A_par.float().cpu().numpy().astype(np.float64)
        Bp = buf.B_par.float().cpu().numpy().astype(np.float64)
    else:
        Ap = buf.A_par.cpu().numpy().astype(np.float64) + buf.A_par_lo.cpu().numpy().astype(np.float64)
        Bp = buf.B_par.cpu().numpy().astype(np.float64) + buf.B_par_lo.cpu().numpy().astype(np.float64)
    for c in range(2):
        assert np.abs(Ap[3 * c:3 * c + 3].sum(0) - case.Abar[n + c]).max() <= 2.0 ** -22 * scaleA
        assert np.abs(Bp[3 * c:3 * c + 3].sum(0) - case.Bbar[:, m + c]).max() <= 2.0 ** -22 * scaleB
    # sum of squares feeding the thresholds
    assert float(buf.sumsq_a) == pytest.approx(float((case.A_h.astype(np.float64) ** 2).sum()), rel=1e-5)
    assert float(buf.sumsq_b) == pytest.approx(float((case.B_h.astype(np.float64) ** 2).sum()), rel=1e-5)
    # data part of the product
    scale = np.abs(case.Cbar[:n, :m]).max()
    assert np.abs(C - case.Cbar[:n, :m]).max() / scale <= TOL_C[dtype]
    # parity blocks of C_bar: P_r = C [1, w], P_c = [1; w] C, P_g
    nl = 3 if dtype == "bf16" else 1
    P_r = buf.P_r.cpu().numpy().astype(np.float64)
    P_c = buf.P_c.cpu().numpy().astype(np.float64)
    P_g = buf.P_g.cpu().numpy().astype(np.float64)
    for c in range(2):
        pr = P_r[:, 3 * c:3 * c + nl].sum(1)
        pc = P_c[3 * c:3 * c + nl].sum(0)
        assert np.abs(pr - case.Cbar[:n, m + c]).max() <= 1e-4 * np.abs(case.Cbar[:n, m + c]).max()
        assert np.abs(pc - case.Cbar[n + c, :m]).max() <= 1e-4 * np.abs(case.Cbar[n + c, :m]).max()
        for c2 in range(2):
            pg = P_g[3 * c:3 * c + nl, 3 * c2:3 * c2 + nl].sum()
            assert abs(pg - case.Cbar[n + c, m + c2]) <= 1e-4 * np.abs(case.Cbar[n:, m:]).max()
    # thresholds: the library reports the formula include/gecc.h states (tests/threshold_spec.py; the oracle has none)
    np.testing.assert_allclose(list(rep.tau), case.tau, rtol=1e-5)
    assert rep.verdict == O.CLEAN and rep.n_row_flags == 0 and rep.n_col_flags == 0
    # fault-free syndromes stay well inside the thresholds (detection-threshold false-positive check)
    for q in range(4):
        assert rep.max_abs_syndrome[q] <= 0.75 * rep.tau[q]


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_plain_product_is_the_same_kernel_without_parity(dtype):
    case = Case(328, 200, 264, dtype, seed=4)
    C = torch.zeros(328, 264, device="cuda")
    lo_a = lo_b = None
    if dtype == "f32":
        case.run_gpu([], level=0)            # fills the low parts
        lo_a, lo_b = case.buf.A_lo, case.buf.B_lo
    G.gecc_matmul_plain(case.A_dev0, lo_a, case.B_dev0, lo_b, C)
    torch.cuda.synchronize()
    ref = case.Cbar[:328, :264]
    assert np.abs(C.cpu().numpy() - ref).max() / np.abs(ref).max() <= TOL_C[dtype]


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_unfused_syndrome_pass_fills_the_same_partials(dtype):
    """gecc_syndrome_unfused over the stored C must lead the decoder to the same answer as the fused epilogue."""
    case = Case(200, 136, 328, dtype, seed=5)
    rep0, C0, _, _ = case.run_gpu([], level=0)
    buf = case.buf
    buf.C[17, 301] += 5.0                                   # corrupt C at rest: the fused sums know nothing of it
    buf.C[150, 2] -= 9.0
    G.gecc_syndrome_unfused(buf.code, 136, buf.C, buf.workspace)
    G.gecc_decode_correct(buf.code, 200, 136, 328, buf.C, buf.P_r, buf.P_c, None, buf.sumsq_a, buf.sumsq_b, 0,
                          None, None, None, None, None, None, buf.report, buf.workspace)
    torch.cuda.synchronize()
    rep = G.read_report(buf.report)
    assert rep.verdict == O.CORRECTED and rep.located() == [(2, 17, 301), (2, 150, 2)]
    assert np.abs(buf.C.cpu().numpy() - C0).max() <= 1e-4 * np.abs(C0).max()


# ---------------------------------------------------------------------------------------------------------------
# config 0 (BASELINE.json): tiny oracle case, every scenario class and forced sub-case, both decoder levels
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("seed", [0, 1])
def test_config0_tiny_all_scenarios(dtype, seed):
    case = Case(64, 64, 64, dtype, seed=seed)
    compare(case, [], 1)
    for scen in ("a", "b", "c") + TWO:
        for faults in scenario_trials(case, scen, trials=12, seed0=1000 * seed + 17 * len(scen) + ord(scen[0])):
            for level in (0, 1):
                compare(case, faults, level)


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("shape", [(200, 136, 328), (136, 264, 72)])
def test_ragged_shapes_all_scenarios(dtype, shape):
    """Sizes that are not multiples of the 128 x 256 x 64 tile: several tiles plus a ragged tail in every dimension."""
    case = Case(*shape, dtype, seed=7)
    for scen in ("a", "b", "c") + TWO:
        for faults in scenario_trials(case, scen, trials=4, seed0=ord(scen[0]) * 31 + len(scen)):
            compare(case, faults, 1)


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_padded_leading_dimensions(dtype):
    """A, B, their lo planes and C as views into wider allocations (ld > cols, include/gecc.h): every kernel must step by
    the leading dimension, not by the width, and must leave the padding alone."""
    n, k, m, pad = 200, 136, 328, 24
    case = Case(n, k, m, dtype, seed=12)
    buf = case.buf

    def widen(t, fill):
        big = torch.full((t.shape[0], t.shape[1] + pad), fill, dtype=t.dtype, device=t.device)
        big[:, : t.shape[1]] = t
        return big, big[:, : t.shape[1]]

    bigC, buf.C = widen(buf.C, 7.0)
    if buf.A_lo is not None:
        _, buf.A_lo = widen(buf.A_lo, 0.0)
        _, buf.B_lo = widen(buf.B_lo, 0.0)
    for faults in ([], [(0, 17, 101, 9.0)], [(1, 64, 300, -6.0), (2, 199, 327, 11.0)], [(2, 5, 9, 3.0), (2, 130, 260, -4.0)]):
        bigA, A = widen(case.A_dev0, 3.0)   # the padding holds junk that must never be read as data
        bigB, B = widen(case.B_dev0, -5.0)
        real = case.realise(faults)
        G.protected_matmul(A, B, buf, faults=faults, level=1)
        torch.cuda.synchronize()
        rep = G.read_report(buf.report)
        orc = case.run_oracle(real, 1)
        assert rep.verdict == orc.verdict and rep.located() == orc.located(), (faults, rep.verdict, rep.located(), orc.located())
        C = buf.C.cpu().numpy().astype(np.float64)
        assert np.abs(C - orc.C).max() <= TOL_C[dtype] * np.abs(orc.C).max()
        assert torch.equal(A.float().cpu(), torch.from_numpy(case.A_h)) and torch.equal(B.float().cpu(), torch.from_numpy(case.B_h))
        assert bool((bigA[:, k:] == 3.0).all()) and bool((bigB[:, m:] == -5.0).all()) and bool((bigC[:, m:] == 7.0).all())


def test_edge_positions():
    """First / last rows and columns, tile borders, and both parity-adjacent corners."""
    case = Case(264, 72, 520, "bf16", seed=8)
    n, k, m = 264, 72, 520
    for (i, j) in [(0, 0), (n - 1, m - 1), (127, 255), (128, 256), (263, 0), (0, 519), (31, 32)]:
        compare(case, [(2, i, j, 13.0)], 1)
    for (i, l) in [(0, 0), (n - 1, k - 1), (128, 64), (127, 63)]:
        compare(case, [(0, i, l, -21.0)], 1)
    for (l, j) in [(0, 0), (k - 1, m - 1), (64, 256), (63, 255)]:
        compare(case, [(1, l, j, 17.0)], 1)
    compare(case, [(2, 5, 9, 3.0), (2, 5, 10, 4.0)], 1)          # adjacent columns, same row
    compare(case, [(2, 5, 9, 3.0), (2, 6, 10, 3.0)], 1)          # adjacent diagonal, equal magnitudes


def test_uncorrectable_patterns_are_refused():
    """min(s,t) >= 3: three point errors on distinct rows and columns; the e_1 pattern of PAPER.md:170."""
    case = Case(64, 64, 64, "f32", seed=9)
    rep, orc = compare(case, [(2, 1, 2, 5.0), (2, 10, 20, 6.0), (2, 30, 40, 7.0)], 0)
    assert rep.verdict == O.UNCORRECTABLE
    e1 = [(2, 0, 0, 1.0), (2, 0, 1, -2.0), (2, 0, 2, 1.0), (2, 1, 0, -1.0), (2, 1, 1, 2.0), (2, 1, 2, -1.0)]
    rep, orc = compare(case, e1, 0)
    assert rep.verdict == O.UNCORRECTABLE


# ---------------------------------------------------------------------------------------------------------------
# config 1 / 2 (BASELINE.json): 1024^3 fp32 U(-1,1), log-uniform magnitudes; 4096^3 both dtypes (the bench workload)
# ---------------------------------------------------------------------------------------------------------------
def _rate_run(case, scens, trials, lo, hi, law, seed0):
    """Runs trials; trials whose oracle answer is threshold-stable must match bit-exactly; returns counts."""
    stats = {"match": 0, "guard": 0}
    for scen in scens:
        for t in range(trials):
            faults = I.draw_faults(case.n, case.k, case.m, I.SCENARIOS[scen], seed=seed0 + 101 * t + ord(scen[0]) + len(scen), lo=lo, hi=hi, law=law)
            real = case.realise(faults)
            if any(f[3] == 0.0 for f in real) or case.in_guard_band(real, 1):
                stats["guard"] += 1
                continue
            compare(case, faults, 1)
            stats["match"] += 1
    return stats


def test_config1_1024_fp32_uniform_log_magnitudes():
    case = Case(1024, 1024, 1024, "f32", seed=0, dist="uniform")
    stats = _rate_run(case, ("a", "b", "c") + TWO, trials=10, lo=1e-2, hi=1e3, law="log", seed0=5000)
    assert stats["match"] >= 60, stats


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_config2_4096_bench_workload(dtype):
    """The configuration bench.py times (4096^3), full element-wise comparison against the fp64 product."""
    case = Case(4096, 4096, 4096, dtype, seed=0)
    compare(case, [], 1)
    stats = _rate_run(case, ("a", "b", "c", "d", "e", "f", "aa", "bb", "ab"), trials=3, lo=1.0, hi=100.0, law="uniform", seed0=9000)
    assert stats["match"] >= 20, stats


def test_config3_transformer_shapes_bf16():
    """Llama-like projection shape (BASELINE.json config 4, forward product): X 8192 x 4096 N(0,1), W 4096 x 4096
    N(0, 0.02); two faults per product, classes d / e / f."""
    case = Case(8192, 4096, 4096, "bf16", seed=1, std_b=0.02)
    stats = _rate_run(case, ("d", "e", "f"), trials=2, lo=1.0, hi=100.0, law="uniform", seed0=12000)
    assert stats["match"] >= 4, stats


# ---------------------------------------------------------------------------------------------------------------
# C ABI error behaviour
# ---------------------------------------------------------------------------------------------------------------
def test_error_codes():
    lib = G.load()
    assert lib.gecc_workspace_bytes(7, 64, 64, 64) == 0
    buf = G.Buffers(64, 64, 64, torch.bfloat16)
    A = torch.zeros(64, 64, dtype=torch.bfloat16, device="cuda")
    with pytest.raises(RuntimeError, match="GECC_EWORKSPACE"):
        G.gecc_matmul_protected(A, buf.A_par, None, None, A, buf.B_par, None, None, buf.C, buf.P_r, buf.P_c, buf.P_g, None, 0,
                                buf.workspace[:128])
    with pytest.raises(RuntimeError, match="GECC_EINVAL"):
        G.gecc_matmul_plain(A[:, :60], None, A, None, buf.C)          # k = 60 is not a multiple of 8
    with pytest.raises(RuntimeError, match="GECC_EINVAL"):
        G.gecc_encode(G.GECC_LEFT, A, None, None, None, buf.A_par64, buf.sumsq_a, buf.workspace)


# ---------------------------------------------------------------------------------------------------------------
# the paper's own workload (Table I): M(n = 1024, k = 4096, m = 1024), scenarios a-f
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_paper_shape_table1_scenarios(dtype):
    case = Case(1024, 4096, 1024, dtype, seed=2)
    stats = _rate_run(case, ("a", "b", "c", "d", "e", "f"), trials=4, lo=1.0, hi=100.0, law="uniform", seed0=31000)
    assert stats["match"] >= 20, stats      # Table I: 100 % for every scenario; trials in the guard band are not compared


# ---------------------------------------------------------------------------------------------------------------
# config 4 (BASELINE.json): detection-threshold false positives on fault-free runs over the size sweep
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["bf16", "f32"])
@pytest.mark.parametrize("size", [512, 1024, 2048, 4096])
def test_fault_free_runs_raise_no_flag(dtype, size):
    tdt = torch.bfloat16 if dtype == "bf16" else torch.float32
    buf = G.Buffers(size, size, size, tdt)
    gen = torch.Generator(device="cuda")
    worst = 0.0
    for seed in range(6):
        gen.manual_seed(4000 + seed)
        A = torch.randn(size, size, device="cuda", generator=gen).to(tdt)
        B = torch.randn(size, size, device="cuda", generator=gen).to(tdt)
        G.protected_matmul(A, B, buf, faults=(), level=1)
        torch.cuda.synchronize()
        rep = G.read_report(buf.report)
        assert rep.verdict == O.CLEAN and rep.n_row_flags == 0 and rep.n_col_flags == 0, (size, seed, rep.n_row_flags, rep.n_col_flags)
        worst = max(worst, max(rep.max_abs_syndrome[q] / rep.tau[q] for q in range(4)))
    # the largest fault-free syndrome stays inside its threshold (kappa = 16 sigma; heavy tails: 0.78 tau was measured once for
    # a weighted column syndrome of 3xTF32 at 4096, everything else stays below 0.56 tau)
    assert worst <= 0.9, worst


# ---------------------------------------------------------------------------------------------------------------
# transposed operands: the backward products of a linear layer, dX = dY W^T (B stored transposed) and dW = X^T dY
# (A stored transposed) -- BASELINE.json config 3.  Both decoder levels.
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["bf16", "f32"])
@pytest.mark.parametrize("trans", [(1, 0), (0, 1), (1, 1)])
@pytest.mark.parametrize("shape", [(264, 136, 328), (512, 256, 384)])
def test_transposed_operands_small(dtype, trans, shape):
    case = Case(*shape, dtype, seed=12, trans_a=trans[0], trans_b=trans[1])
    rep, C, _, _ = case.run_gpu([], level=0)
    n, k, m = shape
    ref = case.Cbar[:n, :m]
    assert np.abs(C - ref).max() / np.abs(ref).max() <= TOL_C[dtype]
    assert rep.verdict == O.CLEAN
    # the encoder's checks are those of the operand, whatever the storage
    assert np.abs(case.buf.A_par64.cpu().numpy() - case.Abar[n:]).max() <= 1e-6 * np.abs(case.Abar[n:]).max()
    assert np.abs(case.buf.B_par64.cpu().numpy() - case.Bbar[:, m:].T).max() <= 1e-6 * np.abs(case.Bbar[:, m:]).max()
    for scen in ("a", "b", "c", "d", "e", "f"):
        for faults in scenario_trials(case, scen, trials=2, seed0=700 + ord(scen)):
            compare(case, faults, 0)
    for scen in ("a", "b", "c") + TWO:
        for faults in scenario_trials(case, scen, trials=2, seed0=900 + ord(scen[0]) + len(scen)):
            compare(case, faults, 1)

@pytest.mark.parametrize("trans", [(0, 1), (1, 0)])
def test_same_direction_encoders_are_ordered(trans):
    """trans_a != trans_b: both encoders reduce in the same direction and then share scratch and arrival counters in the
    workspace (include/gecc.h), so they must not overlap on two streams.  Repeated fault-free products: every one CLEAN,
    checks and sums of squares equal to the oracle's every time (overlapping launches fold strips from mixed arrivals)."""
    n, k, m = 1024, 2048, 2304
    case = Case(n, k, m, "bf16", seed=31, trans_a=trans[0], trans_b=trans[1])
    scaleA, scaleB = np.abs(case.Abar[n:]).max(), np.abs(case.Bbar[:, m:]).max()
    ssa, ssb = float((case.A_h.astype(np.float64) ** 2).sum()), float((case.B_h.astype(np.float64) ** 2).sum())
    for _ in range(40):
        rep, _, _, _ = case.run_gpu([], level=1)
        assert rep.verdict == O.CLEAN
        assert np.abs(case.buf.A_par64.cpu().numpy() - case.Abar[n:]).max() <= 1e-6 * scaleA
        assert np.abs(case.buf.B_par64.cpu().numpy() - case.Bbar[:, m:].T).max() <= 1e-6 * scaleB
        assert float(case.buf.sumsq_a) == pytest.approx(ssa, rel=1e-5) and float(case.buf.sumsq_b) == pytest.approx(ssb, rel=1e-5)


def test_config3_backward_products_bf16():
    """Llama-like projection (BASELINE.json config 3), backward products at a quarter of the token count to bound the oracle's
    time: dX = dY W^T (n = 2048 tokens, k = 4096, m = 4096, B = W^T stored as W) and dW = X^T dY (n = 4096, k = 2048, m = 4096,
    A = X^T stored as X); two faults per product, classes d / e / f."""
    dx = Case(2048, 4096, 4096, "bf16", seed=21, std_b=0.02, trans_b=1)
    stats = _rate_run0(dx, ("d", "e", "f"), trials=2, seed0=41000)
    assert stats["match"] >= 4, stats
    stats = _rate_run(dx, ("d", "e", "f", "ab"), trials=2, lo=1.0, hi=100.0, law="uniform", seed0=43000)
    assert stats["match"] >= 6, stats
    dw = Case(4096, 2048, 4096, "bf16", seed=22, trans_a=1)
    stats = _rate_run0(dw, ("d", "e", "f"), trials=2, seed0=42000)
    assert stats["match"] >= 4, stats
    stats = _rate_run(dw, ("d", "e", "f", "ab"), trials=2, lo=1.0, hi=100.0, law="uniform", seed0=44000)
    assert stats["match"] >= 6, stats


def test_config3_up_projection_full_size_bf16():
    """The wide weight of config 3 at its full size: X 8192 x 4096 N(0,1) times W 4096 x 14336 N(0, 0.02), forward, two faults
    per product (one input + one output, both outputs), level X."""
    case = Case(8192, 4096, 14336, "bf16", seed=3, std_b=0.02)
    compare(case, [], 1)
    stats = _rate_run(case, ("d", "e", "f"), trials=1, lo=1.0, hi=100.0, law="uniform", seed0=13000)
    assert stats["match"] >= 2, stats


def _rate_run0(case, scens, trials, seed0):
    stats = {"match": 0, "guard": 0}
    for scen in scens:
        for t in range(trials):
            faults = I.draw_faults(case.n, case.k, case.m, I.SCENARIOS[scen], seed=seed0 + 101 * t + ord(scen[0]) + len(scen))
            real = case.realise(faults)
            if any(f[3] == 0.0 for f in real) or case.in_guard_band(real, 0):
                stats["guard"] += 1
                continue
            compare(case, faults, 0)
            stats["match"] += 1
    return stats


# ---------------------------------------------------------------------------------------------------------------
# single-checksum mode, faults in parity symbols of C_bar (global parity, Eq. 4), recompute fallback
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_single_checksum_mode(dtype):
    """Only P_n1 / P_m1 consulted (ref [8]; Table I's "Checksum" columns): scenario c is corrected,
    everything else is detected and refused with C untouched -- the same answers as the oracle's single-checksum decoder."""
    case = Case(200, 136, 328, dtype, seed=41)
    for scen in ("c", "a", "b", "d", "e", "f"):
        for faults in scenario_trials(case, scen, trials=3, seed0=2100 + ord(scen)):
            real = case.realise(faults)
            rep, C, _, _ = case.run_gpu(faults, level=G.SINGLE_CHECKSUM)
            Cb = O.fault_effects(case.Cbar, case.Abar, case.Bbar, real)
            orc = O.decode_single_checksum(Cb, case.tau)
            assert rep.verdict == orc.verdict and rep.located() == orc.located(), (faults, rep.verdict, rep.located(), orc.verdict, orc.located())
            assert (rep.verdict == O.CORRECTED) == (scen == "c")
            assert np.abs(C - orc.C).max() <= TOL_C[dtype] * np.abs(case.Cbar[:200, :328]).max()
    rep, _, _, _ = case.run_gpu([], level=G.SINGLE_CHECKSUM)
    assert rep.verdict == O.CLEAN


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_parity_symbol_faults_are_classified_by_the_global_parity(dtype):
    """A fault in a local parity symbol of C_bar (after the product, before the decoder): without P_g the flagged line holds
    nothing locatable (UNCORRECTABLE); with P_g (Eq. 4) the symbol is named and repaired, C untouched."""
    n, k, m = 264, 136, 328
    case = Case(n, k, m, dtype, seed=42)
    buf = case.buf
    tg_rows, tg_cols = stated_global_tolerances(case.tau, n, m)
    A, B = case.A_dev0.clone(), case.B_dev0.clone()

    def product():  # without thresholds: the sums are left for the decoder, which then sees the corrupted parity symbol
        buf.lo_planes_for(A, B)
        G.gecc_encode(G.GECC_LEFT, A, buf.A_par, buf.A_par_lo, buf.A_lo, buf.A_par64, buf.sumsq_a, buf.workspace)
        G.gecc_encode(G.GECC_RIGHT, B, buf.B_par, buf.B_par_lo, buf.B_lo, buf.B_par64, buf.sumsq_b, buf.workspace)
        G.gecc_matmul_protected(A, buf.A_par, buf.A_lo, buf.A_par_lo, B, buf.B_par, buf.B_lo, buf.B_par_lo, buf.C, buf.P_r, buf.P_c, buf.P_g, None, 0,
                                buf.workspace)

    def decode(with_pg):
        G.gecc_decode_correct(buf.code, n, k, m, buf.C, buf.P_r, buf.P_c, None, buf.sumsq_a, buf.sumsq_b, 1, A, buf.A_lo, buf.A_par64, B, buf.B_lo,
                              buf.B_par64, buf.report, buf.workspace, P_g=buf.P_g if with_pg else None)
        torch.cuda.synchronize()
        return G.read_report(buf.report)

    product()
    C0 = buf.C.clone()
    for side, line, c in (("r", 17, 0), ("r", 263, 1), ("r", 0, 1), ("c", 5, 0), ("c", 327, 1), ("c", 130, 0)):
        product()
        tol = (tg_rows if side == "r" else tg_cols)[0][c]
        sym = buf.P_r[line, 3 * c:3 * c + 1] if side == "r" else buf.P_c[3 * c:3 * c + 1, line]
        before = float(sym)
        sym += 40.0 * tol
        delta = float(sym) - before                                   # the realised fault (fp32 storage)
        limbs_before = (buf.P_r[line, 3 * c:3 * c + 3] if side == "r" else buf.P_c[3 * c:3 * c + 3, line]).double().sum().item() - delta
        rep = decode(False)
        assert rep.verdict == O.UNCORRECTABLE
        product(); sym += 40.0 * tol
        rep = decode(True)
        Cb = case.Cbar.copy()
        if side == "r":
            Cb[line, m + c] += delta
        else:
            Cb[n + c, line] += delta
        orc = O.decode_level_p(Cb, case.tau, {"rows": tg_rows, "cols": tg_cols})
        assert orc.verdict == O.CORRECTED and orc.located() == [(O.KIND_PR, line, c) if side == "r" else (O.KIND_PC, c, line)]
        assert rep.verdict == orc.verdict and rep.located() == orc.located(), (side, line, c, rep.verdict, rep.located())
        assert rep.magnitudes()[0] == pytest.approx(delta, rel=1e-3, abs=4 * tol)
        assert torch.equal(buf.C, C0)                                  # C untouched
        limbs_after = (buf.P_r[line, 3 * c:3 * c + 3] if side == "r" else buf.P_c[3 * c:3 * c + 3, line]).double().sum().item()
        assert abs(limbs_after - limbs_before) <= 4 * tol + 1e-3 * abs(delta)     # the symbol is what was corrected


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_recompute_fallback(dtype):
    """PAPER.md:219 "needs to be recalculated": patterns the code cannot correct (three errors on distinct rows and columns,
    a non-finite symbol) are recomputed block-wise and re-checked -> CORRECTED_BY_RECOMPUTE, C equal to the fault-free
    product, as the oracle's fallback.  Operands corrupted beyond repair stay refused."""
    n, k, m = 520, 136, 584
    case = Case(n, k, m, dtype, seed=43)
    scale = np.abs(case.Cbar[:n, :m]).max()
    for faults in ([(2, 1, 2, 5.0), (2, 300, 20, 6.0), (2, 519, 583, 7.0)], [(2, 40, 500, float("nan"))],
                   [(2, i, i + 7, 3.0 + i) for i in range(0, 500, 100)]):
        A, B = case.A_dev0.clone(), case.B_dev0.clone()
        blocks = G.protected_matmul(A, B, case.buf, faults=faults, level=1, fallback=True)
        torch.cuda.synchronize()
        rep = G.read_report(case.buf.report)
        Cb = O.inject_output_faults(case.Cbar, faults)
        orc = O.recompute_fallback(Cb, case.Abar, case.Bbar, case.tau)
        assert orc.verdict == O.CORRECTED_BY_RECOMPUTE
        assert rep.verdict == orc.verdict and blocks > 0, (faults, rep.verdict, blocks)
        assert np.abs(case.buf.C.cpu().numpy() - orc.C).max() <= TOL_C[dtype] * scale
    # a correctable pattern: the fallback has nothing to do
    A, B = case.A_dev0.clone(), case.B_dev0.clone()
    assert G.protected_matmul(A, B, case.buf, faults=[(2, 7, 9, 4.0)], level=1, fallback=True) == 0
    assert G.read_report(case.buf.report).verdict == O.CORRECTED
    # two faults in one column of A: UNCORRECTABLE_INPUT stays (recomputing from a corrupted operand reproduces the error)
    A, B = case.A_dev0.clone(), case.B_dev0.clone()
    assert G.protected_matmul(A, B, case.buf, faults=[(0, 10, 33, 9.0), (0, 400, 33, -5.0)], level=1, fallback=True) == 0
    assert G.read_report(case.buf.report).verdict == O.UNCORRECTABLE_INPUT
