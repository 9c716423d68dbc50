"""Tile-local grid (include/gecc.h gecc_tl_*): the CUDA path against the oracle's encode_panels /
decode_panels (oracle/gecc_oracle.py), through the C ABI, on the same operand bits.

One code per 128 x 128 block of C: positions and verdicts bit-exact, corrected values within the north-star tolerance and
the regression bound, parity products element by element against fp64.
"""
import numpy as np
import pytest
import torch

from oracle import gecc_oracle as O
from paper_2508_04355_b200 import binding as G
from paper_2508_04355_b200 import inputs as I

from gpu_harness import REGRESSION_TOL, TORCH_DT
from threshold_spec import stated_thresholds

pytestmark = pytest.mark.gpu
P = Q = G.TL_PANEL


class TlCase:
    def __init__(self, n, k, m, dtype, seed):
        self.n, self.k, self.m, self.dtype = n, k, m, dtype
        self.A_h, self.B_h = I.make_operands(n, k, m, seed, dtype=dtype)
        self.A64, self.B64 = self.A_h.astype(np.float64), self.B_h.astype(np.float64)
        self.A_dev0 = torch.from_numpy(self.A_h).cuda().to(TORCH_DT[dtype])
        self.B_dev0 = torch.from_numpy(self.B_h).cuda().to(TORCH_DT[dtype])
        self.buf = G.TlBuffers(n, k, m, TORCH_DT[dtype])
        self.par = O.encode_panels(self.A64, self.B64, P, Q)          # from the clean operands (reading R1)
        self.C = self.A64 @ self.B64
        self.ssa, self.ssb = float((self.A64 ** 2).sum()), float((self.B64 ** 2).sum())

    def tau_of_block(self, rows, cols):
        """include/gecc.h: the stated formula with n -> rows, m -> cols, sigma_a / sigma_b the RMS of the whole operands."""
        return stated_thresholds(self.dtype, rows, self.k, cols, self.ssa * rows / self.n, self.ssb * cols / self.m)

    def realise(self, faults):
        out = []
        for kind, r, c, e in faults:
            if kind == I.KIND_C:
                out.append((kind, r, c, float(np.float32(e))))
            else:
                X = self.A_h if kind == I.KIND_A else self.B_h
                out.append((kind, r, c, float(np.float64(I.realise_input_fault(X, r, c, e, self.dtype)) - np.float64(X[r, c]))))
        return out

    def run_gpu(self, faults):
        A, B = self.A_dev0.clone(), self.B_dev0.clone()
        G.tl_protected_matmul(A, B, self.buf, faults=faults)
        torch.cuda.synchronize()
        return G.read_tl_report(self.buf.report), self.buf.C.cpu().numpy().astype(np.float64)

    def run_oracle(self, real, scale=1.0):
        Af, Bf = self.A64.copy(), self.B64.copy()
        for kind, r, c, e in real:
            if kind == I.KIND_A:
                Af[r, c] += e
            elif kind == I.KIND_B:
                Bf[r, c] += e
        Cf = Af @ Bf
        for kind, r, c, e in real:
            if kind == I.KIND_C:
                Cf[r, c] += e
        return O.decode_panels(Cf, Af, Bf, P, Q, lambda rows, cols: tuple(scale * t for t in self.tau_of_block(rows, cols)), parity=self.par)

    def in_guard_band(self, real):
        lo, mid, hi = self.run_oracle(real, 0.5), self.run_oracle(real), self.run_oracle(real, 2.0)
        return not (lo.verdict == mid.verdict == hi.verdict and lo.located() == mid.located() == hi.located())

    def compare(self, faults, allow_guard=False):
        """allow_guard: random draws may land a footprint within [tau / 2, 2 tau] of a block (guard band): such a
        trial is outside the bit-exact requirement and returns None; hand-picked cases must not."""
        real = self.realise(faults)
        rep, C_gpu = self.run_gpu(faults)
        orc = self.run_oracle(real)
        ctx = f"faults={faults} gpu=({rep.verdict},{rep.located()}) oracle=({orc.verdict},{orc.located()})"
        if self.in_guard_band(real):
            assert allow_guard, ctx + " (test case sits in the guard band: choose other magnitudes)"
            return None
        assert rep.verdict == orc.verdict, ctx
        assert rep.n_found == len(orc.found), ctx
        if len(orc.found) <= G.TL_MAX_FOUND:
            assert rep.located() == orc.located(), ctx                 # bit-exact positions, global coordinates
        assert (rep.n_row_flags, rep.n_col_flags) == (orc.n_row_flags, orc.n_col_flags), ctx
        scale = np.abs(self.C).max()
        err = np.abs(C_gpu - orc.C).max() / scale                      # reading R15; blocks the oracle refused stay as computed on both sides
        assert err <= REGRESSION_TOL[self.dtype], f"{ctx} corrected C off by {err:.3e}"
        if len(orc.found) <= G.TL_MAX_FOUND:
            tau = self.tau_of_block(P, Q)
            for (kd, r, c, mag_o), mag_g in zip(orc.found, rep.magnitudes()):
                if kd == O.KIND_C:
                    assert abs(mag_g - mag_o) <= 1e-3 * abs(mag_o) + 4 * max(tau[0], tau[2]), f"{ctx} magnitude {mag_g} vs {mag_o}"
        return rep, orc


SHAPES = [(256, 256, 256), (264, 136, 328), (512, 1024, 384)]


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
@pytest.mark.parametrize("shape", SHAPES)
def test_panel_encoder_and_parity_products_match_the_oracle(shape, dtype):
    n, k, m = shape
    case = TlCase(n, k, m, dtype, seed=11)
    rep, C_gpu = case.run_gpu([])
    buf = case.buf
    AP, BP = case.par
    nl = 3 if dtype == "bf16" else 1
    A_PL = buf.A_PL.double().cpu().numpy() + (buf.A_PL_lo.double().cpu().numpy() if dtype == "f32" else 0.0)
    B_PL = buf.B_PL.double().cpu().numpy() + (buf.B_PL_lo.double().cpu().numpy() if dtype == "f32" else 0.0)
    for p, ap in enumerate(AP):                                         # PAPER.md:71-83 per panel: limbs add up to the checks
        for c in range(2):
            got = A_PL[8 * p + 3 * c: 8 * p + 3 * c + nl].sum(0)
            assert np.abs(got - ap[c]).max() <= 2.0 ** -21 * np.abs(ap[c]).max(), (p, c)
    for q, bp in enumerate(BP):                                         # PAPER.md:89-101 per panel
        for c in range(2):
            got = B_PL[8 * q + 3 * c: 8 * q + 3 * c + nl].sum(0)
            assert np.abs(got - bp[:, c]).max() <= 2.0 ** -20 * np.abs(bp[:, c]).max(), (q, c)
    assert abs(buf.sumsq_a.item() - case.ssa) <= 1e-5 * case.ssa and abs(buf.sumsq_b.item() - case.ssb) <= 1e-5 * case.ssb
    # product and parity products (PAPER.md:115-127 per block) against fp64
    assert np.abs(C_gpu - case.C).max() <= 1e-4 * np.abs(case.C).max()
    P_cL, P_rL = buf.P_cL.double().cpu().numpy(), buf.P_rL.double().cpu().numpy()
    for p, ap in enumerate(AP):
        want = ap @ case.B64                                            # 2 x m
        for c in range(2):
            got = P_cL[8 * p + 3 * c: 8 * p + 3 * c + nl].sum(0)
            assert np.abs(got - want[c]).max() <= 1e-4 * np.abs(want[c]).max(), (p, c)
    for q, bp in enumerate(BP):
        want = case.A64 @ bp                                            # n x 2
        for c in range(2):
            got = P_rL[:, 8 * q + 3 * c: 8 * q + 3 * c + nl].sum(1)
            assert np.abs(got - want[:, c]).max() <= 1e-4 * np.abs(want[:, c]).max(), (q, c)
    # fault-free: no flag anywhere, syndromes well inside the thresholds of a full block
    assert rep.verdict == G.CLEAN and rep.n_found == 0 and rep.n_row_flags == 0 and rep.n_col_flags == 0
    tau = case.tau_of_block(min(P, n), min(Q, m))
    assert all(abs(rep.tau[q] - tau[q]) <= 1e-5 * tau[q] for q in range(4))           # the stated formula (sumsq is accumulated in fp32 pieces)
    assert all(rep.max_abs_syndrome[q] <= 0.9 * tau[q] for q in range(4)), (list(rep.max_abs_syndrome), tau)


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_errors_in_many_blocks_are_corrected_block_by_block(dtype):
    """Six errors on distinct rows and columns defeat the global code (min(s, t) >= 3); they fall into different
    blocks, two at most per block, and every block corrects its own."""
    case = TlCase(512, 256, 384, dtype, seed=3)
    faults = [(I.KIND_C, 5, 17, 9.0), (I.KIND_C, 100, 90, -6.0),          # block (0, 0): two errors on a diagonal
              (I.KIND_C, 130, 140, 12.0), (I.KIND_C, 131, 300, -5.0),     # blocks (1, 1), (1, 2)
              (I.KIND_C, 300, 10, 7.5), (I.KIND_C, 300, 60, -8.5),        # block (2, 0): two errors in one row
              (I.KIND_C, 400, 200, 4.0), (I.KIND_C, 500, 200, -11.0),     # block (3, 1): two errors in one column
              (I.KIND_C, 511, 383, 6.0)]                                  # the last symbol of the last block
    rep, orc = case.compare(faults)
    assert orc.verdict == O.CORRECTED and orc.located() == sorted((f[0], f[1], f[2]) for f in faults)


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_ragged_blocks_and_theorem2_patterns(dtype):
    """n, m not multiples of 128 (short last panels with their own weights and thresholds); E(1, t) and E(2, t) point patterns
    inside one block (Theorem 2; reading R21); a block with errors on three rows and three columns is refused
     while the other blocks are still served."""
    case = TlCase(264, 136, 328, dtype, seed=7)
    case.compare([(I.KIND_C, 260, 300, 9.0), (I.KIND_C, 263, 327, -7.0)])                       # ragged corner block (8 rows x 72 columns)
    case.compare([(I.KIND_C, 20, c, 5.0 + c % 3) for c in (3, 40, 77)])                           # E(1, 3): listed one by one
    case.compare([(I.KIND_C, 20, c, 5.0 + c % 3) for c in (3, 40, 77, 90, 101, 120)])             # E(1, 6): reported as a whole row of the block
    case.compare([(I.KIND_C, 150 + (c % 2), c, 6.0) for c in (130, 141, 152, 163)])               # E(2, 4)
    rep, orc = case.compare([(I.KIND_C, 1, 1, 5.0), (I.KIND_C, 2, 2, 6.0), (I.KIND_C, 3, 3, 7.0), (I.KIND_C, 200, 200, 8.0)])
    assert orc.verdict == O.UNCORRECTABLE and orc.located() == [(O.KIND_C, 200, 200)]


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_input_faults_show_as_whole_lines_in_every_block_they_touch(dtype):
    """A fault in a symbol of A after encoding (E1) corrupts row i of C in every column panel; each block
    locates the row by the weighted ratio with local weights (R7) and restores its piece of it (R6).  Likewise B (E2)."""
    case = TlCase(384, 256, 512, dtype, seed=5)
    rep, orc = case.compare([(I.KIND_A, 200, 31, 40.0)])
    assert orc.located() == [(O.KIND_ROW, 200, -1)] * 4
    rep, orc = case.compare([(I.KIND_B, 100, 300, -35.0)])
    assert orc.located() == [(O.KIND_COL, -1, 300)] * 3
    case.compare([(I.KIND_A, 10, 5, 30.0), (I.KIND_C, 300, 400, 9.0)])                            # scenario d, different blocks


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_random_error_patterns_against_the_oracle(dtype):
    """Seeded random draws: 1 to 6 errors in C, positions uniform (so that blocks with 0, 1, 2 and sometimes 3 errors occur),
    |e| log-uniform in [0.1, 1000], and in every third draw one input fault on top (then |e| >= 2: a point error in a block
    that also holds a whole-line fault is resolved by the 2 x 2 solve, whose weighted right-hand side carries fp32 noise divided by
    the weight difference -- DESIGN.md R26 states the limit 2 tau_2 / |w2 - w1| below which the library refuses the block).
    Verdict, located set and flag counts bit-exact, values within the regression bound; draws in the guard band are
    counted, not compared."""
    case = TlCase(384, 512, 384, dtype, seed=17)
    rng = np.random.default_rng(2024)
    guard = compared = 0
    for trial in range(40):
        faults = []
        lo = 2.0 if trial % 3 == 0 else 0.1
        for _ in range(int(rng.integers(1, 7))):
            mag = float(np.exp(rng.uniform(np.log(lo), np.log(1000.0)))) * (1 if rng.integers(2) else -1)
            faults.append((I.KIND_C, int(rng.integers(0, case.n)), int(rng.integers(0, case.m)), mag))
        if trial % 3 == 0:
            kind = I.KIND_A if rng.integers(2) else I.KIND_B
            pos = (int(rng.integers(0, case.n)), int(rng.integers(0, case.k))) if kind == I.KIND_A else (int(rng.integers(0, case.k)), int(rng.integers(0, case.m)))
            faults.append((kind, pos[0], pos[1], float(rng.uniform(20.0, 60.0))))
        if len({(f[0], f[1], f[2]) for f in faults}) < len(faults):
            continue
        out = case.compare(faults, allow_guard=True)
        guard += out is None
        compared += out is not None
    assert compared >= 25, (compared, guard)


def test_caller_thresholds_long_found_list_and_argument_checks():
    """tau passed by the caller (HOST, used for every block) gives the automatic result when it equals the stated thresholds of
    a full block; an input fault crossing more blocks than the report lists (70 > GECC_TL_MAX_FOUND) is still corrected
    everywhere and counted in full; unsupported modes and bad arguments are refused before anything is launched."""
    case = TlCase(256, 128, 128 * 70, "bf16", seed=9)
    faults = [(I.KIND_A, 130, 40, 30.0)]
    real = case.realise(faults)
    A, B = case.A_dev0.clone(), case.B_dev0.clone()
    G.tl_protected_matmul(A, B, case.buf, faults=faults, tau=case.tau_of_block(P, Q))
    torch.cuda.synchronize()
    rep = G.read_tl_report(case.buf.report)
    orc = case.run_oracle(real)
    assert orc.verdict == O.CORRECTED and len(orc.found) == 70
    assert rep.verdict == G.CORRECTED and rep.n_found == 70
    assert rep.located() == [(G.KIND_ROW, 130, -1)] * G.TL_MAX_FOUND
    assert (rep.n_row_flags, rep.n_col_flags) == (orc.n_row_flags, orc.n_col_flags)
    assert np.abs(case.buf.C.cpu().numpy() - orc.C).max() <= REGRESSION_TOL["bf16"] * np.abs(case.C).max()
    lib, buf = G.load(), case.buf
    import ctypes
    args = [buf.code, buf.n, buf.k, buf.m, ctypes.c_void_p(buf.C.data_ptr()), buf.C.stride(0), ctypes.c_void_p(buf.P_rL.data_ptr()), buf.P_rL.stride(0),
            ctypes.c_void_p(buf.P_cL.data_ptr()), buf.P_cL.stride(0), None, ctypes.c_void_p(buf.sumsq_a.data_ptr()), ctypes.c_void_p(buf.sumsq_b.data_ptr())]
    tail = [ctypes.c_void_p(buf.report.data_ptr()), ctypes.c_void_p(buf.workspace.data_ptr()), buf.workspace.numel(), None]
    assert lib.gecc_tl_decode(*args, G.SINGLE_CHECKSUM, *tail) == -2          # GECC_EUNSUPPORTED
    assert lib.gecc_tl_decode(*args, 7, *tail) == -1                          # GECC_EINVAL
    assert lib.gecc_tl_decode(*args[:-2], None, None, 0, *tail) == -1         # no thresholds and no sums of squares
    assert lib.gecc_tl_decode(*args, 0, tail[0], tail[1], 16, None) == -4      # GECC_EWORKSPACE


def test_bench_size_bf16_errors_in_sixteen_blocks():
    """4096^3 (BASELINE.json configs[2]): 32 errors, two per block on 16 blocks, the oracle in error space (the checks are linear
    and the panel parity of a valid product cancels: decode the faults' effect on a zero product)."""
    n = k = m = 4096
    dtype = "bf16"
    A_h, B_h = I.make_operands(n, k, m, 21, dtype=dtype)
    A = torch.from_numpy(A_h).cuda().to(torch.bfloat16)
    B = torch.from_numpy(B_h).cuda().to(torch.bfloat16)
    buf = G.TlBuffers(n, k, m, torch.bfloat16)
    rng = np.random.default_rng(5)
    faults = []
    for b in range(16):
        rb, cb = int(rng.integers(0, 32)), b * 2
        i1, i2 = rng.choice(128, 2, replace=False)
        j1, j2 = rng.choice(128, 2, replace=False)
        faults += [(I.KIND_C, rb * 128 + int(i1), cb * 128 + int(j1), float(rng.uniform(20, 100))),
                   (I.KIND_C, rb * 128 + int(i2), cb * 128 + int(j2), -float(rng.uniform(20, 100)))]
    G.tl_protected_matmul(A, B, buf, faults=faults)
    torch.cuda.synchronize()
    rep = G.read_tl_report(buf.report)
    ssa, ssb = float((A_h.astype(np.float64) ** 2).sum()), float((B_h.astype(np.float64) ** 2).sum())
    tau = stated_thresholds(dtype, P, k, Q, ssa * P / n, ssb * Q / m)
    E = np.zeros((n, m))
    for _, r, c, e in faults:
        E[r, c] += np.float32(e)
    orc = O.decode_panels(E, np.zeros((n, 1)), np.zeros((1, m)), P, Q, lambda rows, cols: tau)
    assert orc.verdict == O.CORRECTED and rep.verdict == G.CORRECTED
    assert rep.n_found == len(orc.found) == 32 and rep.located() == orc.located()
    assert np.abs(orc.C).max() < 1e-9
    # values: every touched row against fp64 dot products, and the untouched sample
    A64, B64 = A_h.astype(np.float64), B_h.astype(np.float64)
    scale = 5.0 * np.sqrt(k)
    for _, r, c, _e in faults[::4]:
        assert np.abs(buf.C[r].double().cpu().numpy() - A64[r] @ B64).max() <= 1e-4 * scale
    # a fault-free product of the same operands raises no flag
    G.tl_protected_matmul(A, B, buf)
    torch.cuda.synchronize()
    rep = G.read_tl_report(buf.report)
    assert rep.verdict == G.CLEAN and rep.n_row_flags == 0 and rep.n_col_flags == 0
    assert all(rep.max_abs_syndrome[q] <= 0.9 * rep.tau[q] for q in range(4))
