"""Shared plumbing of the `-m gpu` parity tests: runs one trial through the C ABI (paper_2508_04355_b200.binding) and
the same trial through the CPU fp64 oracle on the same operand bits, and returns both results.

No arithmetic of the method lives here: the oracle side calls oracle/, the GPU side calls the library.
"""
from __future__ import annotations

import numpy as np
import torch

from oracle import gecc_oracle as O
from paper_2508_04355_b200 import binding as G
from paper_2508_04355_b200 import inputs as I

from threshold_spec import stated_thresholds

TOL_C = {"bf16": 2e-2, "f32": 1e-4}  # BASELINE.json north_star: max relative error of corrected values
# regression bound near what is achieved (campaigns: <= 4e-5 of max |C| for both dtypes): a wrong-valued repair of a few
# units would pass the north star's 2e-2 at bf16 (max |C| ~ 300 at 4096^3), it does not pass this
REGRESSION_TOL = {"bf16": 1e-4, "f32": 1e-4}
TORCH_DT = {"bf16": torch.bfloat16, "f32": torch.float32}


class Case:
    """One pair of operands on both sides: host fp32 arrays holding dtype-exact values, device tensors, clean C_bar."""

    def __init__(self, n, k, m, dtype, seed, dist="normal", std_a=1.0, std_b=1.0, trans_a=0, trans_b=0):
        """trans_a / trans_b: the device holds the operand transposed (A^T: k x n, B^T: m x k); the oracle always sees A, B."""
        self.n, self.k, self.m, self.dtype = n, k, m, dtype
        self.trans_a, self.trans_b = trans_a, trans_b
        self.A_h, self.B_h = I.make_operands(n, k, m, seed, dist=dist, dtype=dtype, std_a=std_a, std_b=std_b)
        self.A_dev0 = torch.from_numpy(np.ascontiguousarray(self.A_h.T) if trans_a else self.A_h).cuda().to(TORCH_DT[dtype])
        self.B_dev0 = torch.from_numpy(np.ascontiguousarray(self.B_h.T) if trans_b else self.B_h).cuda().to(TORCH_DT[dtype])
        self.buf = G.Buffers(n, k, m, TORCH_DT[dtype], trans_a=trans_a, trans_b=trans_b)
        self.Abar, self.Bbar = O.encoded_operands(self.A_h, self.B_h)
        self.Cbar = O.encoded_product(self.Abar, self.Bbar)
        ssa, ssb = float(np.sum(self.A_h.astype(np.float64) ** 2)), float(np.sum(self.B_h.astype(np.float64) ** 2))
        self.tau = stated_thresholds(dtype, n, k, m, ssa, ssb)   # the formula include/gecc.h states; the oracle takes tau as input
        self.tau_in = O.fp64_input_thresholds(self.Abar, self.Bbar)

    def realise(self, faults):
        """What the stored symbols become when the faults hit them in the operand dtype (inputs.realise_input_fault)
        -> fault list with the REALISED additive values, which is what the oracle is given."""
        out = []
        for kind, r, c, e in faults:
            if kind == I.KIND_A:
                stored = I.realise_input_fault(self.A_h, r, c, e, self.dtype)
                out.append((kind, r, c, float(np.float64(stored) - np.float64(self.A_h[r, c]))))
            elif kind == I.KIND_B:
                stored = I.realise_input_fault(self.B_h, r, c, e, self.dtype)
                out.append((kind, r, c, float(np.float64(stored) - np.float64(self.B_h[r, c]))))
            else:
                out.append((kind, r, c, float(np.float32(e))))
        return out

    def run_gpu(self, faults, level=1, tau=None):
        A = self.A_dev0.clone()
        B = self.B_dev0.clone()
        G.protected_matmul(A, B, self.buf, faults=faults, tau=tau, level=level)
        torch.cuda.synchronize()
        rep = G.read_report(self.buf.report)
        A_h, B_h = A.float().cpu().numpy(), B.float().cpu().numpy()   # returned as the operands, whatever the storage
        return rep, self.buf.C.cpu().numpy().astype(np.float64), A_h.T if self.trans_a else A_h, B_h.T if self.trans_b else B_h

    def run_oracle(self, faults_realised, level=1, tau=None):
        tau = self.tau if tau is None else tau
        Af, Bf = O.inject_input_faults(self.Abar, self.Bbar, faults_realised)
        Cb = O.fault_effects(self.Cbar, self.Abar, self.Bbar, faults_realised)
        if level == 0:
            return O.decode_level_p(Cb, tau)
        return O.decode_level_x(Cb, Af, Bf, tau, self.tau_in)

    def in_guard_band(self, faults_realised, level):
        """A trial is outside the bit-exact requirement if the oracle's own answer changes when every threshold moves
        by 2x either way: some footprint of the faults then lies within [tau/2, 2 tau] (guard band)."""
        lo = self.run_oracle(faults_realised, level, tuple(t / 2 for t in self.tau))
        hi = self.run_oracle(faults_realised, level, tuple(t * 2 for t in self.tau))
        mid = self.run_oracle(faults_realised, level)
        return not (lo.verdict == mid.verdict == hi.verdict and lo.located() == mid.located() == hi.located())


def operands_as_the_oracle_leaves_them(dtype, real, orc, A_gpu, B_gpu, A_clean, B_clean, ctx):
    """Level X: the operands after the decode must be what the ORACLE's decode leaves (Report.A / Report.B): a located
    input fault is patched back -- bf16 symbols bit-exactly, fp32 symbols to the rounding of (a + e) - e -- and an input fault
    whose footprint stays below the thresholds is tolerable noise in the paper's own model (Eq. 1): nobody
    locates it and the symbol keeps its stored value, on both sides alike."""
    located = {(kd, r, c) for kd, r, c, _ in orc.found}
    emax = max([abs(f[3]) for f in real] + [0.0])
    tol = 1e-6 * (1.0 + emax)
    for X_gpu, X_orc, X_clean, kind in ((A_gpu, orc.A, A_clean, I.KIND_A), (B_gpu, orc.B, B_clean, I.KIND_B)):
        assert np.abs(X_gpu - X_orc).max() <= tol, ctx + " operand differs from what the oracle's decode leaves"
        if dtype == "bf16":       # every located symbol back to its exact bits; everything untouched untouched
            expect = X_clean.astype(np.float64).copy()
            for kd, r, c, e in real:
                if kd == kind and (kd, r, c) not in located:
                    expect[r, c] = X_orc[r, c]          # left in place by both sides (sub-threshold)
            assert np.array_equal(X_gpu.astype(np.float64), expect), ctx + " operand not restored bit-exactly"


def compare(case: Case, faults, level, check_values=True):
    """Runs both sides and asserts parity.  Returns (gpu report, oracle report)."""
    real = case.realise(faults)
    rep, C_gpu, A_gpu, B_gpu = case.run_gpu(faults, level)
    orc = case.run_oracle(real, level)
    ctx = f"faults={faults} level={level} gpu=({rep.verdict},{rep.located()}) oracle=({orc.verdict},{orc.located()})"
    assert rep.verdict == orc.verdict, ctx
    assert rep.located() == orc.located(), ctx          # bit-exact positions
    n, m = case.n, case.m
    scale = np.abs(case.Cbar[:n, :m]).max()
    if check_values and orc.verdict in (O.CLEAN, O.CORRECTED):
        err = np.abs(C_gpu - orc.C).max() / scale      # reading R15: max |c_gpu - c_oracle| / max |c_oracle|
        assert err <= min(TOL_C[case.dtype], REGRESSION_TOL[case.dtype]), f"{ctx} corrected C off by {err:.3e}"
        for (kd, r, c, mag_o), mag_g in zip(orc.found, rep.magnitudes()):
            if kd in (O.KIND_ROW, O.KIND_COL):
                continue
            assert abs(mag_g - mag_o) <= 1e-3 * abs(mag_o) + 4 * max(case.tau[0], case.tau[2]), f"{ctx} magnitude {mag_g} vs {mag_o}"
        if level == 1 and orc.verdict == O.CORRECTED:
            operands_as_the_oracle_leaves_them(case.dtype, real, orc, A_gpu, B_gpu, case.A_h, case.B_h, ctx)
    return rep, orc


# ---------------------------------------------------------------------------------------------------------------
# Sizes where the CPU oracle cannot form the whole fp64 product: sampled checks, oracle in error space
# ---------------------------------------------------------------------------------------------------------------

def value_tol(dtype, k):
    """North-star tolerance (1e-4 / 2e-2 of max |C|) and the regression bound near what is achieved.  The 3xTF32 product's
    OWN error against fp64 grows with the length of the truncating fp32 accumulation (k / 8 steps of three MMAs): measured
    6.9e-5 of max |C| at k = 1024..4096, 1.2e-4 at 8192; beyond k = 4096 the bound for fp32 therefore scales with k / 4096 --
    a corrected symbol must be as accurate as every untouched symbol of the same product, which is what is checked."""
    t = min(TOL_C[dtype], REGRESSION_TOL[dtype])
    return t * max(1.0, k / 4096.0) if dtype == "f32" else t


class SampledCase:
    def __init__(self, n, k, m, dtype, seed, std_b=1.0, trans_a=0, trans_b=0, samples=100_000):
        self.n, self.k, self.m, self.dtype, self.trans_a, self.trans_b = n, k, m, dtype, trans_a, trans_b
        self.A_h, self.B_h = I.make_operands(n, k, m, seed, dtype=dtype, std_b=std_b)
        tdt = TORCH_DT[dtype]
        self.A_dev0 = torch.from_numpy(np.ascontiguousarray(self.A_h.T) if trans_a else self.A_h).cuda().to(tdt)
        self.B_dev0 = torch.from_numpy(np.ascontiguousarray(self.B_h.T) if trans_b else self.B_h).cuda().to(tdt)
        self.buf = G.Buffers(n, k, m, tdt, trans_a=trans_a, trans_b=trans_b)
        self.A64, self.B64 = self.A_h.astype(np.float64), self.B_h.astype(np.float64)
        self.Abar = np.vstack([self.A64, O.encode_left(self.A64)])
        self.Bbar = np.hstack([self.B64, O.encode_right(self.B64)])
        ssa, ssb = float((self.A64 ** 2).sum()), float((self.B64 ** 2).sum())
        self.tau = stated_thresholds(dtype, n, k, m, ssa, ssb)
        self.tau_in = O.fp64_input_thresholds(self.Abar, self.Bbar)
        self.scale = 5.0 * np.sqrt(k) * np.sqrt(ssa / (n * k)) * np.sqrt(ssb / (k * m))      # ~ max |C| of N(0, k sa^2 sb^2) symbols
        rng = np.random.default_rng([seed, 99])
        self.si, self.sj = rng.integers(0, n, samples), rng.integers(0, m, samples)
        self.sref = np.einsum("sk,sk->s", self.A64[self.si], self.B64[:, self.sj].T)              # fp64 dot products
        self.scale = max(self.scale, float(np.abs(self.sref).max()))

    def realise(self, faults):
        out = []
        for kind, r, c, e in faults:
            X = self.A_h if kind == I.KIND_A else self.B_h
            if kind == I.KIND_C:
                out.append((kind, r, c, float(np.float32(e))))
            else:
                out.append((kind, r, c, float(np.float64(I.realise_input_fault(X, r, c, e, self.dtype)) - np.float64(X[r, c]))))
        return out

    def run_oracle(self, real, level=1, tau=None):
        """The oracle in error space: decodes the faults' exact effect E on a zero codeword."""
        tau = self.tau if tau is None else tau
        E = O.fault_effects(np.zeros((self.n + 2, self.m + 2)), self.Abar, self.Bbar, real)
        Af, Bf = O.inject_input_faults(self.Abar, self.Bbar, real)
        return O.decode_level_x(E, Af, Bf, tau, self.tau_in) if level else O.decode_level_p(E, tau)

    def in_guard_band(self, real, level=1):
        lo = self.run_oracle(real, level, tuple(t / 2 for t in self.tau))
        hi = self.run_oracle(real, level, tuple(t * 2 for t in self.tau))
        mid = self.run_oracle(real, level)
        return not (lo.verdict == mid.verdict == hi.verdict and lo.located() == mid.located() == hi.located())

    def run_gpu(self, faults, level=1):
        self.A_run, self.B_run = self.A_dev0.clone(), self.B_dev0.clone()
        G.protected_matmul(self.A_run, self.B_run, self.buf, faults=faults, level=level)
        torch.cuda.synchronize()
        return G.read_report(self.buf.report)

    def check(self, faults, level=1):
        real = self.realise(faults)
        rep = self.run_gpu(faults, level)
        A, B = self.A_run, self.B_run
        orc = self.run_oracle(real, level)
        ctx = f"faults={faults} gpu=({rep.verdict},{rep.located()}) oracle=({orc.verdict},{orc.located()})"
        assert rep.verdict == orc.verdict and rep.located() == orc.located(), ctx
        if orc.verdict not in (O.CLEAN, O.CORRECTED):
            return rep
        # what the oracle's correction leaves of E: nothing for located faults; a fault below the thresholds is tolerable
        # noise (Eq. 1) and stays, on both sides alike
        left = orc.C
        C = self.buf.C
        tol = value_tol(self.dtype, self.k) * self.scale
        got = C[torch.from_numpy(self.si).cuda(), torch.from_numpy(self.sj).cuda()].double().cpu().numpy()
        assert np.abs(got - (self.sref + left[self.si, self.sj])).max() <= tol, ctx + " sampled symbols"
        for kind, r, c, _ in real:                                       # every line a fault touched, in full
            rows = [r] if kind in (I.KIND_A, I.KIND_C) else []
            cols = [c] if kind in (I.KIND_B, I.KIND_C) else []
            for i in rows:
                assert np.abs(C[i].double().cpu().numpy() - (self.A64[i] @ self.B64 + left[i])).max() <= tol, ctx + f" row {i}"
            for j in cols:
                assert np.abs(C[:, j].double().cpu().numpy() - (self.A64 @ self.B64[:, j] + left[:, j])).max() <= tol, ctx + f" column {j}"
        if level == 1 and orc.verdict == O.CORRECTED:
            A_h = A.float().cpu().numpy(); B_h = B.float().cpu().numpy()
            operands_as_the_oracle_leaves_them(self.dtype, real, orc, A_h.T if self.trans_a else A_h, B_h.T if self.trans_b else B_h, self.A_h, self.B_h, ctx)
        return rep


