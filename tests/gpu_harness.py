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
        assert err <= TOL_C[case.dtype], f"{ctx} corrected C off by {err:.3e}"
        for (kd, r, c, mag_o), mag_g in zip(orc.found, rep.magnitudes()):
            if kd in (O.KIND_ROW, O.KIND_COL):
                continue
            assert abs(mag_g - mag_o) <= 1e-3 * abs(mag_o) + 4 * max(case.tau[0], case.tau[2]), f"{ctx} magnitude {mag_g} vs {mag_o}"
        if level == 1 and orc.verdict == O.CORRECTED:
            # operands restored (Level-X): bf16 symbols bit-exactly, fp32 symbols to rounding of (a + e) - e
            tolA = 0.0 if case.dtype == "bf16" else 1e-6 * (1.0 + max(abs(f[3]) for f in real))
            assert np.abs(A_gpu - case.A_h).max() <= tolA, ctx
            assert np.abs(B_gpu - case.B_h).max() <= tolA, ctx
    return rep, orc
