"""The library's AUTOMATIC detection thresholds as include/gecc.h states them (reading R4).

This is a SPECIFICATION restated for the tests, not part of the oracle and not part of the product: the paper
compares every check with one delta in {0.5, 0.1, 0.01} of unstated dtype and data scale, so the
oracle's decoders take their thresholds as INPUT and define none.  The header states

    sigma_plain(len) = c(k) * u * sqrt(k * len) * sigma_a * sigma_b,   c(k) = c_floor + c0 * (k / 1024)^(2/3)
    tau_r1 = kappa * sigma_plain(m)          tau_r2 = tau_r1 * sqrt((m + 1)(2m + 1) / 6)
    tau_q1 = kappa * sigma_plain(n)          tau_q2 = tau_q1 * sqrt((n + 1)(2n + 1) / 6)

with u = 2^-24, kappa = 16, c_floor = 2, c0 = 4.5 (bf16 inputs) / 20 (fp32 inputs via 3xTF32), and sigma_a, sigma_b
the RMS of the operands.  tests/test_threshold_spec.py pins this formula against what mathematics fixes (scale
covariance, the RMS weight of 1..m, the noise of an fp32 product); the `-m gpu` tests assert that the thresholds the
library reports equal it.
"""
from __future__ import annotations

import math

U = 2.0 ** -24
KAPPA = 16.0
C_FLOOR = 2.0
C0 = {"bf16": 4.5, "f32": 20.0}


def noise_coeff(dtype: str, k: int) -> float:
    return C_FLOOR + C0[dtype] * (k / 1024.0) ** (2.0 / 3.0)


def rms_weight(length: int) -> float:
    """sqrt(mean of w^2 over w = 1..length) = sqrt((length + 1)(2 length + 1) / 6)."""
    return math.sqrt((length + 1) * (2 * length + 1) / 6.0)


def stated_thresholds(dtype: str, n: int, k: int, m: int, sumsq_a: float, sumsq_b: float):
    """(tau_r1, tau_r2, tau_q1, tau_q2) for a product of shape (n, k, m) whose operands have the given sums of squares."""
    sigma_a = math.sqrt(sumsq_a / (n * k))
    sigma_b = math.sqrt(sumsq_b / (k * m))
    base = KAPPA * noise_coeff(dtype, k) * U * sigma_a * sigma_b
    t_r1 = base * math.sqrt(k * m)
    t_q1 = base * math.sqrt(k * n)
    return (t_r1, t_r1 * rms_weight(m), t_q1, t_q1 * rms_weight(n))


def stated_global_tolerances(tau, n: int, m: int):
    """Tolerances of the global checks of Eq. (4) as include/gecc.h states them under gecc_decode_correct: the line's
    thresholds times sqrt(len) (times the RMS weight of 1..len for the weighted check).  Returns (rows, cols), each [d][c]."""
    t_r1, t_r2, t_q1, t_q2 = tau
    rows = [[t * math.sqrt(n) for t in (t_r1, t_r2)], [t * math.sqrt(n) * rms_weight(n) for t in (t_r1, t_r2)]]
    cols = [[t * math.sqrt(m) for t in (t_q1, t_q2)], [t * math.sqrt(m) * rms_weight(m) for t in (t_q1, t_q2)]]
    return rows, cols
