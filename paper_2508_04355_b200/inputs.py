"""Seeded synthetic input generators shared by the tests, bench.py and the oracle's callers.

This module holds NONE of the method's arithmetic (no checksums, no products, no syndromes):
only random matrices of the shapes / distributions of BASELINE.json's configs, dtype rounding
of those inputs, and random fault lists.  numpy only -- it never touches the CUDA library, so
the oracle side can be fed from it without importing the product path.

Recipe:
  * matrices: numpy PCG64 stream `default_rng([seed, tag])`, N(0, std) or U(-1, 1), generated in
    fp64, rounded once to the operand dtype (fp32 by IEEE round-to-nearest-even cast, bf16 by
    round-to-nearest-even of the fp32 bit pattern).  The rounded values are what BOTH sides see.
  * faults: (kind, row, col, value) with kind 0 = symbol of A, 1 = symbol of B, 2 = symbol of C
    (E1/E2/E3), 0-based positions in the DATA parts, additive.
"""
from __future__ import annotations

import numpy as np

KIND_A, KIND_B, KIND_C = 0, 1, 2

# scenario classes: PAPER.md:241 (a-f) plus the input-pair classes the paper never tests
SCENARIOS = {
    "none": (),
    "a": (KIND_A,), "b": (KIND_B,), "c": (KIND_C,),
    "d": (KIND_A, KIND_C), "e": (KIND_B, KIND_C), "f": (KIND_C, KIND_C),
    "aa": (KIND_A, KIND_A), "bb": (KIND_B, KIND_B), "ab": (KIND_A, KIND_B),
}


def round_to_bf16(x: np.ndarray) -> np.ndarray:
    """Round fp32/fp64 values to the nearest bf16 (ties to even); returned as fp32 holding bf16 values."""
    f = np.ascontiguousarray(x, dtype=np.float32)
    u = f.view(np.uint32).astype(np.uint64)
    lsb = (u >> 16) & 1
    u = (u + 0x7FFF + lsb) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(f.shape)


def bf16_bits(x_f32_holding_bf16: np.ndarray) -> np.ndarray:
    """Upper 16 bits of fp32 values that are exactly bf16-representable (uint16, same shape)."""
    f = np.ascontiguousarray(x_f32_holding_bf16, dtype=np.float32)
    return (f.view(np.uint32) >> 16).astype(np.uint16).reshape(f.shape)


def bf16_bits_to_f32(bits: np.ndarray) -> np.ndarray:
    b = np.ascontiguousarray(bits, dtype=np.uint16)
    return (b.astype(np.uint32) << 16).view(np.float32).reshape(b.shape)


def round_to_dtype(x: np.ndarray, dtype: str) -> np.ndarray:
    """dtype 'f32' or 'bf16'; result is fp32 storage holding values exact in that dtype."""
    if dtype == "f32":
        return np.ascontiguousarray(x, dtype=np.float32)
    if dtype == "bf16":
        return round_to_bf16(x)
    raise ValueError(dtype)


def make_matrix(rows: int, cols: int, seed: int, tag: int, dist: str = "normal", std: float = 1.0,
                dtype: str = "f32") -> np.ndarray:
    """rows x cols matrix, i.i.d. N(0, std) ('normal') or U(-1, 1) ('uniform'), rounded to dtype."""
    rng = np.random.default_rng([int(seed), int(tag)])
    if dist == "normal":
        x = rng.standard_normal((rows, cols)) * std
    elif dist == "uniform":
        x = rng.uniform(-1.0, 1.0, (rows, cols))
    else:
        raise ValueError(dist)
    return round_to_dtype(x, dtype)


def make_operands(n: int, k: int, m: int, seed: int, dist: str = "normal", dtype: str = "f32",
                  std_a: float = 1.0, std_b: float = 1.0):
    """A (n x k), B (k x m) of one config, PAPER.md:31 notation."""
    return (make_matrix(n, k, seed, 1, dist, std_a, dtype),
            make_matrix(k, m, seed, 2, dist, std_b, dtype))


def draw_magnitude(rng, lo: float, hi: float, law: str) -> float:
    """|e| uniform in [lo, hi] ('uniform') or log-uniform ('log'), random sign."""
    if law == "uniform":
        mag = rng.uniform(lo, hi)
    elif law == "log":
        mag = float(np.exp(rng.uniform(np.log(lo), np.log(hi))))
    else:
        raise ValueError(law)
    return float(mag if rng.random() < 0.5 else -mag)


def draw_faults(n: int, k: int, m: int, kinds, seed: int, lo: float = 1.0, hi: float = 100.0,
                law: str = "uniform", force: str | None = None):
    """Random fault list for one trial.  `kinds` is a tuple from SCENARIOS.

    `force` selects the sub-cases DESIGN.md lists for two-fault classes:
      'same_row'  - both faults land in the same row of C (A-row = C-row, or two C in one row)
      'same_col'  - same column of C
      'same_l'    - both input faults share the inner index l
    Positions are distinct symbols (two faults on one symbol are one fault, reading R16).
    """
    rng = np.random.default_rng([int(seed), 77])
    dims = {KIND_A: (n, k), KIND_B: (k, m), KIND_C: (n, m)}
    for _ in range(1000):
        faults = []
        for kind in kinds:
            r, c = dims[kind]
            faults.append([kind, int(rng.integers(r)), int(rng.integers(c)), draw_magnitude(rng, lo, hi, law)])
        if len(faults) == 2 and force:
            f0, f1 = faults

            def c_row(f):  # row of C a fault touches (None if it touches a whole column)
                return f[1] if f[0] in (KIND_A, KIND_C) else None

            def c_col(f):
                return f[2] if f[0] in (KIND_B, KIND_C) else None

            if force == "same_row" and c_row(f0) is not None and c_row(f1) is not None:
                f1[1] = f0[1]
            elif force == "same_col" and c_col(f0) is not None and c_col(f1) is not None:
                f1[2] = f0[2]
            elif force == "same_l":
                l0 = f0[2] if f0[0] == KIND_A else (f0[1] if f0[0] == KIND_B else None)
                if l0 is not None and f1[0] == KIND_A:
                    f1[2] = l0
                elif l0 is not None and f1[0] == KIND_B:
                    f1[1] = l0
        sites = {(f[0], f[1], f[2]) for f in faults}
        if len(sites) == len(faults):
            return [tuple(f) for f in faults]
    raise RuntimeError("could not draw distinct fault sites")


def realise_input_fault(x_rounded: np.ndarray, row: int, col: int, e: float, dtype: str) -> float:
    """Value stored when fault e hits a dtype-rounded operand symbol: round_dtype(x + e).

    Returns the stored value; the realised additive fault is stored - x (exact in fp64).
    """
    v = np.float64(x_rounded[row, col]) + np.float64(e)
    return float(round_to_dtype(np.array([v]), dtype)[0])
