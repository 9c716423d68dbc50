"""`-m gpu` parity at BASELINE.json's FULL sizes, where the CPU oracle cannot form the whole fp64 product: sampled checks
(SURVEY 8(d)).

The detection / correction algebra is linear, so the oracle runs in ERROR SPACE: the encoded product of the fault-free
operands has zero syndromes, hence the syndromes of the faulty C_bar are those of the faults' exact
effect E alone (O.fault_effects on a zero matrix).  The oracle decodes E (verdict, located set, what it leaves behind), and
the GPU's corrected C is compared with (fp64 dot products + what the oracle left) on every row / column a fault touched
and on 1e5 random symbols.  Verdict and located positions bit-exact, values within the north-star tolerance AND within
the regression bound near what is achieved.
"""
import pytest

from paper_2508_04355_b200 import inputs as I

pytestmark = pytest.mark.gpu

from gpu_harness import SampledCase  # noqa: E402,F401


def _trials(case, scens, seed0, lo=1.0, hi=100.0):
    done = 0
    for t, scen in enumerate(scens):
        faults = I.draw_faults(case.n, case.k, case.m, I.SCENARIOS[scen], seed=seed0 + 17 * t, lo=lo, hi=hi)
        real = case.realise(faults)
        if any(f[3] == 0.0 for f in real):
            continue
        case.check(faults, 1)
        done += 1
    return done


def test_config3_dX_full_size_bf16():
    """dX = dY W^T of the wide projection (BASELINE.json config 3): n = 8192 tokens, k = 14336, m = 4096, B = W^T stored as W."""
    case = SampledCase(8192, 14336, 4096, "bf16", seed=51, std_b=0.02, trans_b=1)
    case.check([], 1)
    assert _trials(case, ("d", "e", "f", "a"), 61000) >= 3


def test_config3_dW_full_size_bf16():
    """dW = X^T dY of the wide projection: n = 4096, k = 8192 tokens, m = 14336, A = X^T stored as X."""
    case = SampledCase(4096, 8192, 14336, "bf16", seed=52, trans_a=1)
    case.check([], 1)
    assert _trials(case, ("d", "e", "f", "b"), 62000) >= 3


def test_config3_square_projection_backward_full_size_bf16():
    """The 4096 x 4096 weight: dX = dY W^T (8192 x 4096 x 4096, B^T stored) and dW = X^T dY (4096 x 8192 x 4096, A^T stored)."""
    case = SampledCase(8192, 4096, 4096, "bf16", seed=53, std_b=0.02, trans_b=1)
    assert _trials(case, ("d", "e", "f"), 63000) >= 2
    case = SampledCase(4096, 8192, 4096, "bf16", seed=54, trans_a=1)
    assert _trials(case, ("d", "e", "f"), 64000) >= 2


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
@pytest.mark.parametrize("size", [8192, 16384])
def test_config4_large_squares_sampled(dtype, size):
    """The top of the size sweep (BASELINE.json config 4).  At 16384^3 fp32 the plain threshold is ~2 (c(k) grows with k):
    faults are drawn with |e| in [8, 100] so that every footprint is far above it, and the oracle decides at the same tau."""
    case = SampledCase(size, size, size, dtype, seed=55, samples=50_000)
    case.check([], 1)
    assert _trials(case, ("a", "c", "e", "f") if size == 8192 else ("a", "f"), 65000 + size, lo=8.0, hi=100.0) >= 2
