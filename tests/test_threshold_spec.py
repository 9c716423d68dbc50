"""CPU pins (`-m "not gpu"`) for the threshold formula that include/gecc.h states (tests/threshold_spec.py).

The paper fixes no threshold (one delta of unstated scale; Eq. 1, PAPER.md:51-57 only says that
noise below delta is tolerated and errors above it are detected), so these pins are what the mathematics of the
checks fixes: how a threshold must transform when the data is rescaled, how the weighted check relates to the plain
one, and that the formula separates the rounding noise of an fp32-accumulated product from an injected error.
"""
import numpy as np
import pytest

from oracle import gecc_oracle as O
from threshold_spec import KAPPA, noise_coeff, rms_weight, stated_thresholds


def test_header_states_the_same_constants():
    """include/gecc.h is the statement of record: the constants restated in threshold_spec.py must appear there."""
    import os
    import re
    hdr = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "gecc.h")).read()
    m = re.search(r"c\(k\) = (\d+(?:\.\d+)?) \+ c0 \(k / 1024\)\^\(2/3\)", hdr)
    assert m and float(m.group(1)) == 2.0
    assert re.search(r"c0 = 4\.5 \(GECC_BF16\)", hdr) and re.search(r"20 \(GECC_F32\)", hdr)
    assert re.search(r"kappa = 16", hdr)


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_scale_covariance(dtype):
    """Syndromes are bilinear in (A, B): tau(alpha A, beta B) = alpha beta tau(A, B)."""
    n, k, m = 96, 160, 224
    ssa, ssb = 1234.5, 987.6
    t = stated_thresholds(dtype, n, k, m, ssa, ssb)
    for alpha, beta in ((3.0, 1.0), (0.02, 5.0), (1e-3, 1e3)):
        t2 = stated_thresholds(dtype, n, k, m, alpha ** 2 * ssa, beta ** 2 * ssb)
        np.testing.assert_allclose(t2, [alpha * beta * x for x in t], rtol=1e-12)


def test_weighted_thresholds_follow_the_rms_of_the_weights():
    """The weighted check sums the same noise with weights 1..len: independent terms add in
    quadrature, so tau_2 / tau_1 = sqrt(sum w^2 / len) = sqrt((len+1)(2 len+1)/6), computed here from the weights."""
    for n, m in ((5, 9), (64, 64), (1024, 4096)):
        t = stated_thresholds("bf16", n, 128, m, 1.0, 1.0)
        assert t[1] / t[0] == pytest.approx(np.sqrt(np.mean(np.arange(1, m + 1.0) ** 2)), rel=1e-12)
        assert t[3] / t[2] == pytest.approx(np.sqrt(np.mean(np.arange(1, n + 1.0) ** 2)), rel=1e-12)
        assert rms_weight(m) == pytest.approx(np.sqrt(np.mean(np.arange(1, m + 1.0) ** 2)), rel=1e-12)
    # transposing the product swaps the row and the column thresholds
    a = stated_thresholds("f32", 200, 300, 500, 7.0, 11.0)
    b = stated_thresholds("f32", 500, 300, 200, 11.0, 7.0)           # C^T = B^T A^T: the operands swap roles
    np.testing.assert_allclose([a[2], a[3], a[0], a[1]], b, rtol=1e-12)


@pytest.mark.parametrize("size", [256, 512, 1024, 2048])
def test_fp32_product_noise_stays_below_and_a_4tau_error_is_flagged(size):
    """An fp32-accumulated product (numpy sgemm, no GPU) of N(0,1) operands: every fault-free syndrome stays below its
    stated threshold (no false positive), and a C error of 4 tau_r1 raises exactly the flags of its row and column
    (Eq. 1: noise <= delta tolerated, errors > delta detected)."""
    n = k = m = size
    rng = np.random.default_rng(size)
    A = rng.standard_normal((n, k)).astype(np.float32)
    B = rng.standard_normal((k, m)).astype(np.float32)
    Abar, Bbar = O.encoded_operands(A, B)                            # parity in fp64 from the fp32 data ...
    Cbar = (Abar.astype(np.float32) @ Bbar.astype(np.float32)).astype(np.float64)   # ... product accumulated in fp32
    tau = stated_thresholds("f32", n, k, m, float((A.astype(np.float64) ** 2).sum()), float((B.astype(np.float64) ** 2).sum()))
    syn = O.syndromes(Cbar)
    for s, t in zip(syn, tau):
        assert np.abs(s).max() < t
    R, Q = O.flag_sets(*syn, tau)
    assert R == [] and Q == []
    # the plain syndromes of an fp32 product have sigma ~ c u sqrt(k m) with c of order 1..10: the
    # threshold sits kappa = 16 standard deviations of the MODEL above zero and at least 4 measured ones
    assert tau[0] >= 4.0 * np.std(syn[0]) and tau[2] >= 4.0 * np.std(syn[2])
    assert tau[0] == pytest.approx(KAPPA * noise_coeff("f32", k) * 2.0 ** -24 * np.sqrt(k * m) * A.std() * B.std(), rel=2e-2)
    i, j = size // 3, size // 5
    Cb = O.inject_output_faults(Cbar, [(O.KIND_C, i, j, 4.0 * tau[0])])
    R, Q = O.flag_sets(*O.syndromes(Cb), tau)
    assert R == [i] and Q == [j]
    rep = O.decode_level_p(Cb, tau)
    assert rep.verdict == O.CORRECTED and rep.located() == [(O.KIND_C, i, j)]
