"""Pins for the CPU fp64 oracle (oracle/gecc_oracle.py) against what the paper and the mathematics fix.

None of these tests retypes an oracle formula and compares it with itself: each one checks the oracle against
(a) a value the paper prints, (b) an identity / theorem the paper states, (c) ground truth of an injection
(the fault-free product, the injected positions), or (d) brute force on tiny inputs.
Citations are PAPER.md lines.
"""
import itertools
import os

import numpy as np
import pytest

from oracle import gecc_oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _ops(n, k, m, seed):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((n, k)), rng.standard_normal((k, m)), rng


# ---------------------------------------------------------------- encoder + product -----------
def test_encoder_against_plain_python_sums():
    """PAPER.md:77-83 / 95-101 written out as scalar python loops over 1-based indices."""
    A, B, _ = _ops(5, 4, 6, 1)
    AP, BP = O.encode_left(A), O.encode_right(B)
    for l in range(4):
        assert AP[0, l] == pytest.approx(sum(A[i - 1, l] for i in range(1, 6)), abs=1e-13)
        assert AP[1, l] == pytest.approx(sum(i * A[i - 1, l] for i in range(1, 6)), abs=1e-13)
        assert BP[l, 0] == pytest.approx(sum(B[l, j - 1] for j in range(1, 7)), abs=1e-13)
        assert BP[l, 1] == pytest.approx(sum(j * B[l, j - 1] for j in range(1, 7)), abs=1e-13)


def test_encoder_is_generator_matrix_product():
    """A_bar = G_A A with G_A = [I_n; 1; (1..n)] and B_bar = B G_B (reading R2 for the shapes)."""
    A, B, _ = _ops(7, 3, 5, 2)
    GA = np.vstack([np.eye(7), np.ones((1, 7)), np.arange(1, 8)[None, :]])
    GB = np.hstack([np.eye(5), np.ones((5, 1)), np.arange(1, 6)[:, None]])
    Abar, Bbar = O.encoded_operands(A, B)
    assert Abar.shape == (9, 3) and Bbar.shape == (3, 7)
    np.testing.assert_allclose(Abar, GA @ A, atol=1e-13)
    np.testing.assert_allclose(Bbar, B @ GB, atol=1e-13)


def test_block_identities_of_encoded_product():
    """C_bar = [[C, P_r], [P_c, P_g]] with P_r = C [1, w_m], P_c = [1; w_n] C, P_g = [1; w_n] C [1, w_m]
    (PAPER.md:117-135).  Fails if a weight vector starts at 0, is transposed, or belongs to the wrong side."""
    n, k, m = 6, 5, 4
    A, B, _ = _ops(n, k, m, 3)
    Cbar = O.encoded_product(*O.encoded_operands(A, B))
    C = A @ B
    wn, wm = np.arange(1, n + 1.0), np.arange(1, m + 1.0)
    np.testing.assert_allclose(Cbar[:n, :m], C, atol=1e-12)
    np.testing.assert_allclose(Cbar[:n, m], C.sum(1), atol=1e-12)
    np.testing.assert_allclose(Cbar[:n, m + 1], C @ wm, atol=1e-12)
    np.testing.assert_allclose(Cbar[n, :m], C.sum(0), atol=1e-12)
    np.testing.assert_allclose(Cbar[n + 1, :m], wn @ C, atol=1e-12)
    np.testing.assert_allclose(Cbar[n:, m:], np.array([[C.sum(), (C @ wm).sum()], [wn @ C.sum(1), wn @ C @ wm]]), atol=1e-10)


def test_product_matches_scalar_triple_loop():
    """c_ij = sum_l a_il b_lj as a pure-python triple loop over the encoded operands."""
    A, B, _ = _ops(4, 5, 3, 4)
    Abar, Bbar = O.encoded_operands(A, B)
    np.testing.assert_allclose(O.encoded_product(Abar, Bbar), O.encoded_product_loops(Abar.tolist(), Bbar.tolist()), atol=1e-12)


# ---------------------------------------------------------------- syndromes -------------------
@pytest.mark.parametrize("shape", [(4, 3, 4), (64, 64, 64), (33, 70, 129)])
def test_syndromes_vanish_on_fault_free_data(shape):
    """Def. 1 constraints (2)(3): every row / column check is 0 on a valid codeword."""
    n, k, m = shape
    A, B, _ = _ops(n, k, m, 5)
    Cbar = O.encoded_product(*O.encoded_operands(A, B))
    scale = np.abs(Cbar).max()
    for s in O.syndromes(Cbar):
        assert np.abs(s).max() <= 1e-11 * scale
    rep = O.decode_level_p(Cbar, O.fp64_thresholds(n, m, Cbar))
    assert rep.verdict == O.CLEAN and rep.found == [] and rep.n_row_flags == 0 and rep.n_col_flags == 0


def test_fault_before_encoding_is_undetectable():
    """Reading R1 of PAPER.md:45: parity generated from already-corrupted data is a valid codeword of the wrong product."""
    A, B, _ = _ops(6, 4, 5, 6)
    A[2, 1] += 37.0
    Cbar = O.encoded_product(*O.encoded_operands(A, B))
    assert O.decode_level_p(Cbar, O.fp64_thresholds(6, 5, Cbar)).verdict == O.CLEAN


def test_syndrome_signatures_of_single_faults():
    """What each fault class does to the four syndrome vectors (PAPER.md:43 and Def. 1), signs included:
    C(i,j,e): r=(e, j e) at i, q=(e, i e) at j.  A(i,l,e): r = 0, q_y = (e b_ly, i e b_ly).  B(l,j,e): mirrored."""
    n, k, m = 5, 4, 6
    A, B, _ = _ops(n, k, m, 7)
    Abar, Bbar = O.encoded_operands(A, B)
    e = 3.5
    # C fault at 1-based (2, 5)
    Cb = O.inject_output_faults(O.encoded_product(Abar, Bbar), [(O.KIND_C, 1, 4, e)])
    r1, r2, q1, q2 = O.syndromes(Cb)
    exp = np.zeros(n); exp[1] = e
    np.testing.assert_allclose(r1, exp, atol=1e-10); np.testing.assert_allclose(r2, 5 * exp, atol=1e-10)
    exp = np.zeros(m); exp[4] = e
    np.testing.assert_allclose(q1, exp, atol=1e-10); np.testing.assert_allclose(q2, 2 * exp, atol=1e-10)
    # A fault at 1-based (4, 3)
    Af, Bf = O.inject_input_faults(Abar, Bbar, [(O.KIND_A, 3, 2, e)])
    r1, r2, q1, q2 = O.syndromes(O.encoded_product(Af, Bf))
    assert np.abs(r1).max() < 1e-10 and np.abs(r2).max() < 1e-9
    np.testing.assert_allclose(q1, e * B[2, :], atol=1e-10); np.testing.assert_allclose(q2, 4 * e * B[2, :], atol=1e-10)
    # B fault at 1-based (2, 6)
    Af, Bf = O.inject_input_faults(Abar, Bbar, [(O.KIND_B, 1, 5, e)])
    r1, r2, q1, q2 = O.syndromes(O.encoded_product(Af, Bf))
    assert np.abs(q1).max() < 1e-10 and np.abs(q2).max() < 1e-9
    np.testing.assert_allclose(r1, e * A[:, 1], atol=1e-10); np.testing.assert_allclose(r2, 6 * e * A[:, 1], atol=1e-10)


def test_linearity_shortcut_equals_full_recompute():
    n, k, m = 7, 6, 5
    A, B, rng = _ops(n, k, m, 8)
    Abar, Bbar = O.encoded_operands(A, B)
    Cc = O.encoded_product(Abar, Bbar)
    for faults in ([(0, 2, 3, 5.0), (1, 3, 4, -7.0)], [(0, 2, 3, 5.0), (1, 1, 4, -7.0), (2, 6, 0, 2.0)], [(0, 0, 0, 1.5), (0, 6, 5, 2.5)]):
        Af, Bf = O.inject_input_faults(Abar, Bbar, faults)
        full = O.inject_output_faults(O.encoded_product(Af, Bf), faults)
        np.testing.assert_allclose(O.fault_effects(Cc, Abar, Bbar, faults), full, atol=1e-10)
