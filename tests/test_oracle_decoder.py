"""Pins for the oracle's decoder: theorems, printed formulas and worked example of the paper, plus brute force.

Ground truth of every injection (fault-free product, injected positions) is the reference, never the oracle itself.
"""
import itertools
import os

import numpy as np
import pytest

from oracle import gecc_oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _setup(n, k, m, seed):
    rng = np.random.default_rng(seed)
    A, B = rng.standard_normal((n, k)), rng.standard_normal((k, m))
    Abar, Bbar = O.encoded_operands(A, B)
    Cc = O.encoded_product(Abar, Bbar)
    return rng, A, B, Abar, Bbar, Cc, O.fp64_thresholds(n, m, Cc), O.fp64_input_thresholds(Abar, Bbar)


def _sites(n, k, m):
    return ([(O.KIND_A, i, l) for i in range(n) for l in range(k)]
            + [(O.KIND_B, l, j) for l in range(k) for j in range(m)]
            + [(O.KIND_C, i, j) for i in range(n) for j in range(m)])


def _expected(faults):
    """Verdict table of DESIGN.md (from Thm 1/2, PAPER.md:166,176 and the ambiguity argument for input pairs).
    Returns (level_p verdict, level_x verdict)."""
    cls = "".join("ABC"[f[0]] for f in faults)
    if cls in ("A", "B", "C", "AC", "BC", "CC"):
        return O.CORRECTED, O.CORRECTED                      # scenarios a-f
    f0, f1 = faults
    if cls == "AA":
        if f0[1] == f1[1]:
            return O.CORRECTED, O.CORRECTED                  # one row of C: E(1,t)
        return O.UNCORRECTABLE, (O.UNCORRECTABLE_INPUT if f0[2] == f1[2] else O.CORRECTED)
    if cls == "BB":
        if f0[2] == f1[2]:
            return O.CORRECTED, O.CORRECTED
        return O.UNCORRECTABLE, (O.UNCORRECTABLE_INPUT if f0[1] == f1[1] else O.CORRECTED)
    if cls == "AB":
        return O.UNCORRECTABLE, O.CORRECTED                  # min(s,t) >= 3
    raise AssertionError(cls)


@pytest.mark.parametrize("shape", [(4, 3, 4), (5, 4, 6), (3, 4, 3), (6, 3, 5)])
def test_brute_force_every_placement_of_one_and_two_faults(shape):
    """Theorem 1 / Theorem 2 by exhaustion: every single site and every pair of sites of A, B, C.
    Corrected C must equal the fault-free product, located set must equal the injected set, A and B restored."""
    n, k, m = shape
    rng, A, B, Abar, Bbar, Cc, tau, tin = _setup(n, k, m, 11)
    sites = _sites(n, k, m)
    combos = list(itertools.combinations(sites, 1)) + list(itertools.combinations(sites, 2))
    for combo in combos:
        faults = [(kd, r, c, float(rng.uniform(1, 100) * rng.choice([-1.0, 1.0]))) for kd, r, c in combo]
        Af, Bf = O.inject_input_faults(Abar, Bbar, faults)
        Cb = O.fault_effects(Cc, Abar, Bbar, faults)
        exp_p, exp_x = _expected(faults)
        rp = O.decode_level_p(Cb, tau)
        rx = O.decode_level_x(Cb, Af, Bf, tau, tin)
        assert rp.verdict == exp_p, (faults, rp)
        assert rx.verdict == exp_x, (faults, rx)
        if rp.verdict == O.CORRECTED:
            assert np.max(np.abs(rp.C - Cc[:n, :m])) < 1e-6, faults
        else:
            np.testing.assert_array_equal(rp.C, Cb[:n, :m])        # never patch without a verdict
        if rx.verdict == O.CORRECTED:
            assert np.max(np.abs(rx.C - Cc[:n, :m])) < 1e-6, faults
            assert np.max(np.abs(rx.A - A)) < 1e-9 and np.max(np.abs(rx.B - B)) < 1e-9
            assert rx.located() == sorted((f[0], f[1], f[2]) for f in faults), faults
            for (kd, r, c, mag), f in zip(rx.found, sorted(faults)):
                assert mag == pytest.approx(f[3], rel=1e-6)
        # Level-P locates rows / columns / points
        if rp.verdict == O.CORRECTED:
            want = set()
            for kd, r, c, _ in faults:
                want.add((O.KIND_ROW, r, -1) if kd == O.KIND_A else (O.KIND_COL, -1, c) if kd == O.KIND_B else (O.KIND_C, r, c))
            assert set(rp.located()) == want, (faults, rp.found)


@pytest.mark.parametrize("transpose", [False, True])
def test_theorem2_many_errors_confined_to_one_or_two_lines(transpose):
    """Theorem 2 beyond the two-error budget: E(s,t) with min(s,t) <= 2 is corrected whatever t is --
    s = 1 "for any t* in E_t" by PAPER.md:223, s = 2 by the 2x2 solve of PAPER.md:227-231.  Ground truth of the
    injection is the reference: the corrected C equals the fault-free product; up to four located symbols per line are
    listed one by one, more are reported as a whole-line fault."""
    n, k, m = 9, 4, 11
    rng, A, B, Abar, Bbar, Cc, tau, tin = _setup(n, k, m, 21)
    if transpose:                                   # the same patterns confined to COLUMNS of C
        rng, A, B, Abar, Bbar, Cc, tau, tin = _setup(m, k, n, 21)
    nn, mm = (m, n) if transpose else (n, m)

    def run(cells):
        faults = [(O.KIND_C, (c if transpose else r), (r if transpose else c), float(rng.uniform(1, 100) * rng.choice([-1.0, 1.0]))) for r, c in cells]
        Cb = O.inject_output_faults(Cc, faults)
        rep = O.decode_level_p(Cb, tau)
        assert rep.verdict == O.CORRECTED, (cells, rep)
        assert np.max(np.abs(rep.C - Cc[:nn, :mm])) < 1e-6, cells
        repx = O.decode_level_x(Cb, Abar, Bbar, tau, tin)          # operands intact: Level X keeps the Level-P result
        assert repx.verdict == O.CORRECTED and np.max(np.abs(repx.C - Cc[:nn, :mm])) < 1e-6
        return faults, rep

    # E(1,3), E(1,4): listed as points
    for cells in ([(5, 1), (5, 4), (5, 9)], [(0, 0), (0, 3), (0, 7), (0, 10)]):
        faults, rep = run(cells)
        assert rep.located() == sorted((2, f[1], f[2]) for f in faults)
        for (kd, r, c, mag), f in zip(rep.found, sorted(faults)):
            assert mag == pytest.approx(f[3], rel=1e-6)
    # E(1,5) and E(1, every column): too many to list -> whole line, corrected along it
    for cells in ([(5, j) for j in (0, 2, 3, 6, 10)], [(8, j) for j in range(11)]):
        faults, rep = run(cells)
        line = cells[0][0]
        assert rep.located() == ([(O.KIND_COL, -1, line)] if transpose else [(O.KIND_ROW, line, -1)])
    # E(2,3) with errors on both lines in every flagged column, E(2,4) mixed
    for cells in ([(2, 1), (2, 4), (2, 9), (6, 1), (6, 4), (6, 9)], [(1, 0), (1, 5), (1, 6), (4, 5), (4, 8)]):
        faults, rep = run(cells)
        assert rep.located() == sorted((2, f[1], f[2]) for f in faults)
    # E(2,6): one line with six, one with two
    faults, rep = run([(3, j) for j in (0, 1, 4, 6, 7, 10)] + [(7, 4), (7, 9)])
    want = [(O.KIND_COL, -1, 3)] if transpose else [(O.KIND_ROW, 3, -1)]
    want += sorted((2, f[1], f[2]) for f in faults if (f[2] if transpose else f[1]) == 7)
    assert rep.located() == sorted(want)


def test_single_error_formula_as_printed():
    """c_true = c - (sum_i c_{i,t*} - c_{n+1,t*}).  Evaluate the printed right-hand side by hand."""
    n, k, m = 6, 4, 5
    rng, A, B, Abar, Bbar, Cc, tau, _ = _setup(n, k, m, 12)
    Cb = O.inject_output_faults(Cc, [(O.KIND_C, 3, 2, -42.0)])
    printed = Cb[3, 2] - (sum(Cb[i, 2] for i in range(n)) - Cb[n, 2])
    rep = O.decode_level_p(Cb, tau)
    assert rep.verdict == O.CORRECTED and rep.located() == [(O.KIND_C, 3, 2)]
    assert rep.C[3, 2] == pytest.approx(printed, abs=1e-10) == pytest.approx((A @ B)[3, 2], abs=1e-10)


def test_two_row_solve_sign_reading_R8():
    """with the right-hand side as PRINTED (parity minus sum) and the printed subtraction, the
    error doubles; with sum-minus-parity it cancels.  The oracle must land on the clean product."""
    n, k, m = 6, 4, 5
    rng, A, B, Abar, Bbar, Cc, tau, _ = _setup(n, k, m, 13)
    faults = [(O.KIND_C, 1, 2, 10.0), (O.KIND_C, 4, 2, -3.0)]       # same column, two rows: s = 2, t = 1
    Cb = O.inject_output_faults(Cc, faults)
    s1, s2 = 2, 5                                                    # 1-based rows
    M = np.array([[1.0, 1.0], [s1, s2]])
    col = Cb[:n, 2]
    rhs_printed = np.array([Cb[n, 2] - col.sum(), Cb[n + 1, 2] - np.arange(1, n + 1) @ col])
    e_printed = np.linalg.solve(M, rhs_printed)
    assert abs((Cb[1, 2] - e_printed[0]) - Cc[1, 2]) == pytest.approx(20.0, abs=1e-9)      # doubled
    e_fixed = np.linalg.solve(M, -rhs_printed)
    assert abs((Cb[1, 2] - e_fixed[0]) - Cc[1, 2]) < 1e-9
    rep = O.decode_level_p(Cb, tau)
    assert rep.verdict == O.CORRECTED and rep.located() == [(2, 1, 2), (2, 4, 2)]
    np.testing.assert_allclose(rep.C, Cc[:n, :m], atol=1e-9)


def _golden_patterns():
    pats = {"e1": [], "e2": []}
    with open(os.path.join(GOLDEN, "counterexample_e1_e2.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, r, c, v = line.split()
            pats[name].append((int(r), int(c), float(v)))
    return pats


def test_counterexample_e1_e2_from_the_paper():
    """e_1 and e_2 "yield identical local row checksum and column parity symbols".
    As printed e_2's weighted column syndromes are twice e_1's (erratum, DESIGN.md App. A#7); e_2/2 coincides.
    Either way the decoder must refuse (E(2,3) with silent row checks), never miscorrect."""
    n, k, m = 6, 3, 6
    rng, A, B, Abar, Bbar, Cc, tau, _ = _setup(n, k, m, 14)
    pats = _golden_patterns()

    def syn(pattern, scale):
        E = np.zeros_like(Cc)
        for r, c, v in pattern:
            E[r - 1, c - 1] = v * scale
        return [np.round(s, 8) for s in O.syndromes(Cc + E)], Cc + E

    s_e1, C1 = syn(pats["e1"], 1.0)
    s_e2, _ = syn(pats["e2"], 1.0)
    s_e2h, C2h = syn(pats["e2"], 0.5)
    # row checks and plain column checks silent for both (each row sums to 0 with weights (1,-2,1)·(1,2,3) = 0)
    for s in (s_e1, s_e2, s_e2h):
        assert np.all(s[0] == 0) and np.all(s[1] == 0) and np.all(s[2] == 0)
    np.testing.assert_array_equal(s_e1[3], [-1, 2, -1, 0, 0, 0])
    np.testing.assert_array_equal(s_e2[3], [-2, 4, -2, 0, 0, 0])     # as printed: NOT identical
    np.testing.assert_array_equal(s_e2h[3], s_e1[3])                 # erratum: e_2 / 2 is
    for Cb in (C1, C2h):
        rep = O.decode_level_p(Cb, tau)
        assert rep.verdict == O.UNCORRECTABLE
        np.testing.assert_array_equal(rep.C, Cb[:n, :m])


@pytest.mark.parametrize("rows,cols", [((1, 2, 3), (1, 2, 3)), ((2, 5, 7), (1, 4, 6)), ((1, 3, 7), (3, 5, 6))])
def test_lemma3_rank_of_3x3_constraint_system_is_8(rows, cols):
    """Lemma 3: the 16 constraints touching a 3x3 support (6 row-parity, 6 column-parity,
    4 global) have rank 8 < 9.  Built from the constraint definitions (Def. 1), not from the decoder."""
    rowsys = []
    for a, s in enumerate(rows):                                  # row s: sum_j e_sj = 0, sum_j t_j e_sj = 0
        for w in (lambda t: 1.0, lambda t: float(t)):
            v = np.zeros((3, 3)); v[a, :] = [w(t) for t in cols]; rowsys.append(v.ravel())
    for b, t in enumerate(cols):
        for w in (lambda s: 1.0, lambda s: float(s)):
            v = np.zeros((3, 3)); v[:, b] = [w(s) for s in rows]; rowsys.append(v.ravel())
    for wr in (lambda s: 1.0, lambda s: float(s)):                # global parity: [1;w_n] E [1,w_m]
        for wc in (lambda t: 1.0, lambda t: float(t)):
            rowsys.append(np.array([[wr(s) * wc(t) for t in cols] for s in rows]).ravel())
    M = np.array(rowsys)
    assert M.shape == (16, 9)
    assert np.linalg.matrix_rank(M) == 8


def test_huang_abraham_special_case():
    """With only the plain checks (P_n1, P_m1) the scheme is the textbook single-checksum ABFT of ref [8]
    (PAPER.md:258): one C error sits at the intersection of the one bad row and the one bad column and equals
    either plain syndrome.  The oracle's answer must coincide with that textbook rule."""
    n, k, m = 9, 5, 8
    rng, A, B, Abar, Bbar, Cc, tau, _ = _setup(n, k, m, 15)
    for _ in range(20):
        i, j, e = int(rng.integers(n)), int(rng.integers(m)), float(rng.uniform(1, 100))
        Cb = O.inject_output_faults(Cc, [(O.KIND_C, i, j, e)])
        C = Cb[:n, :m]
        row_bad = np.nonzero(np.abs(C.sum(1) - Cb[:n, m]) > 1e-6)[0]
        col_bad = np.nonzero(np.abs(C.sum(0) - Cb[n, :m]) > 1e-6)[0]
        assert list(row_bad) == [i] and list(col_bad) == [j]
        rep = O.decode_level_p(Cb, tau)
        assert rep.located() == [(O.KIND_C, i, j)]
        assert rep.found[0][3] == pytest.approx(C[:, j].sum() - Cb[n, j], abs=1e-9)


def test_faults_in_parity_symbols_never_cause_a_wrong_patch():
    """Reading R11: the fault model names only symbols of A, B, C; a corrupted parity symbol must
    yield CLEAN (global parity is never read by the row/column checks) or UNCORRECTABLE, with C untouched."""
    n, k, m = 5, 4, 6
    rng, A, B, Abar, Bbar, Cc, tau, tin = _setup(n, k, m, 16)
    for r, c in [(n, l) for l in range(k)] + [(n + 1, l) for l in range(k)]:
        Af = Abar.copy(); Af[r, c] += 9.0
        rep = O.decode_level_x(O.encoded_product(Af, Bbar), Af, Bbar, tau, tin)
        assert rep.verdict in (O.UNCORRECTABLE, O.UNCORRECTABLE_INPUT)
    for r in range(n + 2):
        for c in range(m + 2):
            if r < n and c < m:
                continue
            Cb = Cc.copy(); Cb[r, c] += 9.0
            rep = O.decode_level_p(Cb, tau)
            if r >= n and c >= m:
                assert rep.verdict == O.CLEAN
            else:
                assert rep.verdict == O.UNCORRECTABLE
            np.testing.assert_array_equal(rep.C, Cc[:n, :m])


def _table1_rates():
    out = {}
    with open(os.path.join(GOLDEN, "table1_rates.txt")) as f:
        for line in f:
            if not line.startswith("#") and line.strip():
                a, b = line.split(); out[a] = float(b)
    return out


def test_table1_scenarios_at_paper_shape():
    """Table I: 100 % correction for scenarios a-f at M(n=1024, k=4096, m=1024)."""
    from paper_2508_04355_b200 import inputs as I
    n, k, m = 1024, 4096, 1024
    A, B = I.make_operands(n, k, m, seed=0, dist="uniform")
    Abar, Bbar = O.encoded_operands(A, B)
    Cc = O.encoded_product(Abar, Bbar)
    tau, tin = O.fp64_thresholds(n, m, Cc), O.fp64_input_thresholds(Abar, Bbar)
    for scen, want in _table1_rates().items():
        ok = 0
        trials = 6
        for t in range(trials):
            faults = I.draw_faults(n, k, m, I.SCENARIOS[scen], seed=1000 * ord(scen) + t)
            Af, Bf = O.inject_input_faults(Abar, Bbar, faults)
            rep = O.decode_level_x(O.fault_effects(Cc, Abar, Bbar, faults), Af, Bf, tau, tin)
            good = (rep.verdict == O.CORRECTED and rep.located() == sorted((f[0], f[1], f[2]) for f in faults)
                    and np.max(np.abs(rep.C - Cc[:n, :m])) < 1e-6)
            ok += good
        assert 100.0 * ok / trials == want, scen


# ---------------------------------------------------------------- global parity, single checksum, recompute ----
def test_global_parity_identities_and_parity_symbol_faults():
    """Eq. (4), PAPER.md:151-158 / 131-135: P_g = [1; w_n] C [1, w_m], so the parity columns P_r and the parity rows P_c are
    themselves checked by the four global symbols.  A fault in one local parity symbol of C_bar is classified by them
    (kind, position, magnitude), C is left untouched; without the global checks the same fault is only refused."""
    n, k, m = 7, 4, 9
    rng, A, B, Abar, Bbar, Cc, tau, tin = _setup(n, k, m, 31)
    C = A @ B
    wn, wm = np.arange(1, n + 1.0), np.arange(1, m + 1.0)
    g_r, g_c = O.global_checks(Cc)
    assert np.abs(g_r).max() < 1e-9 and np.abs(g_c).max() < 1e-9
    np.testing.assert_allclose(Cc[n:, m:], [[C.sum(), (C @ wm).sum()], [wn @ C.sum(1), wn @ C @ wm]], atol=1e-9)
    tau_g = (1e-7, 1e-6)
    for c in range(2):
        for i in range(n):
            Cb = Cc.copy(); Cb[i, m + c] += 5.5
            assert O.decode_level_p(Cb, tau).verdict == O.UNCORRECTABLE
            rep = O.decode_level_p(Cb, tau, tau_g)
            assert rep.verdict == O.CORRECTED and rep.located() == [(O.KIND_PR, i, c)], (i, c, rep)
            assert rep.found[0][3] == pytest.approx(5.5, abs=1e-9)
            np.testing.assert_array_equal(rep.C, Cc[:n, :m])
            assert O.decode_level_x(Cb, Abar, Bbar, tau, tin, tau_g).located() == [(O.KIND_PR, i, c)]
        for j in range(m):
            Cb = Cc.copy(); Cb[n + c, j] -= 3.25
            rep = O.decode_level_p(Cb, tau, tau_g)
            assert rep.verdict == O.CORRECTED and rep.located() == [(O.KIND_PC, c, j)], (c, j, rep)
            assert rep.found[0][3] == pytest.approx(-3.25, abs=1e-9)
    # a symbol of C moves BOTH of its line's checks and a column's too: never taken for a parity fault
    Cb = O.inject_output_faults(Cc, [(O.KIND_C, 2, 3, 4.0)])
    assert O.decode_level_p(Cb, tau, tau_g).located() == [(O.KIND_C, 2, 3)]
    # a parity symbol off in a codeword whose global symbol does not confirm it (here: the global symbol is off too): refused
    Cb = Cc.copy(); Cb[1, m] += 5.5; Cb[n, m] += 2.0
    assert O.decode_level_p(Cb, tau, tau_g).verdict == O.UNCORRECTABLE


def test_single_checksum_mode_capability():
    """With P_n1 / P_m1 alone (ref [8], the scheme behind Table I's "Checksum" columns): every single
    error in C is located and corrected (scenario c); two errors (d, e, f: the "-" entries) and input faults seen through
    C_bar alone are detected and refused, never miscorrected."""
    n, k, m = 5, 3, 6
    rng, A, B, Abar, Bbar, Cc, tau, tin = _setup(n, k, m, 32)
    for i in range(n):
        for j in range(m):
            Cb = O.inject_output_faults(Cc, [(O.KIND_C, i, j, 17.0)])
            rep = O.decode_single_checksum(Cb, tau)
            assert rep.verdict == O.CORRECTED and rep.located() == [(O.KIND_C, i, j)]
            assert np.abs(rep.C - Cc[:n, :m]).max() < 1e-9
    assert O.decode_single_checksum(Cc, tau).verdict == O.CLEAN
    sites = _sites(n, k, m)
    for combo in itertools.combinations(sites, 2):
        faults = [(kd, r, c, float(rng.uniform(1, 100))) for kd, r, c in combo]
        rep = O.decode_single_checksum(O.fault_effects(Cc, Abar, Bbar, faults), tau)
        assert rep.verdict == O.UNCORRECTABLE, faults
        np.testing.assert_array_equal(rep.C, O.fault_effects(Cc, Abar, Bbar, faults)[:n, :m])
    for kd, r, c in sites:
        if kd != O.KIND_C:
            rep = O.decode_single_checksum(O.fault_effects(Cc, Abar, Bbar, [(kd, r, c, 9.0)]), tau)
            assert rep.verdict == O.UNCORRECTABLE


def test_recompute_fallback_restores_what_the_code_cannot():
    """min(s,t) >= 3 "needs to be recalculated".  Lemma-3 supports (3 x 3 errors), the e_1 pattern of
    PAPER.md:170 and a non-finite symbol: the fallback recomputes the flagged lines and the result is the fault-free
    product.  Operands that are themselves corrupted beyond repair stay refused."""
    n, k, m = 8, 5, 9
    rng, A, B, Abar, Bbar, Cc, tau, tin = _setup(n, k, m, 33)
    pats = [[(O.KIND_C, i, j, float(rng.uniform(1, 50))) for i in (1, 4, 6) for j in (0, 3, 8)],
            [(O.KIND_C, 0, 0, 1.0), (O.KIND_C, 0, 1, -2.0), (O.KIND_C, 0, 2, 1.0), (O.KIND_C, 1, 0, -1.0), (O.KIND_C, 1, 1, 2.0), (O.KIND_C, 1, 2, -1.0)],
            [(O.KIND_C, 2, 5, float("nan"))],
            [(O.KIND_C, i, i, 3.0) for i in range(5)]]
    for faults in pats:
        Cb = O.inject_output_faults(Cc, faults)
        assert O.decode_level_p(Cb, tau).verdict == O.UNCORRECTABLE
        rep = O.recompute_fallback(Cb, Abar, Bbar, tau)
        assert rep.verdict == O.CORRECTED_BY_RECOMPUTE, faults
        assert np.abs(rep.C - Cc[:n, :m]).max() < 1e-9
    # two faults in one column of A (UNCORRECTABLE_INPUT): recomputing from the corrupted operand reproduces the error
    faults = [(O.KIND_A, 1, 2, 7.0), (O.KIND_A, 5, 2, -4.0)]
    Af, Bf = O.inject_input_faults(Abar, Bbar, faults)
    Cb = O.fault_effects(Cc, Abar, Bbar, faults)
    assert O.decode_level_x(Cb, Af, Bf, tau, tin).verdict == O.UNCORRECTABLE_INPUT
    assert O.recompute_fallback(Cb, Af, Bf, tau).verdict == O.UNCORRECTABLE
    assert O.recompute_fallback(Cc, Abar, Bbar, tau).verdict == O.CLEAN


def test_tile_local_grid_corrects_two_errors_per_block():
    """SURVEY 8(f)-1, a variant of Def. 1: one code per panel of P rows x Q columns with weights local
    to the panel.  Four errors on distinct rows and columns defeat the global code (min(s,t) >= 3) but fall
    into different blocks, two at most per block, and are corrected; the per-panel parity obeys the block identities
     with local weights; three errors on distinct lines INSIDE one block are still refused."""
    n, k, m, P, Q = 12, 5, 10, 4, 5
    rng, A, B, Abar, Bbar, Cc, tau, tin = _setup(n, k, m, 41)
    C = A @ B
    AP, BP = O.encode_panels(A, B, P, Q)
    assert len(AP) == 3 and len(BP) == 2
    for bi, (r0, r1) in enumerate(O.panel_ranges(n, P)):
        np.testing.assert_allclose(AP[bi][0], A[r0:r1].sum(0), atol=1e-12)
        np.testing.assert_allclose(AP[bi][1], np.arange(1, r1 - r0 + 1.0) @ A[r0:r1], atol=1e-12)      # weights restart at 1
        for bj, (c0, c1) in enumerate(O.panel_ranges(m, Q)):
            np.testing.assert_allclose(AP[bi] @ B[:, c0:c1], np.vstack([C[r0:r1, c0:c1].sum(0), np.arange(1, r1 - r0 + 1.0) @ C[r0:r1, c0:c1]]), atol=1e-10)
            np.testing.assert_allclose(A[r0:r1] @ BP[bj], np.column_stack([C[r0:r1, c0:c1].sum(1), C[r0:r1, c0:c1] @ np.arange(1, c1 - c0 + 1.0)]), atol=1e-10)
    tau_of = lambda rows, cols: (1e-8, 1e-8 * cols, 1e-8, 1e-8 * rows)
    faults = [(O.KIND_C, 0, 1, 5.0), (O.KIND_C, 5, 3, -7.0), (O.KIND_C, 6, 8, 11.0), (O.KIND_C, 11, 6, 2.5), (O.KIND_C, 3, 9, -4.0), (O.KIND_C, 2, 7, 6.0)]
    Cb = O.inject_output_faults(Cc, faults)
    assert O.decode_level_p(Cb, tau).verdict == O.UNCORRECTABLE            # the paper's global code: six rows, six columns
    rep = O.decode_panels(Cb[:n, :m], A, B, P, Q, tau_of)
    assert rep.verdict == O.CORRECTED and rep.located() == sorted((f[0], f[1], f[2]) for f in faults)
    assert np.abs(rep.C - C).max() < 1e-9
    # three errors on distinct rows and columns inside ONE block: that block is refused, the others are still served
    faults = [(O.KIND_C, 0, 0, 5.0), (O.KIND_C, 1, 2, -7.0), (O.KIND_C, 3, 4, 11.0), (O.KIND_C, 9, 8, 2.0)]
    rep = O.decode_panels(O.inject_output_faults(Cc, faults)[:n, :m], A, B, P, Q, tau_of)
    assert rep.verdict == O.UNCORRECTABLE and rep.located() == [(O.KIND_C, 9, 8)]
    assert O.decode_panels(C, A, B, P, Q, tau_of).verdict == O.CLEAN


def test_tile_local_grid_input_fault_after_encoding():
    """decode_panels(parity=...): an input fault strikes after the panels were encoded (reading R1).  A fault in
    a_il corrupts row i of C in every column panel; P_r of those blocks shifts with it (own-side syndromes silent, R7), the
    column syndromes of each block locate row i by the weighted ratio with LOCAL weights and each block restores its piece
    of the row (R6).  A fault before encoding is a valid codeword of the wrong product in every block (R1)."""
    n, k, m, P, Q = 12, 5, 10, 4, 5
    rng, A, B, Abar, Bbar, Cc, tau, tin = _setup(n, k, m, 43)
    C = A @ B
    tau_of = lambda rows, cols: (1e-8, 1e-8 * cols, 1e-8, 1e-8 * rows)
    par = O.encode_panels(A, B, P, Q)
    Af = A.copy()
    Af[6, 2] += 3.0                                                   # row 6 = local row 2 of panel 1
    rep = O.decode_panels(Af @ B, Af, B, P, Q, tau_of, parity=par)
    assert rep.verdict == O.CORRECTED and rep.located() == [(O.KIND_ROW, 6, -1)] * 2      # once per column panel
    assert np.abs(rep.C - C).max() < 1e-9
    assert rep.n_row_flags == 0 and rep.n_col_flags == m
    Bf = B.copy()
    Bf[1, 7] -= 2.0                                                   # column 7 = local column 2 of panel 1
    rep = O.decode_panels(A @ Bf, A, Bf, P, Q, tau_of, parity=par)
    assert rep.verdict == O.CORRECTED and rep.located() == [(O.KIND_COL, -1, 7)] * 3
    assert np.abs(rep.C - C).max() < 1e-9
    assert O.decode_panels(Af @ B, Af, B, P, Q, tau_of).verdict == O.CLEAN                # encoded from the faulty operand


def test_tile_local_grid_ragged_panels_and_unequal_panel_sizes():
    """Panels that do not divide n, m (short last panels with their own weights 1..len) and P != Q: the last row of a short
    panel carries weight len, not P; an error there is located by the ratio of the block's two column syndromes; every block
    of a fault-free product is a codeword of its own code (all syndromes vanish); thresholds are asked per block shape."""
    n, k, m, P, Q = 11, 4, 13, 4, 5            # row panels 4, 4, 3; column panels 5, 5, 3
    rng, A, B, Abar, Bbar, Cc, tau, tin = _setup(n, k, m, 47)
    C = A @ B
    AP, BP = O.encode_panels(A, B, P, Q)
    assert [a.shape for a in AP] == [(2, k)] * 3 and [b.shape for b in BP] == [(k, 2)] * 3
    np.testing.assert_allclose(AP[2][1], np.array([1.0, 2.0, 3.0]) @ A[8:11], atol=1e-12)          # weights restart at 1 in the short panel
    np.testing.assert_allclose(BP[2][:, 1], B[:, 10:13] @ np.array([1.0, 2.0, 3.0]), atol=1e-12)
    asked = []

    def tau_of(rows, cols):
        asked.append((rows, cols))
        return (1e-8, 1e-8 * cols, 1e-8, 1e-8 * rows)

    assert O.decode_panels(C, A, B, P, Q, tau_of).verdict == O.CLEAN
    assert sorted(set(asked)) == [(3, 3), (3, 5), (4, 3), (4, 5)]
    faults = [(O.KIND_C, 10, 12, 4.0), (O.KIND_C, 8, 10, -3.0), (O.KIND_C, 3, 4, 2.0)]         # the corner block (3 x 3) twice, block (0, 0) once
    rep = O.decode_panels(O.inject_output_faults(Cc, faults)[:n, :m], A, B, P, Q, tau_of)
    assert rep.verdict == O.CORRECTED and rep.located() == sorted((f[0], f[1], f[2]) for f in faults)
    assert np.abs(rep.C - C).max() < 1e-9
    assert rep.n_row_flags == 3 and rep.n_col_flags == 3
