"""CPU fp64 ORACLE for the grid-like error-correcting code for matrix multiplication (arxiv 2508.04355).

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import it.  It shares no code with the CUDA path
(paper_2508_04355_b200/csrc) and imports nothing from the package.  Plain numpy, fp64 throughout,
written in the paper's order and notation so it can be checked against PAPER.md by eye.

Citations are PAPER.md line numbers (+ section / equation).  Indices in the paper are 1-based;
here arrays are 0-based and the weight of 0-based index r is r + 1 (PAPER.md:83 P_n2 = (1..n),
PAPER.md:101 P_m2 = (1..m)).

Functions and what pins them (tests/test_oracle_*.py, `-m "not gpu"`):
  encode_left / encode_right      PAPER.md:71-113   pinned by block identities P_r = C[1,w] etc.
  encoded_product                 PAPER.md:115-117  pinned by a pure-python triple loop and the block identities
  syndromes                       PAPER.md:194-200  pinned: exactly ~0 on fault-free data; signatures of App. B of DESIGN.md
  decode_level_p (paper decoder)  PAPER.md:186-233  pinned by brute force over every 1- and 2-fault placement (Thm 1/2,
                                                    PAPER.md:166,176), the e_1 / e_2 counter-example,
                                                    the s=1 formula and the Huang-Abraham special case
  decode_level_x (input check)    DESIGN.md R9      pinned by brute force: A, B and C restored for every <=2-fault placement
  parity_symbol_fault             PAPER.md:151-158  Eq. (4), the global parity: pinned by injecting into every parity symbol of C_bar
                                                    (classified, C untouched, symbol restored) and by the identities of P_g
  decode_single_checksum          PAPER.md:202-213  the "Checksum" columns' capability with P_n1 / P_m1 only (ref [8]): pinned by the
                                                    textbook rule and by exhaustion (every C error corrected, every pair refused)
  encode_panels / decode_panels   PAPER.md:139-158  tile-local variant of Def. 1 (one code per panel pair): pinned by patterns the global code
                                                    refuses and the panel codes correct, and by the block identities per panel
  recompute_fallback              PAPER.md:19, 219  "needs to be recalculated": pinned against the fault-free product on patterns the
                                                    code cannot correct (Lemma 3 supports, non-finite symbols)
  flag_sets                       PAPER.md:215-217  pinned with syndromes (signatures) and by every decoder pin; thresholds are INPUTS:
                                                    the paper gives one delta with unstated dtype / scale, so
                                                    the oracle defines none.  The library's automatic thresholds are stated in
                                                    include/gecc.h and restated / pinned in tests/threshold_spec.py.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

# verdicts
CLEAN, CORRECTED, UNCORRECTABLE, UNCORRECTABLE_INPUT, CORRECTED_BY_RECOMPUTE = 0, 1, 2, 3, 4
# kinds of located faults.  KIND_PR / KIND_PC: a parity symbol of C_bar itself (row i, check c) / (check c, column j)
KIND_A, KIND_B, KIND_C, KIND_ROW, KIND_COL, KIND_PR, KIND_PC = 0, 1, 2, 3, 4, 5, 6


# ----------------------------------------------------------------------------------------------
# O1  Encoder  (section III)
# ----------------------------------------------------------------------------------------------
def encode_left(A: np.ndarray) -> np.ndarray:
    """A_P (2 x k): row 0 = P_n1 a_{*l} = sum_i a_{i,l}; row 1 = P_n2 a_{*l} = sum_i i a_{i,l}."""
    A = np.asarray(A, dtype=np.float64)
    n, k = A.shape
    A_P = np.zeros((2, k), dtype=np.float64)
    for i in range(n):                      # sequential fp64 sums over the rows of A
        A_P[0, :] += A[i, :]
        A_P[1, :] += (i + 1) * A[i, :]
    return A_P


def encode_right(B: np.ndarray) -> np.ndarray:
    """B_P (k x 2): column 0 = P_m1 b_{l*}^T = sum_j b_{l,j}; column 1 = sum_j j b_{l,j}."""
    B = np.asarray(B, dtype=np.float64)
    k, m = B.shape
    B_P = np.zeros((k, 2), dtype=np.float64)
    for j in range(m):
        B_P[:, 0] += B[:, j]
        B_P[:, 1] += (j + 1) * B[:, j]
    return B_P


def encoded_operands(A: np.ndarray, B: np.ndarray):
    """A_bar = G_A A = [A; A_P] ((n+2) x k), B_bar = B G_B = [B, B_P] (k x (m+2))."""
    A = np.asarray(A, dtype=np.float64)
    B = np.asarray(B, dtype=np.float64)
    return np.vstack([A, encode_left(A)]), np.hstack([B, encode_right(B)])


# ----------------------------------------------------------------------------------------------
# O2 / O3'  Fault injection (PAPER.md:39-45 E1/E2/E3; reading R1: input faults strike the data part
# of A_bar / B_bar AFTER the parity was generated from clean data)
# ----------------------------------------------------------------------------------------------
def inject_input_faults(Abar: np.ndarray, Bbar: np.ndarray, faults):
    """Add e to A_bar[i,l] (kind 0) / B_bar[l,j] (kind 1), data parts only.  Returns copies."""
    Abar = Abar.copy()
    Bbar = Bbar.copy()
    n, m = Abar.shape[0] - 2, Bbar.shape[1] - 2
    for kind, r, c, e in faults:
        if kind == KIND_A:
            assert 0 <= r < n
            Abar[r, c] += e
        elif kind == KIND_B:
            assert 0 <= c < m
            Bbar[r, c] += e
    return Abar, Bbar


def inject_output_faults(Cbar: np.ndarray, faults) -> np.ndarray:
    """Add e to C_bar[i,j], i < n, j < m (kind 2: an error during the computation of a symbol of C)."""
    Cbar = Cbar.copy()
    n, m = Cbar.shape[0] - 2, Cbar.shape[1] - 2
    for kind, r, c, e in faults:
        if kind == KIND_C:
            assert 0 <= r < n and 0 <= c < m
            Cbar[r, c] += e
    return Cbar


# ----------------------------------------------------------------------------------------------
# O3  Encoded product
# ----------------------------------------------------------------------------------------------
def encoded_product(Abar: np.ndarray, Bbar: np.ndarray) -> np.ndarray:
    """C_bar = A_bar B_bar = [[C, P_r], [P_c, P_g]].  fp64 matmul is the library step."""
    return np.matmul(np.asarray(Abar, dtype=np.float64), np.asarray(Bbar, dtype=np.float64))


def encoded_product_loops(Abar, Bbar) -> np.ndarray:
    """The same product as the plain definition c_{i,j} = sum_l a_{i,l} b_{l,j}; tiny sizes only."""
    rows, k = len(Abar), len(Abar[0])
    cols = len(Bbar[0])
    out = np.zeros((rows, cols), dtype=np.float64)
    for i in range(rows):
        for j in range(cols):
            acc = 0.0
            for l in range(k):
                acc += float(Abar[i][l]) * float(Bbar[l][j])
            out[i, j] = acc
    return out


def fault_effects(Cbar_clean: np.ndarray, Abar: np.ndarray, Bbar: np.ndarray, faults) -> np.ndarray:
    """Linearity shortcut for many-trial configs: the exact effect of a fault list on a clean C_bar.

    (A_bar + E_A)(B_bar + E_B) + E_C = A_bar B_bar + E_A B_bar + A_bar E_B + E_A E_B + E_C:
    an A fault (i,l,e) adds e * B_bar[l,:] to row i (all m+2 entries), a B fault (l,j,e) adds
    e * A_bar[:,l] to column j, an A and a B fault sharing l add e1 e2 at (i,j), a C fault adds e.
    Abar / Bbar are the CLEAN encoded operands.  Cross-checked against full recomputation in the tests.
    """
    C = Cbar_clean.copy()
    fa = [(r, c, e) for kind, r, c, e in faults if kind == KIND_A]
    fb = [(r, c, e) for kind, r, c, e in faults if kind == KIND_B]
    for i, l, e in fa:
        C[i, :] += e * Bbar[l, :]
    for l, j, e in fb:
        C[:, j] += e * Abar[:, l]
    for i, l1, e1 in fa:
        for l2, j, e2 in fb:
            if l1 == l2:
                C[i, j] += e1 * e2
    return inject_output_faults(C, faults)


# ----------------------------------------------------------------------------------------------
# O4  Syndromes (sign convention "sum minus parity")
# ----------------------------------------------------------------------------------------------
def syndromes(Cbar: np.ndarray):
    """r1_i = sum_j c_ij - c_{i,m+1};  r2_i = sum_j j c_ij - c_{i,m+2}   (i in [n])
       q1_j = sum_i c_ij - c_{n+1,j};  q2_j = sum_i i c_ij - c_{n+2,j}   (j in [m])
    (reading R3: the weighted checks compare with the SECOND parity symbol, as 196/200 print; 217 is a typo)."""
    Cbar = np.asarray(Cbar, dtype=np.float64)
    n, m = Cbar.shape[0] - 2, Cbar.shape[1] - 2
    r1 = np.zeros(n)
    r2 = np.zeros(n)
    q1 = np.zeros(m)
    q2 = np.zeros(m)
    for j in range(m):
        r1 += Cbar[:n, j]
        r2 += (j + 1) * Cbar[:n, j]
    r1 -= Cbar[:n, m]
    r2 -= Cbar[:n, m + 1]
    for i in range(n):
        q1 += Cbar[i, :m]
        q2 += (i + 1) * Cbar[i, :m]
    q1 -= Cbar[n, :m]
    q2 -= Cbar[n + 1, :m]
    return r1, r2, q1, q2


# ----------------------------------------------------------------------------------------------
# O5  Flags (a row / column is flagged if EITHER of its two checks exceeds delta;
# reading R4: four thresholds instead of one delta; non-finite syndromes count as flagged)
# ----------------------------------------------------------------------------------------------
def flag_sets(r1, r2, q1, q2, tau):
    t_r1, t_r2, t_q1, t_q2 = tau
    R = [i for i in range(len(r1)) if not (abs(r1[i]) <= t_r1) or not (abs(r2[i]) <= t_r2)]
    Q = [j for j in range(len(q1)) if not (abs(q1[j]) <= t_q1) or not (abs(q2[j]) <= t_q2)]
    return R, Q


def fp64_thresholds(n, m, Cbar_clean, rel=1e-9):
    """Thresholds for EXACT-ARITHMETIC use of the oracle (brute force, ground truth): fp64 rounding noise only.
    tau_plain = rel * max(1, max|C|) over the DATA part (the global parity block is orders of magnitude larger and
    is never read by the row / column checks); the weighted checks are scaled by the largest weight."""
    s = rel * max(1.0, float(np.max(np.abs(Cbar_clean[:n, :m]))))
    return (s, s * m, s, s * n)


def fp64_input_thresholds(Abar, Bbar, rel=1e-11):
    n, m = Abar.shape[0] - 2, Bbar.shape[1] - 2
    sa = rel * max(1.0, float(np.max(np.abs(Abar[:n])))) * n
    sb = rel * max(1.0, float(np.max(np.abs(Bbar[:, :m])))) * m
    return (sa, sa * n, sb, sb * m)


# ----------------------------------------------------------------------------------------------
# Report
# ----------------------------------------------------------------------------------------------
@dataclass
class Report:
    verdict: int
    found: list = field(default_factory=list)      # sorted [(kind, row, col, magnitude)]; row/col = -1 where not applicable
    n_row_flags: int = 0
    n_col_flags: int = 0
    max_abs_syndrome: tuple = (0.0, 0.0, 0.0, 0.0)  # max |r1|, |r2|, |q1|, |q2| before correction
    C: np.ndarray | None = None                    # data part of C after correction (n x m)
    A: np.ndarray | None = None                    # Level-X only: data part of A after patching
    B: np.ndarray | None = None

    def located(self):
        """Positions without magnitudes: what must match bit-exactly."""
        return [(kd, r, c) for kd, r, c, _ in self.found]


# ----------------------------------------------------------------------------------------------
# O6  Level-P decoder: the paper's decoder on C_bar only, completed where the
# paper is silent (readings R5-R8 of DESIGN.md).
# ----------------------------------------------------------------------------------------------
def _locate_short_side(S_flag, L_flag, p1, p2, n_short, tau_p1, tol):
    """Work "rows-short": all errors are confined to <= 2 rows (the paper's WLOG s <= t).

    S_flag : flagged indices of the short side (rows), |S_flag| <= 2
    L_flag : flagged indices of the long side (columns)
    p1, p2 : plain / weighted syndromes of the long side (q1, q2)
    Returns the sorted row set S (|S| <= 2) or None (uncorrectable).

    A flagged column j is EXPLAINED by S if |S| = 2 (Theorem 2: two known rows can absorb any
    column's two syndromes), or S = {s} and q2_j = (s+1) q1_j (a single error in row s).
    Unexplained columns arise from INPUT faults, whose own-side syndromes vanish (reading R7): the faulty
    row is then located by the weighted ratio q2_j / q1_j, the classical use of P_n2.
    """
    S = sorted(S_flag)

    def explained(j, S):
        if len(S) == 2:
            return True
        if len(S) == 1:
            return abs(p2[j] - (S[0] + 1) * p1[j]) <= tol
        return False

    U = [j for j in L_flag if not explained(j, S)]
    if U:
        votes = {}
        all_valid = True
        for j in U:
            if abs(p1[j]) <= tau_p1:
                continue                                  # flagged by the weighted check only: cannot vote
            if not (np.isfinite(p1[j]) and np.isfinite(p2[j])):
                all_valid = False                         # reading R19: a non-finite syndrome locates nothing
                continue
            ihat = int(round(p2[j] / p1[j])) - 1
            if 0 <= ihat < n_short and abs(p2[j] - (ihat + 1) * p1[j]) <= tol:
                votes[ihat] = votes.get(ihat, 0) + 1
            else:
                all_valid = False
        if len(S) == 0:
            if (not all_valid) or len(votes) == 0 or len(votes) > 2:
                return None
            S = sorted(votes)
        else:
            others = {i: v for i, v in votes.items() if i != S[0]}
            if not others:
                return None
            best = max(others, key=lambda i: (others[i], -i))   # mode; ties -> smallest index
            S = sorted([S[0], best])
        if any(not explained(j, S) for j in L_flag):
            return None
    return S


def _estimate_short_side(S, p1, p2):
    """Error estimates x_hat[s][j] for every long-side index j (PAPER.md:223 for |S| = 1, PAPER.md:227 for |S| = 2).

    |S| = 2 solves [[1, 1], [s1, s2]] [x1, x2]^T = [q1_j, q2_j]^T with the right-hand side "sum minus parity"
    (reading R8: PAPER.md:227 prints parity minus sum, which would double the error when subtracted as 231 says).
    """
    if len(S) == 1:
        return {S[0]: np.array(p1, dtype=np.float64)}
    s1, s2 = S
    w1, w2 = s1 + 1, s2 + 1
    x2 = (np.asarray(p2) - w1 * np.asarray(p1)) / (w2 - w1)
    x1 = np.asarray(p1) - x2
    return {s1: x1, s2: x2}


MAX_POINTS_PER_LINE = 4    # a line with more located symbols than this is reported as a whole-line fault


def _hidden_point(s, s1_syn, s2_syn, n_long, tau_s1, tol_s):
    """Position of a single error explaining line s's OWN two syndromes (ratio of the weighted to the plain one is an
    integer weight, the classical locator of P_m2), or None."""
    if not (abs(s1_syn[s]) > tau_s1) or not (np.isfinite(s1_syn[s]) and np.isfinite(s2_syn[s])):
        return None
    jhat = int(round(s2_syn[s] / s1_syn[s])) - 1
    if 0 <= jhat < n_long and abs(s2_syn[s] - (jhat + 1) * s1_syn[s]) <= tol_s:
        return jhat
    return None


def _decode_oriented(S_flag, L_flag, s1_syn, s2_syn, l1_syn, l2_syn, n_short, n_long, tau_s1, tau_l1, tol_s, tol_l):
    """Decode with errors confined to <= 2 lines of the short side.  Returns None (uncorrectable) or
    (line_faults, points, patches) in short/long coordinates:
       line_faults: [s]                whole-line fault of short-side line s (an input fault)
       points:      [(s, j, x)]        isolated symbol errors
       patches:     {s: (x_hat, mask)} values to subtract from line s at long-side positions where mask
    """
    S = _locate_short_side(S_flag, L_flag, l1_syn, l2_syn, n_short, tau_l1, tol_l)
    if S is None or len(S) == 0:
        return None
    xhat = _estimate_short_side(S, l1_syn, l2_syn)
    line_faults, points, patches = [], [], {}
    for s in S:
        x = xhat[s]
        cols = [j for j in L_flag if abs(x[j]) > tau_l1]      # reading R5: located only if |x_hat| > tau
        if s not in S_flag:
            # found by the ratio locator, own-side syndromes silent: only an input fault does that
            line_faults.append(s)
            patches[s] = (x, np.ones(n_long, dtype=bool))     # reading R6: subtract everywhere on the line
        elif len(cols) >= 3 and _hidden_point(s, s1_syn, s2_syn, n_long, tau_s1, tol_s) is not None:
            # three or more bad symbols in a line whose OWN two syndromes are in the ratio of one column's weight: an
            # input fault shifted the whole line consistently and one C error hides in it.
            line_faults.append(s)
            patches[s] = (x, np.ones(n_long, dtype=bool))
            points.append((s, _hidden_point(s, s1_syn, s2_syn, n_long, tau_s1, tol_s), float(s1_syn[s])))
        elif len(cols) > MAX_POINTS_PER_LINE:
            # E(s, t) with t large and the line's own checks inconsistent with a single hidden error: the errors are
            # known to sit in this line, so every t* is corrected by the long-side syndromes (Theorem 2, PAPER.md:176;
            # s = 1: "for any t* in E_t"; s = 2: PAPER.md:225-231).  Too many to list: reported as a
            # whole-line fault and corrected along the whole line (reading R6).
            line_faults.append(s)
            patches[s] = (x, np.ones(n_long, dtype=bool))
        else:
            if not cols:
                return None                                   # flagged line, nothing locatable (e.g. parity-symbol fault, R11)
            mask = np.zeros(n_long, dtype=bool)
            for j in cols:
                points.append((s, j, float(x[j])))
                mask[j] = True
            patches[s] = (x, mask)
    return line_faults, points, patches


def global_checks(Cbar: np.ndarray):
    """Eq. (4) with the coefficients of reading R13: the parity rows / columns of C_bar are themselves
    codewords whose checks are the four global parity symbols P_g = [1; w_n] C [1, w_m].
      g_r[d, c] = sum_i w_d(i) P_r[i, c] - P_g[d, c]      (w_0 = 1, w_1(i) = i: plain / weighted sum over the rows)
      g_c[c, d] = sum_j w_d(j) P_c[c, j] - P_g[c, d]
    All eight vanish on a valid codeword."""
    Cbar = np.asarray(Cbar, dtype=np.float64)
    n, m = Cbar.shape[0] - 2, Cbar.shape[1] - 2
    wn, wm = np.arange(1, n + 1.0), np.arange(1, m + 1.0)
    P_r, P_c, P_g = Cbar[:n, m:], Cbar[n:, :m], Cbar[n:, m:]
    g_r = np.array([[P_r[:, c].sum() - P_g[0, c] for c in range(2)], [wn @ P_r[:, c] - P_g[1, c] for c in range(2)]])
    g_c = np.array([[P_c[c, :].sum() - P_g[c, 0], wm @ P_c[c, :] - P_g[c, 1]] for c in range(2)])
    return g_r, g_c


def parity_symbol_fault(Cbar: np.ndarray, R, Q, r1, r2, q1, q2, tau, tau_g):
    """A fault in ONE local parity symbol of C_bar (next: use of the global parity).  Signature: exactly one
    flagged line on one side, nothing on the other, and only ONE of the line's two checks off (a symbol of C would move
    both).  The global checks of that parity column / row then show the same error delta, at the line's weight:
        P_r[i, c] += delta  =>  r_{c,i} = -delta,  g_r[0, c] = delta,  g_r[1, c] = (i + 1) delta.
    Returns (kind, row, col, delta) or None.  tau_g = (plain, weighted) tolerances of the global checks."""
    n, m = Cbar.shape[0] - 2, Cbar.shape[1] - 2
    g_r, g_c = global_checks(Cbar)
    if len(R) == 1 and not Q:
        i = R[0]
        syn, tl, g, kind = (r1[i], r2[i]), (tau[0], tau[1]), g_r, KIND_PR
    elif len(Q) == 1 and not R:
        i = Q[0]
        syn, tl, g, kind = (q1[i], q2[i]), (tau[2], tau[3]), g_c.T, KIND_PC      # g[d, c] for the column side too
    else:
        return None
    off = [abs(syn[c]) > tl[c] for c in range(2)]
    if off[0] == off[1]:
        return None
    c = 0 if off[0] else 1
    delta = -syn[c]
    if isinstance(tau_g, dict):                               # separate tolerances for the row side and the column side
        tau_g = tau_g["rows" if kind == KIND_PR else "cols"]
    tg = np.broadcast_to(np.asarray(tau_g, dtype=np.float64).reshape(2, -1), (2, 2))     # [d][c]; a pair (plain, weighted) serves both checks
    if not (abs(delta) > 4.0 * tg[0, c]):
        return None                                           # the global check must CONFIRM the error, not merely fail to contradict it
    if abs(g[0, c] - delta) <= tg[0, c] + tl[c] and abs(g[1, c] - (i + 1) * delta) <= tg[1, c] + (i + 1) * tl[c]:
        return (kind, i, c, float(delta)) if kind == KIND_PR else (kind, c, i, float(delta))
    return None


def decode_level_p(Cbar: np.ndarray, tau, tau_g=None) -> Report:
    """The paper's detection + correction on C_bar alone.  tau = (tau_r1, tau_r2, tau_q1, tau_q2).

    Steps: (1) syndromes; (2) flag sets E_r, E_t; (3) clean if both empty; "needs to be
    recalculated" if min(s,t) >= 3; (4) otherwise WLOG s <= t: correct with the
    column syndromes, s = 1 by subtraction, s = 2 by the 2x2 solve; the
    transposed orientation swaps the roles of rows and columns.
    """
    Cbar = np.asarray(Cbar, dtype=np.float64)
    n, m = Cbar.shape[0] - 2, Cbar.shape[1] - 2
    t_r1, t_r2, t_q1, t_q2 = tau
    r1, r2, q1, q2 = syndromes(Cbar)
    R, Q = flag_sets(r1, r2, q1, q2, tau)

    def mx(v):
        return float(np.max(np.abs(v))) if len(v) else 0.0

    rep = Report(verdict=CLEAN, n_row_flags=len(R), n_col_flags=len(Q),
                 max_abs_syndrome=(mx(r1), mx(r2), mx(q1), mx(q2)), C=Cbar[:n, :m].copy())
    if not R and not Q:
        return rep
    rep.verdict = UNCORRECTABLE
    if len(R) >= 3 and len(Q) >= 3:                            # min(s,t) >= 3
        return rep
    rows_short = len(R) <= len(Q)                               # tie -> rows-short
    if rows_short:
        out = _decode_oriented(R, Q, r1, r2, q1, q2, n, m, t_r1, t_q1, t_r2, t_q2)
    else:
        out = _decode_oriented(Q, R, q1, q2, r1, r2, m, n, t_q1, t_r1, t_q2, t_r2)
    if out is None:
        if tau_g is not None:                                   # nothing locatable in C: a parity symbol of C_bar itself?
            pf = parity_symbol_fault(Cbar, R, Q, r1, r2, q1, q2, tau, tau_g)
            if pf is not None:
                rep.found = [pf]                                # C is intact; the symbol is what is corrected
                rep.verdict = CORRECTED
        return rep
    line_faults, points, patches = out
    C = rep.C
    found = []
    for s in line_faults:
        found.append((KIND_ROW, s, -1, 0.0) if rows_short else (KIND_COL, -1, s, 0.0))
    for s, j, x in points:
        found.append((KIND_C, s, j, x) if rows_short else (KIND_C, j, s, x))
    for s, (x, mask) in patches.items():                       # c_true = c - e
        if rows_short:
            C[s, mask] -= x[mask]
        else:
            C[mask, s] -= x[mask]
    rep.found = sorted(set(found), key=lambda f: (f[0], f[1], f[2]))
    rep.verdict = CORRECTED
    return rep


# ----------------------------------------------------------------------------------------------
# O7  Level-X: input verification (extension, reading R9).  Each column of A_bar is a codeword
# of G_A, each row of B_bar a codeword of G_B, so one corrupted symbol per column of
# A / row of B is located by the same plain + weighted checksum pair.
# ----------------------------------------------------------------------------------------------
def verify_left(Abar: np.ndarray, tau_a1: float, tol_a2: float):
    """Returns (list of (i, l, e), ok).  sA1_l = sum_i a_il - A_P[0,l];  sA2_l = sum_i i a_il - A_P[1,l]."""
    n = Abar.shape[0] - 2
    P = encode_left(Abar[:n, :])
    s1 = P[0] - Abar[n]
    s2 = P[1] - Abar[n + 1]
    out = []
    for l in range(Abar.shape[1]):
        if abs(s1[l]) <= tau_a1 and abs(s2[l]) <= tol_a2:
            continue
        if not (abs(s1[l]) > tau_a1) or not (np.isfinite(s1[l]) and np.isfinite(s2[l])):
            return [], False
        ihat = int(round(s2[l] / s1[l])) - 1
        if not (0 <= ihat < n and abs(s2[l] - (ihat + 1) * s1[l]) <= tol_a2):
            return [], False
        out.append((ihat, l, float(s1[l])))
    return out, True


def verify_right(Bbar: np.ndarray, tau_b1: float, tol_b2: float):
    """Returns (list of (l, j, e), ok) -- the mirror image of verify_left on the rows of B_bar."""
    faults, ok = verify_left(np.ascontiguousarray(Bbar.T), tau_b1, tol_b2)
    return [(l, j, e) for j, l, e in faults], ok


def decode_level_x(Cbar, Abar, Bbar, tau, tau_in, tau_g=None) -> Report:
    """Level-P, then -- if it reports a whole-row / whole-column fault or gives up -- verify the operands against
    their own parity, patch A / B, undo the faults' exact rank-1 footprint on C_bar, and decode what is left.

    tau_in = (tau_a1, tol_a2, tau_b1, tol_b2).
    Repair order: C[i,:] -= e B_faulty[l,:] for every A fault, patch A, then C[:,j] -= e' A_patched[:,l'] for every
    B fault, patch B  (because (A+E_A)(B+E_B) = AB + E_A (B+E_B) + A E_B).
    """
    Cbar = np.asarray(Cbar, dtype=np.float64)
    Abar = np.asarray(Abar, dtype=np.float64)
    Bbar = np.asarray(Bbar, dtype=np.float64)
    n, m = Cbar.shape[0] - 2, Cbar.shape[1] - 2
    rep = decode_level_p(Cbar, tau, tau_g)
    rep.A = Abar[:n].copy()
    rep.B = Bbar[:, :m].copy()
    only_points = rep.verdict == CORRECTED and all(f[0] in (KIND_C, KIND_PR, KIND_PC) for f in rep.found)
    if rep.verdict == CLEAN or only_points:
        return rep
    fa, ok_a = verify_left(Abar, tau_in[0], tau_in[1])
    fb, ok_b = verify_right(Bbar, tau_in[2], tau_in[3])
    if not (ok_a and ok_b):
        rep.verdict = UNCORRECTABLE_INPUT
        rep.found = []
        rep.C = Cbar[:n, :m].copy()
        return rep
    if not fa and not fb:
        return rep                                             # memory intact: keep the Level-P result
    C2, A2, B2 = Cbar.copy(), Abar.copy(), Bbar.copy()
    for i, l, e in fa:
        C2[i, :] -= e * B2[l, :]
    for i, l, e in fa:
        A2[i, l] -= e
    for l, j, e in fb:
        C2[:, j] -= e * A2[:, l]
    for l, j, e in fb:
        B2[l, j] -= e
    rep2 = decode_level_p(C2, tau)
    out = Report(verdict=UNCORRECTABLE, n_row_flags=rep.n_row_flags, n_col_flags=rep.n_col_flags,
                 max_abs_syndrome=rep.max_abs_syndrome, C=Cbar[:n, :m].copy(), A=Abar[:n].copy(), B=Bbar[:, :m].copy())
    if rep2.verdict == CLEAN or (rep2.verdict == CORRECTED and all(f[0] == KIND_C for f in rep2.found)):
        found = [(KIND_A, i, l, e) for i, l, e in fa] + [(KIND_B, l, j, e) for l, j, e in fb] + list(rep2.found)
        out.found = sorted(found, key=lambda f: (f[0], f[1], f[2]))
        out.verdict = CORRECTED
        out.C, out.A, out.B = rep2.C, A2[:n], B2[:, :m]
    return out


# ----------------------------------------------------------------------------------------------
# Single-checksum mode: only P_n1 and P_m1 are used (the scheme of ref [8], which the "Checksum" columns of
# Table I, stand for).  One error in C is located at the crossing of the one bad row and the one bad
# column and equals either plain syndrome; everything else is detected but cannot be corrected from C_bar.
# ----------------------------------------------------------------------------------------------
def decode_single_checksum(Cbar: np.ndarray, tau) -> Report:
    Cbar = np.asarray(Cbar, dtype=np.float64)
    n, m = Cbar.shape[0] - 2, Cbar.shape[1] - 2
    r1, r2, q1, q2 = syndromes(Cbar)
    R = [i for i in range(n) if not (abs(r1[i]) <= tau[0])]
    Q = [j for j in range(m) if not (abs(q1[j]) <= tau[2])]
    rep = Report(verdict=CLEAN, n_row_flags=len(R), n_col_flags=len(Q),
                 max_abs_syndrome=(float(np.max(np.abs(r1))), 0.0, float(np.max(np.abs(q1))), 0.0), C=Cbar[:n, :m].copy())
    if not R and not Q:
        return rep
    rep.verdict = UNCORRECTABLE
    if len(R) == 1 and len(Q) == 1 and abs(r1[R[0]] - q1[Q[0]]) <= tau[0] + tau[2]:
        i, j = R[0], Q[0]
        rep.C[i, j] -= q1[j]
        rep.found = [(KIND_C, i, j, float(q1[j]))]
        rep.verdict = CORRECTED
    return rep


# ----------------------------------------------------------------------------------------------
# Recompute fallback ("cannot correct errors and needs to be recalculated"; "mark the compromised
# data for recomputation"): the flagged rows of C (or the flagged columns, whichever are fewer) are computed again from
# the operands as they are, then the checks are taken again.
# ----------------------------------------------------------------------------------------------
def recompute_fallback(Cbar: np.ndarray, Abar: np.ndarray, Bbar: np.ndarray, tau) -> Report:
    Cbar = np.asarray(Cbar, dtype=np.float64).copy()
    n, m = Cbar.shape[0] - 2, Cbar.shape[1] - 2
    R, Q = flag_sets(*syndromes(Cbar), tau)
    first = Report(verdict=UNCORRECTABLE, n_row_flags=len(R), n_col_flags=len(Q), C=Cbar[:n, :m].copy())
    if not R and not Q:
        first.verdict = CLEAN
        return first
    rows = bool(R) and (len(R) <= len(Q) or not Q)
    if rows:
        Cbar[R, :m] = np.asarray(Abar, dtype=np.float64)[R, :] @ np.asarray(Bbar, dtype=np.float64)[:, :m]
    else:
        Cbar[:n, Q] = np.asarray(Abar, dtype=np.float64)[:n, :] @ np.asarray(Bbar, dtype=np.float64)[:, Q]
    rep = decode_level_p(Cbar, tau)
    if rep.verdict == CLEAN or (rep.verdict == CORRECTED and all(f[0] == KIND_C for f in rep.found)):
        rep.verdict = CORRECTED_BY_RECOMPUTE
        rep.n_row_flags, rep.n_col_flags = first.n_row_flags, first.n_col_flags
        return rep
    return first


# ----------------------------------------------------------------------------------------------
# Tile-local grid (a variant of Def. 1, not something the paper evaluates): one code
# M(P + 2, k, Q + 2) per panel of P rows of A and Q columns of B, weights local to the panel (1..P, 1..Q).  The blocks of
# C are independent codewords: each corrects its own <= 2 errors, the weights never exceed the panel size.
# ----------------------------------------------------------------------------------------------
def panel_ranges(length: int, panel: int):
    return [(s, min(length, s + panel)) for s in range(0, length, panel)]


def encode_panels(A: np.ndarray, B: np.ndarray, P: int, Q: int):
    """Per-panel parity: A_P[rp] = [1; (1..P)] A[rows of panel rp]  (2 x k each), B_P[cp] = B[:, cols of panel cp] [1, (1..Q)]."""
    A = np.asarray(A, dtype=np.float64)
    B = np.asarray(B, dtype=np.float64)
    return ([encode_left(A[r0:r1]) for r0, r1 in panel_ranges(A.shape[0], P)],
            [encode_right(B[:, c0:c1]) for c0, c1 in panel_ranges(B.shape[1], Q)])


def decode_panels(C_faulty: np.ndarray, A: np.ndarray, B: np.ndarray, P: int, Q: int, tau_of_block, parity=None) -> Report:
    """C_faulty: the n x m data part as computed (with errors).  Every block (rp, cp) is completed with its own parity
    -- P_r = A_rp B_P[cp], P_c = A_P[rp] B_cp, P_g -- and decoded on its own by decode_level_p; the report lists the
    located symbols in GLOBAL coordinates.  tau_of_block(rows, cols) -> thresholds.
    parity = (AP, BP) from encode_panels on the CLEAN operands, with A, B the operands as the product read them: an input
    fault strikes after encoding (reading R1), so the parity of the product comes from the faulty operand times
    the clean parity of the other side, as in encoded_product.  Default: A and B are intact and encoded here."""
    A = np.asarray(A, dtype=np.float64)
    B = np.asarray(B, dtype=np.float64)
    n, m = C_faulty.shape
    AP, BP = encode_panels(A, B, P, Q) if parity is None else parity
    out = Report(verdict=CLEAN, C=np.array(C_faulty, dtype=np.float64, copy=True))
    for bi, (r0, r1) in enumerate(panel_ranges(n, P)):
        for bj, (c0, c1) in enumerate(panel_ranges(m, Q)):
            Cbar = np.zeros((r1 - r0 + 2, c1 - c0 + 2))
            Cbar[:-2, :-2] = out.C[r0:r1, c0:c1]
            Cbar[:-2, -2:] = A[r0:r1] @ BP[bj]                    # P_r of the block
            Cbar[-2:, :-2] = AP[bi] @ B[:, c0:c1]                 # P_c
            Cbar[-2:, -2:] = AP[bi] @ BP[bj]                      # P_g
            rep = decode_level_p(Cbar, tau_of_block(r1 - r0, c1 - c0))
            out.n_row_flags += rep.n_row_flags
            out.n_col_flags += rep.n_col_flags
            if rep.verdict == CLEAN:
                continue
            if rep.verdict != CORRECTED:
                out.verdict = UNCORRECTABLE
                continue
            out.C[r0:r1, c0:c1] = rep.C
            out.found += [(kd, (r + r0 if r >= 0 else r), (c + c0 if c >= 0 else c), mag) for kd, r, c, mag in rep.found]
            if out.verdict == CLEAN:
                out.verdict = CORRECTED
    out.found.sort(key=lambda f: (f[0], f[1], f[2]))
    return out


# ----------------------------------------------------------------------------------------------
# Whole path, for convenience: encode -> inject -> product -> inject -> decode
# ----------------------------------------------------------------------------------------------
def protected_matmul(A, B, faults=(), tau=None, tau_in=None, level=1) -> Report:
    """faults: [(kind, row, col, e)], kind 0 = A symbol (i,l), 1 = B symbol (l,j), 2 = C symbol (i,j); additive."""
    A = np.asarray(A, dtype=np.float64)
    B = np.asarray(B, dtype=np.float64)
    n, k = A.shape
    m = B.shape[1]
    Abar, Bbar = encoded_operands(A, B)                         # parity from CLEAN data (reading R1)
    if tau is None:
        tau = fp64_thresholds(n, m, encoded_product(Abar, Bbar))
    if tau_in is None:
        tau_in = fp64_input_thresholds(Abar, Bbar)
    Abar_f, Bbar_f = inject_input_faults(Abar, Bbar, faults)    # E1 / E2
    Cbar = inject_output_faults(encoded_product(Abar_f, Bbar_f), faults)   # product, then E3
    if level == 0:
        return decode_level_p(Cbar, tau)
    return decode_level_x(Cbar, Abar_f, Bbar_f, tau, tau_in)
