/* gecc.h -- C ABI of the B200 (sm_100a) grid-like error-correcting code for matrix multiplication.
 *
 * Method: arxiv 2508.04355, "Grid-like Error-Correcting Codes for Matrix Multiplication with Better Correcting
 * Capability".  Citations below are PAPER.md line numbers (section / equation).  Notation is the paper's
 * (PAPER.md:31-35): A is n x k (left), B is k x m (right), C = A B is n x m.  The paper is 1-based; this ABI is
 * 0-based and the weight of 0-based index r is r + 1 (PAPER.md:83 P_n2 = (1..n), PAPER.md:101 P_m2 = (1..m)).
 *
 * Common rules for every entry point
 *   - Every pointer is a DEVICE pointer owned by the caller unless its comment says HOST.  The library never
 *     allocates, frees or retains user memory; scratch comes from the caller's `workspace`.
 *   - Every call is asynchronous on `stream` (a cudaStream_t passed as void*; NULL = the legacy default stream)
 *     and never synchronises it.  Host-side work is limited to argument checks and building TMA descriptors.
 *   - Matrices are row-major with a leading dimension in ELEMENTS.  Operand base pointers must be 16-byte aligned
 *     and leading dimensions must make every row start 16-byte aligned (ld % 8 == 0 for bf16, ld % 4 == 0 for fp32).
 *   - Return value: GECC_OK (0) or a negative gecc_status_t.  A detected-but-uncorrectable fault is NOT an error
 *     return: it is a verdict in the device-side report.
 */
#ifndef GECC_H_
#define GECC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  GECC_OK = 0,
  GECC_EINVAL = -1,       /* null pointer, non-positive size, bad alignment or leading dimension */
  GECC_EUNSUPPORTED = -2, /* dtype / layout combination not implemented */
  GECC_ECUDA = -3,        /* a CUDA runtime or driver call failed (launch failure, no sm_100 device, ...) */
  GECC_EWORKSPACE = -4,   /* workspace_bytes smaller than gecc_workspace_bytes() */
  GECC_ETOOLARGE = -5     /* operand needs more scratch than the library's fixed array (gecc_encode_noalloc) */
} gecc_status_t;

/* Arithmetic of the encoded product.  Both accumulate in fp32 on the tensor cores and return C in fp32. */
typedef enum {
  GECC_BF16 = 0,  /* A, B hold bf16; parity symbols are carried as 3 bf16 limbs (24 bits) */
  GECC_F32 = 1    /* A, B hold fp32; product by the 3xTF32 split (hi*hi + hi*lo + lo*hi) */
} gecc_dtype_t;

typedef enum {
  GECC_LEFT = 0, /* generator G_A = [I; 1; (1..n)]: two parity ROWS appended below A */
  GECC_RIGHT = 1 /* generator G_B = [I, 1^T, (1..m)^T]: two parity COLUMNS appended to B */
} gecc_side_t;

/* Number of rows of the parity operand buffers (both sides): 2 checks x 3 limbs, padded to 8. */
#define GECC_PAR_ROWS 8
/* Parity of C as the product emits it: P_r is n x GECC_PR_LD fp32, P_c is GECC_PAR_ROWS x m fp32.  Limb l of
 * check c (c = 0 plain, 1 weighted) sits in column / row 3 c + l; the symbol of PAPER.md:121-127 is the sum of its
 * limbs (GECC_F32 uses one limb: column / row 3 c). */
#define GECC_PR_LD 8

/* An injected fault (E1/E2/E3): additive `value` on one symbol. */
typedef struct {
  int32_t kind; /* 0 = symbol of A (row i, col l), 1 = symbol of B (row l, col j), 2 = symbol of C (row i, col j) */
  int32_t row, col;
  float value;
} gecc_fault_t;

enum { GECC_CLEAN = 0, GECC_CORRECTED = 1, GECC_UNCORRECTABLE = 2, GECC_UNCORRECTABLE_INPUT = 3,
       GECC_CORRECTED_BY_RECOMPUTE = 4 /* set by gecc_recompute_fallback only */ };
/* GECC_KIND_PR / GECC_KIND_PC: a local parity symbol of C_bar itself is faulty, C is intact (Eq. 4):
 * PR: (row i, check c of P_r), PC: (check c, column j of P_c); c = 0 plain, 1 weighted. */
enum { GECC_KIND_A = 0, GECC_KIND_B = 1, GECC_KIND_C = 2, GECC_KIND_ROW = 3, GECC_KIND_COL = 4, GECC_KIND_PR = 5, GECC_KIND_PC = 6 };
/* Bits of the `level` argument of gecc_decode_correct / the `mode` argument of gecc_matmul_protected. */
#define GECC_LEVEL_X 1          /* verify the operands against their own parity (input attribution) */
#define GECC_SINGLE_CHECKSUM 2  /* use the plain checks P_n1 / P_m1 only: the single-checksum scheme of ref [8] that
                                   Table I's "Checksum" columns stand for; corrects one error in C, refuses everything else */
#define GECC_MAX_FOUND 8

typedef struct {
  int32_t kind; /* GECC_KIND_*: A symbol (i,l) | B symbol (l,j) | C symbol (i,j) | whole row (i,-1) | whole column (-1,j) */
  int32_t row, col;
  int32_t pad_;
  double magnitude; /* estimated additive error (0 for whole-row / whole-column entries) */
} gecc_found_t;

/* Written to device memory by gecc_decode_correct.  `found` is sorted by (kind, row, col). */
typedef struct {
  int32_t verdict; /* GECC_CLEAN | GECC_CORRECTED | GECC_UNCORRECTABLE (recompute) | GECC_UNCORRECTABLE_INPUT */
  int32_t n_found;
  int32_t n_row_flags, n_col_flags; /* |E_r|, |E_t| of PAPER.md:215 before any repair */
  double max_abs_syndrome[4];       /* max |r1|, |r2|, |q1|, |q2| before any repair */
  double tau[4];                    /* thresholds used for r1, r2, q1, q2 */
  gecc_found_t found[GECC_MAX_FOUND];
} gecc_report_t;

/* Bytes of scratch every call below needs for problem (n, k, m); one buffer may serve all calls of one product.
 * The protected product leaves its per-tile partial sums there and the decoder reads them, so the buffer must
 * stay untouched between gecc_matmul_protected and gecc_decode_correct.  The buffer must be 256-byte aligned and
 * ZERO when first used (it holds arrival counters that every kernel leaves zero again); calls that share a workspace
 * must be ordered on one stream. */
size_t gecc_workspace_bytes(int dtype, int64_t n, int64_t k, int64_t m);

/* Encoder (section III).  X is the operand as stored: rows x cols, row-major, leading dimension ld.
 *   trans = 0: X holds the operand itself (A: n x k, B: k x m).  trans = 1: X holds its transpose (A^T: k x n, B^T: m x k),
 *   as the backward products dW = X^T dY and dX = dY W^T need; the checks are those of the operand either way.
 *   side = GECC_LEFT : X = A (n x k).  Emits A_P: check 0 = sum_i a_il, check 1 = sum_i (i+1) a_il.
 *   side = GECC_RIGHT: X = B (k x m).  Emits B_P: check 0 = sum_j b_lj, check 1 = sum_j (j+1) b_lj.
 * Outputs (all of inner length len = k):
 *   parity   [GECC_PAR_ROWS x len] in the operand dtype, row-major, ld = len: the parity operand of the product.
 *            bf16: rows 0..2 = limbs of check 0, rows 3..5 = limbs of check 1.  fp32: row 0 = check 0, row 3 = check 1.
 *   parity_lo[GECC_PAR_ROWS x len] fp32, GECC_F32 only (else NULL): the 3xTF32 low parts of `parity`.
 *   x_lo     [rows x cols, ld] fp32, GECC_F32 only (else NULL): low parts x - tf32_trunc(x) of the operand.  It shares X's
 *            leading dimension `ld` (one index serves both planes in every kernel): a padded X needs an equally padded x_lo.
 *   parity64 [2 x len] fp64: the two checks as accumulated (before rounding to limbs); input verification uses it.
 *   sumsq    [1] fp64: sum of squares of X (feeds the automatic thresholds).
 * Two calls on the same workspace may run concurrently on two streams only if they reduce in different directions, i.e. a
 * GECC_LEFT and a GECC_RIGHT call with EQUAL `trans` (over the storage rows for LEFT / trans = 0 and RIGHT / trans = 1, along
 * them otherwise): the two directions use disjoint scratch and arrival counters, two reductions of the same direction
 * share them and must be ordered on one stream (or use separate workspaces).
 * Reads X once (HBM-bound).  The parity is computed from X as it is at call time: a fault must be injected AFTER
 * this call to be detectable (reading R1 of DESIGN.md). */
int gecc_encode(int dtype, int side, int trans, const void* X, int64_t rows, int64_t cols, int64_t ld,
                void* parity, float* parity_lo, float* x_lo, double* parity64, double* sumsq,
                void* workspace, size_t workspace_bytes, void* stream);

/* gecc_encode for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): same operation, same arguments and same results as gecc_encode, but there is no workspace argument.  The
 * scratch (arrival counters and the per-chunk partial sums of the reduction) is a fixed array of
 * GECC_NOALLOC_SCRATCH_BYTES inside the library's device image; every GPU that loads the library holds it until the
 * process exits.  The call allocates and frees nothing (no cudaMalloc / cudaFree, no allocating library routine).
 *   Limit: the scratch a rows x cols operand needs -- 8 * 2 * cols * ceil(rows / 64) bytes of partial sums plus about
 *   100 KB, i.e. roughly rows * cols / 4 bytes -- must fit the array: operands up to 4096 x 8192 (either way round) do,
 *   8192 x 8192 does not.  A larger operand is refused with GECC_ETOOLARGE before anything is launched.
 *   Sharing: ALL calls on one GPU use the same array, which keeps the previous call's contents.  Each call clears the
 *   arrival counters itself (a 4 KB memset on `stream` ahead of the kernel); the partial sums are overwritten before they
 *   are read.  Two calls that overlap on the GPU (different streams, or graphs replayed concurrently) RACE on it and
 *   return wrong checks: order them on one stream.  Calls to the other entry points are unaffected (they use the
 *   caller's workspace).
 *   Set-up: the first call on each device looks up the array's device address (cudaGetSymbolAddress, once per device);
 *   make that first call outside stream capture. */
#define GECC_NOALLOC_SCRATCH_BYTES (9u << 20)
int gecc_encode_noalloc(int dtype, int side, int trans, const void* X, int64_t rows, int64_t cols, int64_t ld,
                        void* parity, float* parity_lo, float* x_lo, double* parity64, double* sumsq, void* stream);

/* Both encoders in ONE launch (same outputs as two gecc_encode calls, GECC_LEFT on A and GECC_RIGHT on B): the blocks of
 * the two reductions share the SMs as slots come free, each operand has its own arrival counters and scratch (any
 * combination of trans_a / trans_b), and the product that follows in the stream may begin to launch while this kernel
 * drains (programmatic dependent launch).  The kernel is itself launched as a programmatic dependent: it waits, on the device,
 * for the kernel before it in the stream (the decoder of the previous product releases its dependents early, so this encoder's
 * blocks take their places while that decoder drains) and reads nothing before that kernel has completed.
 * A: n x k (trans_a = 1: A^T stored k x n), B: k x m (trans_b = 1: B^T stored m x k). */
int gecc_encode_both(int dtype, int64_t n, int64_t k, int64_t m, int trans_a, int trans_b,
                     const void* A, int64_t lda, void* A_par, float* A_par_lo, float* A_lo, double* A_par64, double* sumsq_a,
                     const void* B, int64_t ldb, void* B_par, float* B_par_lo, float* B_lo, double* B_par64, double* sumsq_b,
                     void* workspace, size_t workspace_bytes, void* stream);

/* Encoded product C_bar = A_bar B_bar = [[C, P_r], [P_c, P_g]] on the tensor cores, with the row
 * and column sums of the detection step taken from the accumulators in the epilogue and left in
 * `workspace` as per-tile partials, so C is not read again.
 *   A [n x k, lda], B [k x m, ldb] in `dtype` (trans_a = 1: A points to A^T stored k x n; trans_b = 1: B points to B^T
 *   stored m x k; the leading dimensions are those of the storage); A_par / B_par from gecc_encode (GECC_LEFT / GECC_RIGHT);
 *   A_lo, A_par_lo, B_lo, B_par_lo: GECC_F32 only (else NULL).  A_lo / B_lo are the x_lo planes gecc_encode wrote: same shape
 *   and SAME leading dimension as A / B (lda / ldb apply to them too).
 *   C [n x m, ldc] fp32;  P_r [n x GECC_PR_LD] fp32;  P_c [GECC_PAR_ROWS x m] fp32;  P_g [GECC_PAR_ROWS x GECC_PR_LD] fp32.
 *   inject [n_inject], DEVICE, may be NULL: kind-2 faults are added to the accumulator of C(row, col) before it is
 *   summed and stored (E3); other kinds are ignored here.  Production passes NULL, 0.
 *   Detection inside the product: if the thresholds are known -- tau (HOST, 4 values for r1, r2, q1, q2)
 *   or, with tau NULL, sumsq_a and sumsq_b (DEVICE, from gecc_encode; automatic thresholds as stated under
 *   gecc_decode_correct) -- the CTA that completes the last block of a strip of 128 rows / columns folds the strip's
 *   sums into syndromes and flags at once, and a product with no flagged line is settled right here: `report` (DEVICE,
 *   may be NULL) receives the CLEAN verdict and gecc_decode_correct, if still called, returns at once.  With tau, sumsq_a
 *   and sumsq_b all NULL only the per-tile sums are left and gecc_decode_correct folds them itself.  Pass the SAME tau /
 *   sumsq_a / sumsq_b to gecc_decode_correct afterwards.
 *   mode: 0, or GECC_SINGLE_CHECKSUM (lines are flagged by their plain check alone; pass the same bit in `level` below). */
int gecc_matmul_protected(int dtype, int64_t n, int64_t k, int64_t m, int trans_a, int trans_b,
                          const void* A, int64_t lda, const void* A_par, const float* A_lo, const float* A_par_lo,
                          const void* B, int64_t ldb, const void* B_par, const float* B_lo, const float* B_par_lo,
                          float* C, int64_t ldc, float* P_r, float* P_c, float* P_g,
                          const gecc_fault_t* inject, int n_inject,
                          const double* tau, const double* sumsq_a, const double* sumsq_b, gecc_report_t* report, int mode,
                          void* workspace, size_t workspace_bytes, void* stream);

/* The same kernel without parity tiles and epilogue sums: C = A B.  The like-for-like "unprotected GEMM" that the
 * overhead is quoted against. */
int gecc_matmul_plain(int dtype, int64_t n, int64_t k, int64_t m, int trans_a, int trans_b,
                      const void* A, int64_t lda, const float* A_lo, const void* B, int64_t ldb, const float* B_lo,
                      float* C, int64_t ldc, void* stream);

/* Standalone detection sums over a STORED C (HBM-bound, reads C once): fills `workspace` with the same partials
 * the protected product's epilogue leaves.  For checking C at rest and as the unfused baseline.  (n, k, m) is the
 * shape of the product the workspace was sized for (k only places the partials inside it). */
int gecc_syndrome_unfused(int dtype, int64_t n, int64_t k, int64_t m, const float* C, int64_t ldc,
                          void* workspace, size_t workspace_bytes, void* stream);

/* Detection and correction (section V), in place, no host round trip.
 *   Syndromes r1, r2 (rows) and q1, q2 (columns) = sum minus parity from the partials in
 *   `workspace` and P_r, P_c; flag sets against tau; min(s,t) >= 3 -> GECC_UNCORRECTABLE
 *   (PAPER.md:219); otherwise locate and subtract.
 *   tau: HOST pointer to 4 thresholds for r1, r2, q1, q2, or NULL for the automatic ones derived on the device from
 *        sumsq_a, sumsq_b (reading R4; the paper states one delta of unstated scale):
 *          sigma_plain(len) = c(k) 2^-24 sqrt(k len) sigma_a sigma_b,   c(k) = 2 + c0 (k / 1024)^(2/3),
 *          c0 = 4.5 (GECC_BF16), 20 (GECC_F32);  sigma_a = sqrt(sumsq_a / (n k)), sigma_b = sqrt(sumsq_b / (k m));
 *          tau_r1 = kappa sigma_plain(m), tau_q1 = kappa sigma_plain(n), kappa = 16;
 *          tau_r2 = tau_r1 sqrt((m+1)(2m+1)/6), tau_q2 = tau_q1 sqrt((n+1)(2n+1)/6)   (RMS of the weights 1..len).
 *        A line whose measured energy sum c^2 exceeds the expected len k sigma_a^2 sigma_b^2 has its two thresholds scaled
 *        by sqrt of that ratio.  The report carries the four thresholds used.
 *   level 0: the paper's decoder on C_bar alone.  A / B faults are reported as whole-row / whole-column faults.
 *   level 1: additionally, when level 0 reports a whole-row / whole-column fault or gives up, A and B are checked
 *        against their own parity (A_par64 / B_par64), the faulty symbols of A / B are located and patched in place
 *        and their exact rank-1 footprint is removed from C (reading R9).  Needs A, B (and their lo parts
 *        for GECC_F32) writable; trans_a / trans_b say how they are stored, as for gecc_matmul_protected (ignored at
 *        level 0).  GECC_EUNSUPPORTED if k exceeds 65536 (bf16) / 32768 (fp32) with a transposed B, twice that otherwise.
 *   level bit GECC_SINGLE_CHECKSUM: single-checksum mode (level X is then ignored).
 *   P_g (may be NULL): the global parity block the product emitted.  With it, a flagged line in which nothing can be
 *        located is checked against Eq. (4): if the global checks of its parity column / row show the
 *        same error at the line's weight, ONE local parity symbol of C_bar is faulty and C is intact: verdict
 *        GECC_CORRECTED, found = GECC_KIND_PR / GECC_KIND_PC, the symbol is repaired in P_r / P_c.  Tolerances of the global
 *        checks: the line's thresholds times sqrt(n) (times the RMS weight of 1..n for the weighted one); sqrt(m) for P_c.
 *   P_r must be 16-byte aligned.
 *   report: DEVICE pointer to one gecc_report_t. */
int gecc_decode_correct(int dtype, int64_t n, int64_t k, int64_t m,
                        float* C, int64_t ldc, float* P_r, float* P_c, const float* P_g,
                        const double* tau, const double* sumsq_a, const double* sumsq_b, int level,
                        int trans_a, int trans_b, void* A, int64_t lda, float* A_lo, const double* A_par64,
                        void* B, int64_t ldb, float* B_lo, const double* B_par64,
                        gecc_report_t* report, void* workspace, size_t workspace_bytes, void* stream);

/* Recompute fallback ("cannot correct errors and needs to be recalculated").  SYNCHRONOUS: waits
 * for `stream`, reads the report of the preceding gecc_decode_correct; if its verdict is GECC_UNCORRECTABLE, the blocks of
 * 256 rows of C that hold a flagged row (or the blocks of 256 columns that hold a flagged column, whichever are fewer)
 * are computed again from the operands as they are (gecc_matmul_plain on sub-views), the detection sums are taken again
 * over the stored C (gecc_syndrome_unfused) and decoded at level 0 against the parity of the first product.  If that ends
 * CLEAN or with point errors corrected, the report's verdict becomes GECC_CORRECTED_BY_RECOMPUTE.  Other verdicts
 * (including GECC_UNCORRECTABLE_INPUT: the operands themselves are beyond repair) are left alone.
 * Returns the number of blocks recomputed (0: nothing to do) or a negative gecc_status_t.  Arguments as for the calls above. */
int gecc_recompute_fallback(int dtype, int64_t n, int64_t k, int64_t m, int trans_a, int trans_b,
                            const void* A, int64_t lda, const float* A_lo, const void* B, int64_t ldb, const float* B_lo,
                            float* C, int64_t ldc, float* P_r, float* P_c, const double* tau, const double* sumsq_a, const double* sumsq_b,
                            gecc_report_t* report, void* workspace, size_t workspace_bytes, void* stream);

/* ---- Tile-local grid: one code per 128 x 128 block of C (a variant of Def. 1; not evaluated by the paper) ----
 * A is cut into panels of GECC_TL_PANEL rows, B into panels of GECC_TL_PANEL columns; every pair (row panel p, column panel q)
 * carries its own code M(128 + 2, k, 128 + 2) with weights 1..128 LOCAL to the panel (PAPER.md:83, 101 per panel), so every
 * block C[p, q] is a codeword of its own: it corrects its own errors (any pattern confined to <= 2 rows or <= 2 columns of the
 * block, Theorem 2), errors in different blocks never add up, the thresholds do not grow with n or m, and the
 * weights are exact in bf16.  The price: 8 parity rows per panel, i.e. (n + m) / 16 extra rows / columns in the product
 * (+12.5 % of the flops at n = m), computed as ordinary tiles of the same kernel.
 * Operands row-major, NOT transposed (GECC_EUNSUPPORTED otherwise); the common rules above apply.  Level P only: a fault in a
 * symbol of A / B shows up as a whole-row / whole-column fault in every block it touches and is corrected there (R6); the
 * operand itself is not repaired.
 *   A_PL [gecc_tl_parity_rows(n) x k], B_PL [gecc_tl_parity_rows(m) x k], operand dtype, row-major with ld = k: rows 8 p + 3 c + l
 *        hold limb l of check c (0 plain, 1 weighted) of panel p (fp32: row 8 p + 3 c, low parts in A_PL_lo / B_PL_lo).
 *   P_cL [gecc_tl_parity_rows(n) x m, ldpcl] fp32 = A_PL B;   P_rL [n x gecc_tl_parity_rows(m), ldprl] fp32 = A B_PL^T
 *        (PAPER.md:121-127 per block; 16-byte aligned, leading dimensions multiples of 4).
 *   Thresholds of a block of r rows and c columns: `tau` (HOST, 4 values, used for every block) or, with tau NULL, the
 *   automatic ones stated under gecc_decode_correct with n -> r, m -> c and sigma_a, sigma_b the RMS of the WHOLE operands
 *   (sumsq_a, sumsq_b from gecc_tl_encode); the energy rule applies per line of the block.
 *   Report: verdict CLEAN (no block flagged) | CORRECTED (every flagged block corrected) | UNCORRECTABLE (some block refused:
 *   it is left as computed, the others are still corrected); n_found = located entries over all blocks in GLOBAL coordinates
 *   (a whole-row fault is listed once per block it was corrected in), the first GECC_TL_MAX_FOUND of them sorted by (kind,
 *   row, col) when n_found <= GECC_TL_MAX_FOUND (else an arbitrary subset, sorted); n_row_flags / n_col_flags summed over the
 *   blocks; max_abs_syndrome over all blocks; tau: thresholds of a full block.
 * The three calls use `workspace` (gecc_workspace_bytes(dtype, n, k, m), zero when first used) like the global code's calls. */
#define GECC_TL_PANEL 128
#define GECC_TL_MAX_FOUND 64
typedef struct {
  int32_t verdict;
  int32_t n_found;
  int32_t n_row_flags, n_col_flags;
  double max_abs_syndrome[4];
  double tau[4];
  gecc_found_t found[GECC_TL_MAX_FOUND];
} gecc_tl_report_t;

/* Rows of the stacked panel parity of an operand with `len` lines: GECC_PAR_ROWS * ceil(len / GECC_TL_PANEL). */
int64_t gecc_tl_parity_rows(int64_t len);

/* Per-panel encoder (PAPER.md:71-113 applied to each panel): reads A and B once (HBM-bound), one launch for both operands.
 * A_lo / B_lo (GECC_F32 only, else NULL): low parts of the operands for 3xTF32, same leading dimensions as A / B.
 * sumsq_a / sumsq_b [1] fp64: sums of squares of the operands (accumulated in the workspace, written by the last block). */
int gecc_tl_encode(int dtype, int64_t n, int64_t k, int64_t m,
                   const void* A, int64_t lda, float* A_lo, void* A_PL, float* A_PL_lo, double* sumsq_a,
                   const void* B, int64_t ldb, float* B_lo, void* B_PL, float* B_PL_lo, double* sumsq_b,
                   void* workspace, size_t workspace_bytes, void* stream);

/* Encoded product of the tile-local grid: C = A B with the per-block detection sums taken in the epilogue
 * and left in `workspace`, P_cL = A_PL B and P_rL = A B_PL^T.  inject: as for gecc_matmul_protected. */
int gecc_tl_matmul(int dtype, int64_t n, int64_t k, int64_t m,
                   const void* A, int64_t lda, const void* A_PL, const float* A_lo, const float* A_PL_lo,
                   const void* B, int64_t ldb, const void* B_PL, const float* B_lo, const float* B_PL_lo,
                   float* C, int64_t ldc, float* P_rL, int64_t ldprl, float* P_cL, int64_t ldpcl,
                   const gecc_fault_t* inject, int n_inject, void* workspace, size_t workspace_bytes, void* stream);

/* Detection and correction block by block (PAPER.md:186-233 on each block), in place, no host round trip.
 * mode: must be 0 (GECC_SINGLE_CHECKSUM is not offered per block: GECC_EUNSUPPORTED).  report: DEVICE. */
int gecc_tl_decode(int dtype, int64_t n, int64_t k, int64_t m, float* C, int64_t ldc,
                   const float* P_rL, int64_t ldprl, const float* P_cL, int64_t ldpcl,
                   const double* tau, const double* sumsq_a, const double* sumsq_b, int mode,
                   gecc_tl_report_t* report, void* workspace, size_t workspace_bytes, void* stream);

/* Diagnostic (synchronous, HOST output): nanoseconds the last gecc_decode_correct on this workspace spent between
 * its consecutive grid-wide phase boundaries (syndromes | decision | verification ... | patch), from %globaltimer.
 * Returns the number of intervals written to phase_ns (<= max_phases) or a negative gecc_status_t. */
int gecc_decode_phase_ns(int dtype, int64_t n, int64_t k, int64_t m, const void* workspace, size_t workspace_bytes,
                         double* phase_ns, int max_phases);

/* Test / experiment hook: add kind-0 faults to A and kind-1 faults to B in place (E1 / E2), as the
 * operand dtype stores them (bf16: round-to-nearest-even of a + e; fp32: a + e, re-split into hi / lo).  Call it
 * AFTER gecc_encode.  faults: DEVICE pointer; positions are those of the operand (i, l) / (l, j) whatever the storage. */
int gecc_inject_inputs(int dtype, int trans_a, int trans_b, void* A, int64_t lda, float* A_lo, void* B, int64_t ldb, float* B_lo,
                       const gecc_fault_t* faults, int n_faults, void* stream);

/* Library version string (static storage). */
const char* gecc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* GECC_H_ */
