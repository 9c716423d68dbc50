// Internal declarations shared by the translation units of libgecc (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdio>
#include <cstdint>

#include "../../include/gecc.h"

namespace gecc {

// Blocking of the detection sums (must agree between the GEMM epilogue, the unfused pass and the decoder):
// row sums are kept per block of kSumCols columns, column sums per block of kSumRows rows, both with weights local
// to the block (0-based); the decoder restores the global weight (block offset + 1) in fp64.
constexpr int kSumCols = 128;
constexpr int kSumRows = 128;

// Noise law of reading R4, fitted to fault-free runs on B200: the standard deviation of a plain syndrome is
//   sigma = c(k) 2^-24 sqrt(k m) sigma_a sigma_b,   c(k) = c_floor + c0 (k / 1024)^(2/3)
// (tensor-core fp32 accumulation truncates, so its error grows faster than sqrt(k)); c0 = 4.5 for bf16 x bf16 and 20 for
// 3xTF32, c_floor = 2.  Thresholds are kappa = 16 sigma (the noise has heavy tails: maxima of 6-8 sigma were measured).
__host__ __device__ inline double noise_coeff(int dtype, double k) {
  return 2.0 + (dtype == GECC_BF16 ? 4.5 : 20.0) * pow(k / 1024.0, 2.0 / 3.0);
}
constexpr double kKappa = 16.0;

// Encoder blocking (column-direction reduction): rows per partial.
constexpr int kEncMinChunkRows = 64;  // the chunk is a multiple of this, chosen per launch (enc_chunk_rows)
constexpr int kRecompRows = 32;        // row recomputation of the decoder: rows of B per partial
constexpr int kMaxInputFaults = 4;
constexpr int kMaxPointsPerLine = 4;  // a line with more located symbols than this is reported as a whole-line fault
constexpr int kMaxPoints = 2 * kMaxPointsPerLine;
// Repair of an input fault's footprint (reading R20): subtraction is enough when the rounding it leaves behind,
// about (k / 16) 2^-24 |footprint|, stays below this fraction of the RMS of C; otherwise the line is recomputed.
constexpr double kRepairAccuracy = 1e-4;
constexpr int kMaxKeep = 8;            // symbols of recomputed lines set aside for the second decision

// Self-cleaning arrival counters at the start of the workspace (the workspace must be zero when first used; every
// kernel that counts on one leaves it zero again).
constexpr int kCounterBytes = 4096;
constexpr int kCtrEncStrip = 0;     // [0, 512): one per column strip of the column-direction encoder
constexpr int kCtrEncAll = 512;     // last block of a column-direction encoder launch
constexpr int kCtrEncAllRow = 514;  // last block of a row-direction encoder launch (its own slot and partials: the two directions may run concurrently)
constexpr int kEncRowPartBytes = 65536;  // row-direction sum-of-squares partials: one double per block
constexpr int kCtrGemmTile = 513;   // dynamic tile scheduler of the product (reserved)
constexpr int kCtrDecBar = 520;     // decoder: grid barrier arrivals
constexpr int kCtrDecExit = 521;    // decoder: blocks that have left (the last one cleans up)
constexpr int kCtrDecS = 522;       // decoder: flagged rows, flagged columns
constexpr int kCtrDecT = 523;
constexpr int kCtrDecWork = 519;    // decoder: dynamic work counter of the verification pass over B
constexpr int kCtrDecS2 = 532;      // decoder: flagged rows, flagged columns after the repair (second decision)
constexpr int kCtrDecT2 = 533;
constexpr int kCtrBusy = 536;       // kernels of the whole path currently inside this workspace (must never exceed one: see ws_enter)
constexpr int kCtrBusyExit = 537;   // blocks of that kernel that have finished (the last one leaves the workspace)
constexpr int kCtrDecGo = 534;      // decoder: block 0's word to the others after a decision without verification (1: done, 2: verify)
constexpr int kCtrTlArrive = 540;   // tile-local encoder: blocks arrived
constexpr int kCtrTlSumsq = 544;    // tile-local encoder: two fp64 accumulators (sum of squares of A, of B), 8-byte aligned
constexpr int kCtrDecMax = 524;     // decoder: 4 x 64-bit maxima of |syndrome| (bit patterns of non-negative doubles), 8-byte aligned

struct InputFault {
  int32_t row, col;  // position in the operand as stored (A: i, l;  B: l, j)
  double e;
};

// Device-side state of one decode, lives in the workspace.
struct DecodeState {
  // 1: the protected product itself folded the partial sums: syndromes, extra tolerances, flags, the early lists `el`,
  // the flag counts (n_row_flags0 / n_col_flags0), the maxima and the thresholds below are in place and the decoder skips
  // its own first phase.  0: only the partial sums are there (unfused pass, or a product run without thresholds).
  int syn_status;
  int single;               // the flags were taken in single-checksum mode
  double tau[4];            // r1, r2, q1, q2
  double sigma_a, sigma_b;  // RMS of the operands (from sumsq)
  double sigma_c2;          // expected energy of one symbol of C: k sigma_a^2 sigma_b^2 (0 if unknown)
  double maxabs[4];
  int n_row_flags, n_col_flags;
  int n_row_flags0, n_col_flags0;  // before any repair (reported)
  // plan of the Level-P decision
  int verdict;
  int need_verify;  // level 1: Level-P saw a whole-line fault or gave up
  int rows_short;   // orientation of the plan: 1 = errors confined to <= 2 rows (use column syndromes)
  int nS;
  int S[2];
  int whole_line[2];
  int n_points;
  int pt_s[kMaxPoints], pt_l[kMaxPoints];  // short-side / long-side index of each point
  double pt_x[kMaxPoints];
  int n_found;
  gecc_found_t found[GECC_MAX_FOUND];
  // a faulty parity symbol of C_bar (classified by the global parity): kind (-1: none), line, check, magnitude
  int par_kind, par_line, par_c, pad_par;
  double par_delta;
  // Level-X
  int verify_ok_a, verify_ok_b;
  int n_fa, n_fb;
  InputFault fa[kMaxInputFaults], fb[kMaxInputFaults];
  int repaired;  // input faults were found and removed; the second decision accepts CLEAN / points only
  // lines of A / B whose recomputed checks differ from the stored ones (filled by the whole grid, unordered)
  int cnt_a, cnt_b;
  struct Cand { int32_t l, pad_; double d1, d2; } ca[kMaxInputFaults], cb[kMaxInputFaults];
  // line recomputation (one step per faulty row of A / column of B): sums of what the line holds afterwards, its exact
  // parity, and the symbols whose recomputed value was not written because it differs by more than rounding
  double acc[2 * kMaxInputFaults][2], par[2 * kMaxInputFaults][2];
  double accad[2 * kMaxInputFaults];  // sum of |footprint| removed along the line (subtract mode: sizes the line's own tolerance)
  int n_keep, pad_keep;
  // the first (up to 8) flagged lines of each side (rows, columns) with their syndromes and thresholds, in no particular
  // order: written by the blocks that flag them, so that a decision about few lines need not search the flags
  struct Early { int32_t idx[8]; double a1[8], a2[8], t1[8], t2[8]; } el[2];
  struct Keep { int32_t is_row, line, t, pad_; double v; } keep[kMaxKeep];
};

// Per-block results of the syndrome phase of the decoder (no atomics: summed in block order afterwards).
struct BlockStat {
  int row_flags, col_flags;
  double maxabs[4];
};
constexpr int kMaxDecodeBlocks = 1024;

#ifdef __CUDACC__
// The workspace serves ONE call at a time (include/gecc.h: calls that share a workspace must be ordered on one stream): its
// arrival counters and accumulators would silently fold contributions of two products into each other.  The kernels of
// the whole path therefore count themselves in and out; a second kernel entering while another is inside (two streams on
// one workspace) stops the context with a message instead of returning a wrong product.  ws_enter: one thread, after
// griddepcontrol.wait (the predecessor in the stream has left by then).  ws_exit: one thread per block, when the block is done.
__device__ inline void ws_enter(unsigned int* counters, const char* who) {
  if (atomicAdd(counters + kCtrBusy, 1u) != 0u) {
    printf("gecc: %s entered a workspace that another call is using (calls sharing a workspace must be ordered on one stream)\n", who);
    __trap();
  }
}
__device__ inline void ws_exit(unsigned int* counters, unsigned int nblocks) {
  __threadfence();
  if (atomicAdd(counters + kCtrBusyExit, 1u) == nblocks - 1u) {
    counters[kCtrBusyExit] = 0;
    __threadfence();
    atomicExch(counters + kCtrBusy, 0u);
  }
}
#endif

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Rows per partial of the column-direction reduction: the smallest multiple of 64 for which strips x chunks fits ONE block
// per SM (the other block slot of every SM is left to the second operand, which gecc_encode_both encodes in the same
// launch; fewer, fatter blocks also amortise the per-block fold).  The encoders and the decoder's verification pass must
// use the same value: it fixes the order of the sums.
inline int enc_chunk_rows(int64_t rows, int64_t strips, int sms) {
  const int64_t groups = (rows + kEncMinChunkRows - 1) / kEncMinChunkRows;
  const int64_t slots = sms > 0 ? (int64_t)sms : 148;
  // as many chunks per strip as keep strips x chunks within the slots (a second, partly filled wave costs up to half the
  // kernel again), of equal height
  int64_t chunks_max = slots / (strips > 0 ? strips : 1);
  if (chunks_max < 1) chunks_max = 1;
  int64_t per = (groups + chunks_max - 1) / chunks_max;
  if (per < 1) per = 1;
  return (int)(per * kEncMinChunkRows);
}

// Encoder scratch, a function of the operand's storage shape only (gecc_encode does not know the product's shape).
struct EncLayout {
  size_t sumsq_part;  // double [blocks]
  size_t encpart;     // double [chunks][2][cols]   (column-direction reduction only)
  size_t total;
};
inline EncLayout enc_layout(int64_t rows, int64_t cols) {
  EncLayout e;
  const int64_t chunks = (rows + kEncMinChunkRows - 1) / kEncMinChunkRows;  // upper bound on the chunks of any launch
  const int64_t strips = (cols + 127) / 128;  // >= strips of either dtype
  const int64_t nparts = (strips * chunks > (rows + 7) / 8 ? strips * chunks : (rows + 7) / 8) + 1;  // >= blocks of either kernel
  size_t off = kCounterBytes + kEncRowPartBytes;  // the row-direction partials sit at a fixed place right after the counters
  e.sumsq_part = off; off = align_up(off + (size_t)nparts * sizeof(double), 256);
  e.encpart = off; off = align_up(off + (size_t)chunks * 2 * cols * sizeof(double), 256);
  e.total = off;
  return e;
}

struct WsLayout {
  size_t encpart_b;         // double [chunks(m)][2][k]: decoder's verification pass over B^T
  size_t enc;               // counters + encoder scratch (EncLayout offsets are relative to the workspace base)
  size_t rowpart, colpart;  // float4 per (column block, row) / (row block, column): sum, local-weighted sum, sum of squares, 0
  size_t syn;               // double r1[n], r2[n], q1[m], q2[m], then the same four again: extra tolerance per line
  size_t flags;             // uint8 rflag[align16(n)], qflag[align16(m)]
  size_t votes;             // int [max(n, m)]
  size_t lists;             // per side (rows, then columns): int idx[len], double a1[len], a2[len], t1[len], t2[len]
  size_t ver64;             // double [2][k] (A), [2][k] (B)
  size_t recomp;            // double [ceil(k / kRecompRows)][max(n, m)]: partials of a line recomputation (also holds the weight vector of the dot form)
  size_t blockstat;         // BlockStat [kMaxDecodeBlocks] (reserved by the global decoder); the tile-local decoder keeps its TlState here
  size_t state;             // DecodeState
  size_t timing;            // unsigned long long [kMaxPhaseStamps]: %globaltimer at the decoder's phase boundaries (diagnostic)
  size_t lineacc;           // double [n + m][4]: per-line sums accumulated by the product's epilogues when it detects itself (self-cleaning)
  size_t arrive;            // unsigned int [nrb + ncb + 4]: blocks of each 128-row / 128-column strip completed by the product (self-cleaning), folds done
  size_t total;
};
constexpr int kMaxPhaseStamps = 64;

inline WsLayout ws_layout(int dtype, int64_t n, int64_t k, int64_t m) {
  (void)dtype;
  WsLayout w;
  const int64_t ncb = (m + kSumCols - 1) / kSumCols, nrb = (n + kSumRows - 1) / kSumRows;
  // encoder region: large enough for gecc_encode on either operand in either storage (A: n x k or k x n, B: k x m or
  // m x k) and for the decoder's reuse of the scratch (chunk partials of the verification pass over A from A's offset)
  size_t pmax = 0, xmax = 0;
  const int64_t shp[4][2] = {{n, k}, {k, n}, {k, m}, {m, k}};
  for (int s = 0; s < 4; ++s) {
    const EncLayout e = enc_layout(shp[s][0], shp[s][1]);
    const size_t pp = e.encpart - e.sumsq_part, xx = e.total - e.encpart;
    if (pp > pmax) pmax = pp;
    if (xx > xmax) xmax = xx;
  }
  size_t off = 0;
  w.enc = off; off = align_up(kCounterBytes + kEncRowPartBytes + pmax + xmax, 256);
  // the verification pass over a transposed B (stored m x k) runs beside the one over A: its own chunk partials
  w.encpart_b = off; off = align_up(off + (size_t)((m + kEncMinChunkRows - 1) / kEncMinChunkRows) * 2 * k * sizeof(double), 256);
  w.rowpart = off; off = align_up(off + (size_t)ncb * n * 4 * sizeof(float), 256);
  w.colpart = off; off = align_up(off + (size_t)nrb * m * 4 * sizeof(float), 256);
  w.syn = off; off = align_up(off + (size_t)(4 * n + 4 * m) * sizeof(double), 256);
  w.flags = off; off = align_up(off + align_up((size_t)n, 16) + align_up((size_t)m, 16), 256);
  w.votes = off; off = align_up(off + (size_t)(n > m ? n : m) * sizeof(int), 256);
  w.lists = off; off = align_up(off + (size_t)(n + m) * (sizeof(int) + 4 * sizeof(double)) + 64, 256);
  w.ver64 = off; off = align_up(off + (size_t)4 * k * sizeof(double), 256);
  {
    const size_t a = (size_t)((k + kRecompRows - 1) / kRecompRows) * (n > m ? n : m) * sizeof(double), b = (size_t)k * sizeof(double);
    w.recomp = off; off = align_up(off + (a > b ? a : b), 256);
  }
  w.blockstat = off; off = align_up(off + sizeof(BlockStat) * kMaxDecodeBlocks, 256);
  w.state = off; off = align_up(off + sizeof(DecodeState), 256);
  w.timing = off; off = align_up(off + sizeof(unsigned long long) * kMaxPhaseStamps, 256);
  w.lineacc = off; off = align_up(off + (size_t)(n + m) * 4 * sizeof(double), 256);
  w.arrive = off; off = align_up(off + (size_t)(nrb + ncb + 4) * sizeof(unsigned int), 256);
  w.total = off;
  return w;
}

int num_sms();

// gemm_sm100.cu
// Where the protected product leaves the results of its own detection step (all inside the workspace, except `report`).
struct DetectArgs {
  bool detect;             // thresholds are known: fold the partial sums inside the product
  bool single;             // GECC_SINGLE_CHECKSUM
  const double* tau;       // HOST, 4 thresholds, or null: automatic from sumsq_a / sumsq_b (device)
  const double* sumsq_a;
  const double* sumsq_b;
  double* syn;
  uint8_t* flags;
  DecodeState* st;
  unsigned int* counters;
  unsigned int* arrive;
  double* lineacc;
  gecc_report_t* report;   // device, may be null
};
// Tile-local grid (gecc_tl_matmul): A_par / B_par of gemm_dispatch then hold the stacked panel parity A_PL [rows_a x k] / B_PL
// [rows_b x k] (K-major, 8 rows per panel of 128 lines), and the parity products land in PcL = A_PL B [rows_a x m] and
// PrL = A B_PL^T [n x rows_b] instead of P_r / P_c / P_g.
struct TlArgs {
  int64_t rows_a, rows_b;
  float* PcL;
  int64_t ldpcl;
  float* PrL;
  int64_t ldprl;
};
int gemm_dispatch(bool protect, int dtype, int64_t n, int64_t k, int64_t m, bool trans_a, bool trans_b, const void* A, int64_t lda, const void* A_par, const float* A_lo,
                  const float* A_par_lo, const void* B, int64_t ldb, const void* B_par, const float* B_lo, const float* B_par_lo, float* C,
                  int64_t ldc, float* P_r, float* P_c, float* P_g, const gecc_fault_t* inject, int n_inject, float* rowpart, float* colpart,
                  const DetectArgs* det, bool pdl, cudaStream_t stream, const TlArgs* tla = nullptr);

// syndrome.cu
int syndrome_unfused_dispatch(int64_t n, int64_t m, const float* C, int64_t ldc, float* rowpart, float* colpart, DecodeState* st, cudaStream_t stream);

// encode.cu: the two checks of one operand.  reduce_over_rows = true: out[c] = sum over storage rows (len = cols);
// false: out[r] = sum along each storage row (len = rows).  ws: workspace base (counters + EncLayout scratch).
int encode_dispatch(int dtype, bool reduce_over_rows, const void* X, int64_t rows, int64_t cols, int64_t ld, void* parity, float* parity_lo,
                    float* x_lo, double* par64, double* sumsq, uint8_t* ws, cudaStream_t stream);
int encode_noalloc_dispatch(int dtype, bool reduce_over_rows, const void* X, int64_t rows, int64_t cols, int64_t ld, void* parity, float* parity_lo,
                            float* x_lo, double* par64, double* sumsq, cudaStream_t stream);

int encode_both_dispatch(int dtype, bool a_over_rows, bool b_over_rows, const void* A, int64_t ra, int64_t ca, int64_t lda, void* A_par, float* A_par_lo, float* A_lo,
                         double* A_par64, double* sumsq_a, const void* B, int64_t rb, int64_t cb, int64_t ldb, void* B_par, float* B_par_lo, float* B_lo,
                         double* B_par64, double* sumsq_b, uint8_t* ws, double* encpart_b, cudaStream_t stream);

}  // namespace gecc
