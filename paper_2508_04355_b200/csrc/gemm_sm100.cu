// Encoded product C_bar = A_bar B_bar as one persistent, warp-specialised tcgen05 kernel run by CTA
// PAIRS (cluster of 2, cta_group::2): one tcgen05.mma covers a 256 x N tile, each CTA holding 128 rows of A and half of
// the B tile in its shared memory, so every operand byte is fetched from L2 once per pair.
//
//   warp 0 lane 0 : TMA producer   (global -> 128B-swizzled shared tiles; both CTAs' bytes are counted on the leader's barrier)
//   warp 1 lane 0 : MMA issuer     (leader CTA only; accumulators in TMEM, two buffers of 256 columns in each CTA)
//   warp 2        : TMEM allocator
//   warps 4..7    : epilogue       (TMEM -> registers -> shared -> coalesced global stores) of the CTA's own 128 rows, with
//                                   the row and column sums of the detection step taken from the
//                                   accumulators on the way out, so C is never read back.
//
// The parity rows A_P and parity columns B_P are not copied next to A and B: they live in side buffers
// ([GECC_PAR_ROWS x k], K-major) and enter the product as extra, cheap tiles with N = 16:
//   PR tile: rows of A      x B_P   -> P_r
//   PC tile: columns of B^T x A_P   -> P_c^T (operands swapped so that the 8 parity rows are the N side)
//   PG tile: A_P            x B_P   -> P_g
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <type_traits>

#include "../../include/gecc.h"
#include "fold.cuh"
#include "gecc_internal.h"
#include "sm100_ptx.cuh"

namespace gecc {

using namespace ptx;

template <int KIND>
struct Cfg;
template <>
struct Cfg<GECC_BF16> {
  static constexpr int ELT = 2, BK = 64, UK = 16, STAGES = 6;
  static constexpr uint32_t FMT = FMT_BF16;
};
template <>
struct Cfg<GECC_F32> {
  static constexpr int ELT = 4, BK = 32, UK = 8, STAGES = 3;
  static constexpr uint32_t FMT = FMT_TF32;
};

constexpr int BM = 128;    // rows of A per CTA (256 per pair)
constexpr int BN = 256;    // columns of a full data tile (each CTA stages 128 of them)
constexpr int PARN = 16;   // UMMA N of the parity tiles (8 real columns, duplicated by the peer CTA)
constexpr int NUM_THREADS = 256;
constexpr int EPI_WARP0 = 4;
constexpr int STAGE_EPI_BYTES = 4 * 32 * 32 * 4;  // 4 warps x (32 rows x 32 fp32)

// TILE_PCL / TILE_PRL: parity products of the tile-local grid (one code per 128 x 128 block of C, gecc_tl_*): the stacked panel
// parity A_PL [8 n/128 x k] times B, and A times the stacked B_PL [8 m/128 x k]^T, computed as ordinary data-sized tiles.
enum TileKind { TILE_DATA = 0, TILE_PC = 1, TILE_PR = 2, TILE_PG = 3, TILE_PCL = 4, TILE_PRL = 5 };

template <int KIND>
struct Smem {
  using C = Cfg<KIND>;
  static constexpr int NOPS = (KIND == GECC_F32) ? 2 : 1;     // hi and lo planes of each operand for 3xTF32
  static constexpr int A_BYTES = BM * 128;                    // 128 rows x 128 B (one swizzle row = BK elements)
  static constexpr int B_BYTES = (BN / 2) * C::BK * C::ELT;   // this CTA's half of the B tile
  static constexpr int STAGE_BYTES = NOPS * (A_BYTES + B_BYTES);
  static constexpr int PIPE_BYTES = C::STAGES * STAGE_BYTES;
  static constexpr int COLACC_BYTES = 4 * BN * 3 * 4;  // column sums of the four epilogue warps: [warp][column][sum, weighted, squares]
  static constexpr int TOTAL = 1024 /*alignment slack*/ + PIPE_BYTES + STAGE_EPI_BYTES + COLACC_BYTES + 256 /*barriers*/;
};

struct GemmParams {
  int n, k, m;
  int mbp, nbp;          // row-block pairs (256 rows) and column blocks (256 columns) of the data part
  int n_full, n_split;   // data units computed as one 256-wide tile / as two 128-wide tiles (tail balancing)
  int gh;                // data units are numbered in bands of gh row-block pairs (see unit_coords)
  int num_items;         // all tiles, in scheduling order: full, halves, PC, PR, PG
  int n_data_units;      // data units (mbp x nbp); units beyond them are the tile-local parity units (tl != 0)
  int tl;                // tile-local grid: parity units PCL (tl_rb row-block pairs of A_PL x nbp) and PRL (mbp x tl_cb column blocks of B_PL), no PC / PR / PG
  int tl_rb, tl_cb;
  int tl_rows_a, tl_rows_b;  // rows of A_PL / B_PL (8 per panel)
  float* PcL;            // [tl_rows_a x m], leading dimension ldpcl
  float* PrL;            // [n x tl_rows_b], leading dimension ldprl
  int64_t ldpcl, ldprl;
  int protect;           // 1: parity tiles + epilogue sums
  int a_mn, b_mn;        // operand layouts in memory: a_mn = 1: A stored transposed (k x n, M contiguous); b_mn = 1: B stored k x m (N contiguous, the default), 0: B stored transposed (m x k)
  float* C;
  int64_t ldc;
  float* P_r;      // [n x GECC_PR_LD]
  float* P_c;      // [GECC_PAR_ROWS x m]
  float* P_g;      // [GECC_PAR_ROWS x GECC_PR_LD]
  float* rowpart;  // [m / 128][n][4] : per row, per block of 128 columns: sum_j c, sum_j jl c, sum_j c^2, 0   (jl = column within the block)
  float* colpart;  // [n / 128][m][4] : per column, per block of 128 rows: sum_i c, sum_i il c, sum_i c^2, 0 (il = row within the block)
  const gecc_fault_t* inject;
  int n_inject;
  // Detection inside the product: the CTA that completes the last block of a 128-row / 128-column strip
  // (data tiles and the strip's parity tile alike) folds the strip's partial sums into syndromes and flags; the CTA that
  // completes the last strip writes the flag counts, and the CLEAN report if nothing is flagged.
  int detect;
  int nrb128, ncb128;      // strips of 128 rows / 128 columns
  FoldBufs fb;
  ThresholdSpec ts;
  DecodeState* st;
  unsigned int* counters;  // workspace base: kCtrDec* slots
  unsigned int* arrive;    // [nrb128] row strips, [ncb128] column strips, [1] folds done
  double* lineacc;         // [n + m][4]: sum c, sum (index + 1) c, sum c^2 of every row, then of every column (fp64 accumulators, self-cleaning)
  gecc_report_t* report;   // may be null
};

struct Tile {
  int kind;
  int row0;   // first row of the pair's 256 rows (DATA, PR) / first column of the pair's 256 columns (PC)
  int col0;   // first column (DATA)
  int ncols;  // UMMA N: 256 or 128 (DATA), 16 (parity tiles)
};

// Scheduling order: full-width data tiles, then the half-width tiles of the last `n_split` units, then the parity tiles.
// Data units are numbered in bands of gh row-block pairs (gh = all of them while the operands fit in L2), column block major inside a band (unit -> band, then column
// block, then row-block pair): the pairs working at the same time then cover about gh row blocks x (pairs / gh) column
// blocks, so a wave re-reads gh + pairs / gh operand panels instead of mbp + pairs / mbp -- what keeps the operands of
// products much larger than L2 (8192 and up) from streaming out of HBM once per column block.
__device__ __forceinline__ void unit_coords(const GemmParams& p, int u, int& rb, int& cb) {
  const int per = p.gh * p.nbp, g = u / per, r = u - g * per;
  const int left = p.mbp - g * p.gh, h = left < p.gh ? left : p.gh;  // row-block pairs in this band
  cb = r / h;
  rb = g * p.gh + (r - cb * h);
}
// Tile-local grid: parity unit e (counted from the end of the data units) as a full-width tile -- PCL: rows row0.. of A_PL x
// columns col0.. of B; PRL: rows row0.. of A x rows col0.. of B_PL.  Out of line: the data path of decode_item stays as small
// as it was (the producer and MMA warps evaluate it between tiles).
__device__ __noinline__ void tl_unit_tile(const GemmParams& p, int e, Tile& tl) {
  const int npcl = p.tl_rb * p.nbp;
  if (e < npcl) { tl.kind = TILE_PCL; tl.row0 = (e / p.nbp) * 2 * BM; tl.col0 = (e % p.nbp) * BN; return; }
  e -= npcl;
  tl.kind = TILE_PRL; tl.row0 = (e / p.tl_cb) * 2 * BM; tl.col0 = (e % p.tl_cb) * BN;
}
__device__ __forceinline__ Tile decode_item(const GemmParams& p, int t) {
  Tile tl;
  int rb, cb;
  if (t < p.n_full) {
    if (t >= p.n_data_units) { tl_unit_tile(p, t - p.n_data_units, tl); tl.ncols = BN; return tl; }
    unit_coords(p, t, rb, cb);
    tl.kind = TILE_DATA; tl.row0 = rb * 2 * BM; tl.col0 = cb * BN; tl.ncols = BN;
    return tl;
  }
  t -= p.n_full;
  if (t < 2 * p.n_split) {
    const int u = p.n_full + (t >> 1);
    if (u >= p.n_data_units) { tl_unit_tile(p, u - p.n_data_units, tl); tl.col0 += (t & 1) * (BN / 2); tl.ncols = BN / 2; return tl; }
    unit_coords(p, u, rb, cb);
    tl.kind = TILE_DATA; tl.row0 = rb * 2 * BM; tl.col0 = cb * BN + (t & 1) * (BN / 2); tl.ncols = BN / 2;
    return tl;
  }
  t -= 2 * p.n_split;
  tl.ncols = PARN; tl.col0 = 0;
  if (t < p.nbp) { tl.kind = TILE_PC; tl.row0 = t * BN; return tl; }
  t -= p.nbp;
  if (t < p.mbp) { tl.kind = TILE_PR; tl.row0 = t * 2 * BM; return tl; }
  tl.kind = TILE_PG; tl.row0 = 0;
  return tl;
}

// ------------------------------------------------------------------------------------------------
// In-product detection.  Called by the 128 epilogue threads of a CTA at the end of a tile's epilogue, after the tile's
// partial sums / parity symbols were stored: counts the tile's blocks on the arrival counters of the strips it touched
// and folds every strip this CTA completed (one thread per line).  `flags_smem`: three words of shared memory.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void epi_bar() { asm volatile("bar.sync 1, 128;" ::: "memory"); }

// Folds up to three strips this CTA completed (one thread per line of each strip).  The loads of all of them are issued before the
// first line is finished: a CTA that completes its last tile folds a row strip and two column strips, and these folds are on the
// kernel's critical path (nothing is left to hide them behind).
__device__ __noinline__ void fold_strips(const GemmParams& p, int nst, const bool (&is_row_)[3], const int (&strip_)[3], int tid) {
  Thresholds th;
  make_thresholds(p.ts, p.n, p.k, p.m, th);
  const int lane = tid & 31;
  float pv[3][6];
  double2 ab[3], en[3];
  bool live[3];
  int64_t idx[3];
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    live[s] = false; idx[s] = 0;
    ab[s] = make_double2(0.0, 0.0); en[s] = ab[s];
    if (s < nst) {
      const bool is_row = is_row_[s];
      idx[s] = (int64_t)strip_[s] * 128 + tid;
      live[s] = idx[s] < (is_row ? p.n : p.m);
      if (live[s]) {
        // the line's sums were accumulated by the epilogues of every tile that holds a piece of it (fp64 additions of fp32
        // partial sums: exact, hence independent of their order); taken and left zero for the next product
        load_parity(p.fb, is_row, idx[s], pv[s]);
        double2* acc = reinterpret_cast<double2*>(p.lineacc + ((is_row ? 0 : (int64_t)p.n) + idx[s]) * 4);
        ab[s] = __ldcg(acc); en[s] = __ldcg(acc + 1);
        acc[0] = make_double2(0.0, 0.0); acc[1] = make_double2(0.0, 0.0);
      }
    }
  }
#pragma unroll
  for (int s = 0; s < 3; ++s) {
    if (s >= nst) break;
    const bool is_row = is_row_[s];
    FoldResult r;
    r.a = 0.0; r.b = 0.0; r.t1 = 0.0; r.t2 = 0.0; r.flagged = false;
    if (live[s]) r = finish_line(p.fb, th, is_row, idx[s], ab[s].x, ab[s].y, en[s].x, pv[s]);
    // the first 8 flagged lines of each side go to the decoder state with their syndromes and thresholds (slots reserved on
    // the grid-wide count, one atomic per warp), so that a decision about few lines never searches the flags
    const int side = is_row ? 0 : 1;
    const unsigned fb = __ballot_sync(0xffffffffu, r.flagged);
    if (fb) {
      const int lead = __ffs(fb) - 1;
      int base = 0;
      if (lane == lead) base = (int)atomicAdd(p.counters + (is_row ? kCtrDecS : kCtrDecT), (unsigned int)__popc(fb));
      base = __shfl_sync(0xffffffffu, base, lead);
      const int slot = base + __popc(fb & ((1u << lane) - 1u));
      if (r.flagged && slot < 8) {
        DecodeState::Early& E = p.st->el[side];
        E.idx[slot] = (int)idx[s]; E.a1[slot] = r.a; E.a2[slot] = r.b; E.t1[slot] = r.t1; E.t2[slot] = r.t2;
      }
    }
    // maxima of |syndrome| (bit patterns of non-negative doubles compare like integers)
    unsigned long long v1 = live[s] ? (unsigned long long)__double_as_longlong(abs_for_max(r.a)) : 0ull;
    unsigned long long v2 = live[s] ? (unsigned long long)__double_as_longlong(abs_for_max(r.b)) : 0ull;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const unsigned long long w1 = __shfl_xor_sync(0xffffffffu, v1, o), w2 = __shfl_xor_sync(0xffffffffu, v2, o);
      v1 = w1 > v1 ? w1 : v1;
      v2 = w2 > v2 ? w2 : v2;
    }
    if (lane == 0) {
      unsigned long long* gmax = reinterpret_cast<unsigned long long*>(p.counters + kCtrDecMax) + (is_row ? 0 : 2);
      if (v1) atomicMax(gmax, v1);
      if (v2) atomicMax(gmax + 1, v2);
    }
  }
}

// The thread that completed the last strip: every line is folded.  Moves the counts and maxima into the decoder state
// (leaving the counters clean for the next product), and settles a fault-free product at once: verdict CLEAN
// (PAPER.md:215 with both sets empty), report written, no decoder pass needed.
__device__ __noinline__ void fold_finalize(const GemmParams& p) {
  __threadfence();
  Thresholds th;
  make_thresholds(p.ts, p.n, p.k, p.m, th);
  DecodeState* st = p.st;
  const int s = (int)__ldcg(p.counters + kCtrDecS), t = (int)__ldcg(p.counters + kCtrDecT);
  unsigned long long* gmax = reinterpret_cast<unsigned long long*>(p.counters + kCtrDecMax);
  double mx[4];
  for (int q = 0; q < 4; ++q) { mx[q] = __longlong_as_double((long long)__ldcg(gmax + q)); gmax[q] = 0ull; }
  p.counters[kCtrDecS] = 0; p.counters[kCtrDecT] = 0;
  p.arrive[p.nrb128 + p.ncb128] = 0;
  st->n_row_flags0 = s; st->n_col_flags0 = t;
  st->n_row_flags = s; st->n_col_flags = t;
  for (int q = 0; q < 4; ++q) { st->maxabs[q] = mx[q]; st->tau[q] = th.tau[q]; }
  st->sigma_a = th.sigma_a; st->sigma_b = th.sigma_b; st->sigma_c2 = th.sigma_c2;
  st->single = th.single;
  if (s == 0 && t == 0) {
    st->verdict = GECC_CLEAN; st->n_found = 0;
    if (p.report) {
      gecc_report_t* r = p.report;
      r->verdict = GECC_CLEAN; r->n_found = 0; r->n_row_flags = 0; r->n_col_flags = 0;
      for (int q = 0; q < 4; ++q) { r->max_abs_syndrome[q] = mx[q]; r->tau[q] = th.tau[q]; }
      for (int a = 0; a < GECC_MAX_FOUND; ++a) r->found[a] = gecc_found_t{-1, -1, -1, 0, 0.0};
    }
  }
  __threadfence();
  st->syn_status = 1;
  __threadfence();
}

// row_strip / col_strip*: the strips this CTA's tile contributed to (-1: none) and how many blocks it contributed.
__device__ __noinline__ void detect_tail(const GemmParams& p, int row_strip, int row_cnt, int col_strip0, int col_strip1, uint32_t flags_smem, int tid) {
  epi_bar();  // every epilogue thread has stored its partial sums / parity symbols
  if (tid == 0) {
    __threadfence();  // ... and they are visible before the arrival is counted
    unsigned int last = 0;
    // the (up to) three arrivals are issued together, their answers examined afterwards: one round trip, not three
    unsigned int* c0 = p.arrive + (row_strip >= 0 ? row_strip : 0);
    unsigned int* c1 = p.arrive + p.nrb128 + (col_strip0 >= 0 ? col_strip0 : 0);
    unsigned int* c2 = p.arrive + p.nrb128 + (col_strip1 >= 0 ? col_strip1 : 0);
    unsigned int o0 = 0, o1 = 0, o2 = 0;
    if (row_strip >= 0) o0 = atomicAdd(c0, (unsigned int)row_cnt);
    if (col_strip0 >= 0) o1 = atomicAdd(c1, 1u);
    if (col_strip1 >= 0) o2 = atomicAdd(c2, 1u);
    if (row_strip >= 0 && o0 + row_cnt == (unsigned int)p.ncb128 + 1u) { *c0 = 0; last |= 1u; }
    if (col_strip0 >= 0 && o1 + 1u == (unsigned int)p.nrb128 + 1u) { *c1 = 0; last |= 2u; }
    if (col_strip1 >= 0 && o2 + 1u == (unsigned int)p.nrb128 + 1u) { *c2 = 0; last |= 4u; }
    __threadfence();
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(flags_smem), "r"(last) : "memory");
  }
  epi_bar();
  unsigned int last;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(last) : "r"(flags_smem) : "memory");
  if (!last) return;
  int nf = 0;
  bool fr[3] = {false, false, false};
  int fs[3] = {0, 0, 0};
  if (last & 1u) { fr[nf] = true; fs[nf] = row_strip; ++nf; }
  if (last & 2u) { fr[nf] = false; fs[nf] = col_strip0; ++nf; }
  if (last & 4u) { fr[nf] = false; fs[nf] = col_strip1; ++nf; }
  fold_strips(p, nf, fr, fs, tid);
  epi_bar();
  if (tid == 0) {
    __threadfence();
    const unsigned int old = atomicAdd(p.arrive + p.nrb128 + p.ncb128, (unsigned int)nf);
    if (old + nf == (unsigned int)(p.nrb128 + p.ncb128)) fold_finalize(p);
  }
}

template <int KIND>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NUM_THREADS, 1)
gecc_gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                 const __grid_constant__ CUtensorMap tmAp, const __grid_constant__ CUtensorMap tmBp,
                 const __grid_constant__ CUtensorMap tmAlo, const __grid_constant__ CUtensorMap tmBlo,
                 const __grid_constant__ CUtensorMap tmAplo, const __grid_constant__ CUtensorMap tmBplo,
                 const __grid_constant__ GemmParams p) {
  using C = Cfg<KIND>;
  using S = Smem<KIND>;
  constexpr int BK = C::BK, STAGES = C::STAGES;
  constexpr int NSW = 128 / C::ELT;                // elements per 128-byte swizzle row
  constexpr int BOX_BYTES = 128 * BK;              // one MN-major box: NSW columns x BK rows of k
  constexpr int PAR_BYTES = GECC_PAR_ROWS * 128;   // one parity box: 8 rows x BK elements, K-major
  constexpr uint32_t TMEM_COLS = 2 * BN;           // two accumulator buffers

  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t epi_base = smem_base + S::PIPE_BYTES;
  const uint32_t colacc_base = epi_base + STAGE_EPI_BYTES;
  const uint32_t bar_base = colacc_base + S::COLACC_BYTES;
  // barriers: full[STAGES], empty[STAGES], tmem_full[2], tmem_empty[2], then the TMEM base address word
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
  auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + a); };
  auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + 2 + a); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 4);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();  // 0 = leader (issues the MMAs), 1 = peer
  const int pair = blockIdx.x >> 1, npairs = gridDim.x >> 1;
  const int kblocks = (p.k + BK - 1) / BK;

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmA);
    prefetch_tmap(&tmB);
    if (p.protect) { prefetch_tmap(&tmAp); prefetch_tmap(&tmBp); }
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int a = 0; a < 2; ++a) { mbar_init(tfull_bar(a), 1); mbar_init(tempty_bar(a), 8); }  // 4 epilogue warps x 2 CTAs
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc_pair(tmem_slot, TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  cluster_sync();  // both CTAs' barriers are initialised before either touches the other's
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
  const uint32_t lastflags = bar_base + 8u * (2 * STAGES + 4) + 16u;

  // Programmatic dependent launch: everything above overlapped the previous kernel's tail (the encoder's, when the
  // caller launched this kernel with that attribute); its results are read only from here on.  The next kernel in the
  // stream (the decoder) may begin to launch at once: it waits for this grid's completion before it reads anything.
  griddep_wait();
  griddep_launch_dependents();
  if (p.protect && blockIdx.x == 0 && threadIdx.x == 0) {
    ws_enter(p.counters, "gecc_matmul_protected");
    if (!p.detect) p.st->syn_status = 0;  // partial sums only
  }

  if (warp == 0) {
    {
      // ================= TMA producer (both CTAs; the whole warp runs the loop, one elected lane issues) =================
      int stage = 0;
      uint32_t phase = 0;
      // One k-loop per combination of operand layouts (K-major: one box; MN-major: boxes of one swizzle row each), so that
      // the path from "stage free" to "loads issued" holds nothing but the wait, the byte count and the loads: the ring is
      // rarely full (a TMA round trip is of the order of the ring's depth), so every instruction here delays the MMAs.
      auto kloop = [&](auto amn_c, auto bmn_c, const CUtensorMap* mA0, const CUtensorMap* mA1, const CUtensorMap* mB0, const CUtensorMap* mB1, int ac, int bc,
                       int bnb, uint32_t tx_bytes) {
        constexpr bool AMN = decltype(amn_c)::value, BMN = decltype(bmn_c)::value;
        for (int kb = 0; kb < kblocks; ++kb) {
          mbar_wait_bounded(empty_bar(stage), phase ^ 1);
          const uint32_t sA = smem_base + stage * S::STAGE_BYTES;
          const uint32_t sB = sA + S::NOPS * S::A_BYTES;
          const uint32_t bar = mapa(full_bar(stage), 0);
          const int k0 = kb * BK;
          if (elect_one()) {
            if (rank == 0) mbar_expect_tx(full_bar(stage), tx_bytes);  // both CTAs' bytes
#pragma unroll
            for (int pl = 0; pl < S::NOPS; ++pl) {  // plane 0: the operands (tf32: hi parts), plane 1: the lo parts
              const CUtensorMap* mA = pl == 0 ? mA0 : mA1;
              const CUtensorMap* mB = pl == 0 ? mB0 : mB1;
              const uint32_t dA = sA + pl * S::A_BYTES, dB = sB + pl * S::B_BYTES;
              if (!AMN) tma_load_2d_pair(dA, mA, bar, k0, ac);
              else {
#pragma unroll
                for (int bx = 0; bx < BM / NSW; ++bx) tma_load_2d_pair(dA + bx * BOX_BYTES, mA, bar, ac + bx * NSW, k0);
              }
              if (!BMN) tma_load_2d_pair(dB, mB, bar, k0, bc);
              else {
                for (int bx = 0; bx < bnb; ++bx) tma_load_2d_pair(dB + bx * BOX_BYTES, mB, bar, bc + bx * NSW, k0);
              }
            }
          }
          __syncwarp();
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      };
      for (int t = pair; t < p.num_items; t += npairs) {
        const Tile tl = decode_item(p, t);
        const int ncta = tl.ncols / 2;  // columns of the B-role operand this CTA stages (data-sized tiles)
        // A role: 128 rows of A (DATA, PR, PRL; MN-major boxes when A is stored transposed), 128 columns of B (PC: MN-major
        // boxes of the row-major B, one K-major box of a transposed B), the parity rows A_P (PG: one box of 8 rows) or 128 rows
        // of the stacked panel parity A_PL (PCL).  B role: this CTA's share of the columns of B (DATA, PCL), the parity rows of
        // the other side (PC: A_P; PR, PG: B_P) or rows of the stacked B_PL (PRL: K-major box of 128, the first ncta are used).
        const CUtensorMap *mA0, *mA1, *mB0, *mB1;
        bool amn, bmn;
        int ac, bc, bnb = 0;
        uint32_t a_bytes = S::A_BYTES, b_bytes;
        if (tl.kind == TILE_DATA || tl.kind == TILE_PR || tl.kind == TILE_PRL) { mA0 = &tmA; mA1 = &tmAlo; amn = p.a_mn != 0; ac = tl.row0 + (int)rank * BM; }
        else if (tl.kind == TILE_PC) { mA0 = &tmB; mA1 = &tmBlo; amn = p.b_mn != 0; ac = tl.row0 + (int)rank * BM; }
        else { mA0 = &tmAp; mA1 = &tmAplo; amn = false; ac = tl.kind == TILE_PCL ? tl.row0 + (int)rank * BM : 0; if (tl.kind == TILE_PG) a_bytes = PAR_BYTES; }
        if (tl.kind == TILE_DATA || tl.kind == TILE_PCL) {
          mB0 = &tmB; mB1 = &tmBlo; bmn = p.b_mn != 0; bc = tl.col0 + (int)rank * ncta; bnb = ncta / NSW;
          b_bytes = bmn ? (uint32_t)(ncta * BK * C::ELT) : (uint32_t)S::B_BYTES;
        } else if (tl.kind == TILE_PC) { mB0 = &tmAp; mB1 = &tmAplo; bmn = false; bc = 0; b_bytes = PAR_BYTES; }
        else if (tl.kind == TILE_PRL) { mB0 = &tmBp; mB1 = &tmBplo; bmn = false; bc = tl.col0 + (int)rank * ncta; b_bytes = S::B_BYTES; }
        else { mB0 = &tmBp; mB1 = &tmBplo; bmn = false; bc = 0; b_bytes = PAR_BYTES; }
        const uint32_t tx_bytes = 2u * S::NOPS * (a_bytes + b_bytes);
        using T_ = std::true_type;
        using F_ = std::false_type;
        if (!amn && bmn) kloop(F_{}, T_{}, mA0, mA1, mB0, mB1, ac, bc, bnb, tx_bytes);
        else if (!amn && !bmn) kloop(F_{}, F_{}, mA0, mA1, mB0, mB1, ac, bc, bnb, tx_bytes);
        else if (amn && bmn) kloop(T_{}, T_{}, mA0, mA1, mB0, mB1, ac, bc, bnb, tx_bytes);
        else kloop(T_{}, F_{}, mA0, mA1, mB0, mB1, ac, bc, bnb, tx_bytes);
      }
    }
  } else if (warp == 1) {
    if (rank == 0) {
      // ================= MMA issuer (leader CTA; the whole warp runs the loop, one elected lane issues) =================
      int stage = 0;
      uint32_t phase = 0;
      int acc = 0;
      uint32_t acc_phase = 0;
      for (int t = pair; t < p.num_items; t += npairs) {
        const Tile tl = decode_item(p, t);
        const bool a_mn = tl.kind == TILE_PC ? p.b_mn != 0 : ((tl.kind == TILE_PG || tl.kind == TILE_PCL) ? false : p.a_mn != 0);
        const bool b_mn = (tl.kind == TILE_DATA || tl.kind == TILE_PCL) && p.b_mn != 0;
        const uint32_t idesc = make_idesc(C::FMT, a_mn ? 1u : 0u, b_mn ? 1u : 0u, 2 * BM, tl.ncols);
        mbar_wait_bounded(tempty_bar(acc), acc_phase ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * BN;
        const uint32_t k_step = (C::UK * C::ELT) >> 4;  // K-major: UK elements along the swizzle row
        const uint32_t mn_step = (C::UK * 128) >> 4;    // MN-major: UK rows of k
        const uint32_t a_step = a_mn ? mn_step : k_step, b_step = b_mn ? mn_step : k_step;
        for (int kb = 0; kb < kblocks; ++kb) {
          mbar_wait_bounded(full_bar(stage), phase);
          tc_fence_after();
          const uint32_t sA = smem_base + stage * S::STAGE_BYTES;
          const uint32_t sB = sA + S::NOPS * S::A_BYTES;
          // K-major: 8-row groups 1024 B apart.  MN-major: 128 B of m/n per row of k, 8-row k groups 1024 B apart (SBO;
          // 512 B for the 32-byte-atom swizzle of 32-bit elements), 128-byte m/n groups BOX_BYTES apart (LBO).
          auto mn_desc = [&](uint32_t s) { return KIND == GECC_BF16 ? smem_desc_sw128(s, BOX_BYTES, 1024) : smem_desc_sw128_base32(s, BOX_BYTES, 512); };
          const uint64_t a_hi = a_mn ? mn_desc(sA) : smem_desc_sw128(sA, 16, 1024);
          const uint64_t b_hi = b_mn ? mn_desc(sB) : smem_desc_sw128(sB, 16, 1024);
          if (elect_one()) {
#pragma unroll
          for (int ks = 0; ks < BK / C::UK; ++ks) {
            const uint32_t accum = (kb | ks) ? 1u : 0u;
            if (KIND == GECC_BF16) {
              mma_bf16_pair(d_tmem, a_hi + ks * a_step, b_hi + ks * b_step, idesc, accum);
            } else {
              // 3xTF32: a b ~ a_lo b_hi + a_hi b_lo + a_hi b_hi, small terms first
              const uint64_t a_lo = a_hi + (S::A_BYTES >> 4), b_lo = b_hi + (S::B_BYTES >> 4);
              mma_tf32_pair(d_tmem, a_lo + ks * a_step, b_hi + ks * b_step, idesc, accum);
              mma_tf32_pair(d_tmem, a_hi + ks * a_step, b_lo + ks * b_step, idesc, 1u);
              mma_tf32_pair(d_tmem, a_hi + ks * a_step, b_hi + ks * b_step, idesc, 1u);
            }
          }
          mma_commit_pair(empty_bar(stage));  // frees the stage in both CTAs
          }
          __syncwarp();
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        if (elect_one()) mma_commit_pair(tfull_bar(acc));  // accumulator ready in both CTAs
        __syncwarp();
        if (++acc == 2) { acc = 0; acc_phase ^= 1; }
      }
    }
  } else if (warp >= EPI_WARP0) {
    // ================= epilogue (both CTAs, own 128 TMEM lanes) =================
    const int wq = warp - EPI_WARP0;  // TMEM lane quarter this warp may read: lanes 32 wq .. 32 wq + 31
    const uint32_t stg = epi_base + wq * (32 * 32 * 4);
    const uint32_t tempty_leader0 = mapa(tempty_bar(0), 0), tempty_leader1 = mapa(tempty_bar(1), 0);
    int acc = 0;
    uint32_t acc_phase = 0;
    for (int t = pair; t < p.num_items; t += npairs) {
      const Tile tl = decode_item(p, t);
      const bool reduce = p.protect && tl.kind == TILE_DATA;
      const int lane0 = tl.row0 + (int)rank * BM;            // what TMEM lane 0 of this CTA holds: a row (DATA, PR, PG) or a column (PC)
      const int my_line = lane0 + wq * 32 + lane;
      float* out = nullptr;
      int64_t ld = 0;
      int rows_valid = 0, cols_valid = 0;
      if (tl.kind == TILE_DATA) { out = p.C + (int64_t)lane0 * p.ldc + tl.col0; ld = p.ldc; rows_valid = p.n - lane0; cols_valid = p.m - tl.col0; }
      else if (tl.kind == TILE_PR) { out = p.P_r + (int64_t)lane0 * GECC_PR_LD; ld = GECC_PR_LD; rows_valid = p.n - lane0; cols_valid = GECC_PR_LD; }
      else if (tl.kind == TILE_PG) { out = p.P_g; ld = GECC_PR_LD; rows_valid = rank == 0 ? GECC_PAR_ROWS : 0; cols_valid = GECC_PR_LD; }
      else if (tl.kind == TILE_PCL) { out = p.PcL + (int64_t)lane0 * p.ldpcl + tl.col0; ld = p.ldpcl; rows_valid = p.tl_rows_a - lane0; cols_valid = p.m - tl.col0; }
      else if (tl.kind == TILE_PRL) { out = p.PrL + (int64_t)lane0 * p.ldprl + tl.col0; ld = p.ldprl; rows_valid = p.n - lane0; cols_valid = p.tl_rows_b - tl.col0; }
      const int nchunks = (tl.kind == TILE_DATA || tl.kind >= TILE_PCL) ? tl.ncols / 32 : 1;

      mbar_wait_bounded(tfull_bar(acc), acc_phase);
      tc_fence_after();
      float s1 = 0.f, s2 = 0.f, ss = 0.f;
#ifdef GECC_NO_EPI
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(acc ? tempty_leader1 : tempty_leader0);
      if (++acc == 2) { acc = 0; acc_phase ^= 1; }
      continue;
#endif
      for (int c = 0; c < nchunks; ++c) {
        uint32_t v[32];
        tmem_ld32(tmem_base + acc * BN + c * 32 + ((uint32_t)(wq * 32) << 16), v);
        tmem_ld_wait();
        if (c == nchunks - 1) {  // accumulator buffer fully read: hand it back to the MMA warp of the leader
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(acc ? tempty_leader1 : tempty_leader0);
        }
        if (tl.kind == TILE_PC) {  // lanes are columns of C, TMEM columns 0..7 the parity rows: P_c[r][column]
          if (my_line < p.m) {
#pragma unroll
            for (int r = 0; r < GECC_PAR_ROWS; ++r) p.P_c[(int64_t)r * p.m + my_line] = __uint_as_float(v[r]);
          }
          continue;
        }
        if (p.n_inject > 0 && tl.kind == TILE_DATA) {  // E3: fault on a symbol of C during its computation
          for (int f = 0; f < p.n_inject; ++f) {
            const gecc_fault_t ft = p.inject[f];
            const int cc = ft.col - (tl.col0 + c * 32);
            if (ft.kind == GECC_KIND_C && ft.row == my_line && cc >= 0 && cc < 32) {
#pragma unroll
              for (int q = 0; q < 32; ++q)
                if (q == cc) v[q] = __float_as_uint(__uint_as_float(v[q]) + ft.value);
            }
          }
        }
        if (reduce) {  // row sums of PAPER.md:194,196 over this block of 128 columns, local weights
#pragma unroll
          for (int q = 0; q < 32; ++q) {
            const float x = __uint_as_float(v[q]);
            s1 += x;
            s2 = fmaf((float)((c & 3) * 32 + q), x, s2);
            ss = fmaf(x, x, ss);  // line energy: scales the line's threshold (rounding noise is relative)
          }
        }
        // registers -> shared, 16-byte chunks XOR-swizzled by row so both directions are conflict-free
#pragma unroll
        for (int c4 = 0; c4 < 8; ++c4) {
          const uint32_t addr = stg + lane * 128 + ((c4 ^ (lane & 7)) << 4);
          asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v[4 * c4]), "r"(v[4 * c4 + 1]), "r"(v[4 * c4 + 2]), "r"(v[4 * c4 + 3]) : "memory");
        }
        __syncwarp();
        float cs1[4] = {0.f, 0.f, 0.f, 0.f}, cs2[4] = {0.f, 0.f, 0.f, 0.f}, css[4] = {0.f, 0.f, 0.f, 0.f};
        const int c4 = lane & 7;
        const int col = c * 32 + 4 * c4;  // column within the tile
#pragma unroll
        for (int it = 0; it < 8; ++it) {
          const int r = it * 4 + (lane >> 3);
          const uint32_t addr = stg + r * 128 + ((c4 ^ (r & 7)) << 4);
          float4 x;
          asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(x.x), "=f"(x.y), "=f"(x.z), "=f"(x.w) : "r"(addr) : "memory");
          if (wq * 32 + r < rows_valid && col < cols_valid)
            *reinterpret_cast<float4*>(out + (int64_t)(wq * 32 + r) * ld + col) = x;
          if (reduce) {  // column sums of PAPER.md:198,200 over this warp's 32 rows, local weights
            const float w = (float)r;
            cs1[0] += x.x; cs1[1] += x.y; cs1[2] += x.z; cs1[3] += x.w;
            cs2[0] = fmaf(w, x.x, cs2[0]); cs2[1] = fmaf(w, x.y, cs2[1]); cs2[2] = fmaf(w, x.z, cs2[2]); cs2[3] = fmaf(w, x.w, cs2[3]);
            css[0] = fmaf(x.x, x.x, css[0]); css[1] = fmaf(x.y, x.y, css[1]); css[2] = fmaf(x.z, x.z, css[2]); css[3] = fmaf(x.w, x.w, css[3]);
          }
        }
        if (reduce) {
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            cs1[e] += __shfl_xor_sync(0xffffffffu, cs1[e], 8);
            cs2[e] += __shfl_xor_sync(0xffffffffu, cs2[e], 8);
            cs1[e] += __shfl_xor_sync(0xffffffffu, cs1[e], 16);
            cs2[e] += __shfl_xor_sync(0xffffffffu, cs2[e], 16);
            css[e] += __shfl_xor_sync(0xffffffffu, css[e], 8);
            css[e] += __shfl_xor_sync(0xffffffffu, css[e], 16);
          }
          if (lane < 8) {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const uint32_t a = colacc_base + ((wq * BN + col + e) * 3) * 4;
              asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(cs1[e]) : "memory");
              asm volatile("st.shared.f32 [%0], %1;" ::"r"(a + 4), "f"(cs2[e]) : "memory");
              asm volatile("st.shared.f32 [%0], %1;" ::"r"(a + 8), "f"(css[e]) : "memory");
            }
          }
          if ((c & 3) == 3) {  // 128 columns done: one row partial (weights local to the block of 128 columns)
            if (my_line < p.n && tl.col0 + (c & ~3) * 32 < p.m) {
              const int cbg = (tl.col0 + c * 32) / kSumCols;  // block of 128 columns these sums belong to
              if (p.detect) {  // straight into the row's accumulators, global weight (index + 1) restored
                double* acc = p.lineacc + (int64_t)my_line * 4;
                atomicAdd(acc, (double)s1);
                atomicAdd(acc + 1, (double)(cbg * kSumCols + 1) * (double)s1 + (double)s2);
                atomicAdd(acc + 2, (double)ss);
              } else *reinterpret_cast<float4*>(p.rowpart + ((int64_t)cbg * p.n + my_line) * 4) = make_float4(s1, s2, ss, 0.f);
            }
            s1 = 0.f; s2 = 0.f; ss = 0.f;
          }
        }
        __syncwarp();
      }
      if (reduce) {
        // column sums of this CTA's 128-row block: add the four warps' 32-row slabs (slab w carries the row offset 32 w)
        asm volatile("bar.sync 1, 128;" ::: "memory");
        for (int cc = threadIdx.x - EPI_WARP0 * 32; cc < tl.ncols; cc += 128) {
          float a = 0.f, b = 0.f, e2 = 0.f;
#pragma unroll
          for (int w4 = 0; w4 < 4; ++w4) {
            float x1, x2, x3;
            const uint32_t ad = colacc_base + ((w4 * BN + cc) * 3) * 4;
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(x1) : "r"(ad) : "memory");
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(x2) : "r"(ad + 4) : "memory");
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(x3) : "r"(ad + 8) : "memory");
            a += x1;
            b += fmaf((float)(32 * w4), x1, x2);
            e2 += x3;
          }
          const int gcol = tl.col0 + cc;
          if (gcol < p.m && lane0 < p.n) {
            if (p.detect) {
              double* acc = p.lineacc + ((int64_t)p.n + gcol) * 4;
              atomicAdd(acc, (double)a);
              atomicAdd(acc + 1, (double)(lane0 + 1) * (double)a + (double)b);  // lane0: first row of this block of 128 rows
              atomicAdd(acc + 2, (double)e2);
            } else *reinterpret_cast<float4*>(p.colpart + ((int64_t)(lane0 / kSumRows) * p.m + gcol) * 4) = make_float4(a, b, e2, 0.f);
          }
        }
        asm volatile("bar.sync 1, 128;" ::: "memory");
      }
      if (p.detect && tl.kind <= TILE_PR) {
        // which strips of 128 rows / 128 columns this CTA's tile completed a block of (lane0: its first row; PC: first column)
        int row_strip = -1, row_cnt = 0, cs0 = -1, cs1 = -1;
        if (tl.kind == TILE_DATA) {
          if (lane0 < p.n) {
            const int c_lo = tl.col0 / kSumCols;
            const int c_hi = (min(p.m, tl.col0 + tl.ncols) + kSumCols - 1) / kSumCols;  // one past the last valid block
            row_cnt = max(0, c_hi - c_lo);
            if (row_cnt > 0) row_strip = lane0 / kSumRows;
            if (row_cnt > 0) cs0 = c_lo;
            if (row_cnt > 1) cs1 = c_lo + 1;
          }
        } else if (tl.kind == TILE_PR) {
          if (lane0 < p.n) { row_strip = lane0 / kSumRows; row_cnt = 1; }
        } else {  // TILE_PC
          if (lane0 < p.m) cs0 = lane0 / kSumCols;
        }
        if (row_strip >= 0 || cs0 >= 0) detect_tail(p, row_strip, row_cnt, cs0, cs1, lastflags, (int)threadIdx.x - EPI_WARP0 * 32);
      }
      if (++acc == 2) { acc = 0; acc_phase ^= 1; }
    }
  }

  tc_fence_before();
  __syncthreads();
  cluster_sync();  // neither CTA leaves (or frees TMEM) while the other may still signal its barriers
  if (warp == 2) tmem_dealloc_pair(tmem_base, TMEM_COLS);
  if (p.protect && threadIdx.x == 0) ws_exit(p.counters, gridDim.x);
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (fn) return fn;
  void* sym = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) != cudaSuccess || qres != cudaDriverEntryPointSuccess)
    return nullptr;
  fn = reinterpret_cast<EncodeTiledFn>(sym);
  return fn;
}

// 2-D row-major tensor [outer x inner] with leading dimension ld (elements); box = {box_inner, box_outer}; 128 B swizzle.
// Out-of-bounds elements of a box are filled with zeros (ragged edges, rows of the peer CTA past the end).
static int make_tmap(CUtensorMap* tm, int kind, const void* ptr, int64_t inner, int64_t outer, int64_t ld, int box_inner, int box_outer,
                     CUtensorMapSwizzle swz = CU_TENSOR_MAP_SWIZZLE_128B) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return GECC_ECUDA;
  const int elt = (kind == GECC_BF16) ? 2 : 4;
  cuuint64_t dims[2] = {(cuuint64_t)inner, (cuuint64_t)outer};
  cuuint64_t strides[1] = {(cuuint64_t)ld * elt};
  cuuint32_t box[2] = {(cuuint32_t)box_inner, (cuuint32_t)box_outer};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(tm, kind == GECC_BF16 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(ptr), dims,
                  strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, swz, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    fprintf(stderr, "gecc: cuTensorMapEncodeTiled failed (%d) inner=%lld outer=%lld ld=%lld box=%dx%d\n", (int)r, (long long)inner,
            (long long)outer, (long long)ld, box_inner, box_outer);
    return GECC_ECUDA;
  }
  return GECC_OK;
}

// SM count of the CURRENT device (cached per device: a process may drive several GPUs).
int num_sms() {
  constexpr int kMaxDev = 64;
  static int sms[kMaxDev] = {0};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0) return 0;
  if (dev >= kMaxDev) {
    int v = 0;
    return cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess ? v : 0;
  }
  if (!sms[dev] && cudaDeviceGetAttribute(&sms[dev], cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) sms[dev] = 0;
  return sms[dev];
}

template <int KIND>
static int launch_gemm(bool protect, int64_t n, int64_t k, int64_t m, bool trans_a, bool trans_b, const void* A, int64_t lda, const void* A_par, const float* A_lo,
                       const float* A_par_lo, const void* B, int64_t ldb, const void* B_par, const float* B_lo, const float* B_par_lo,
                       float* Cout, int64_t ldc, float* P_r, float* P_c, float* P_g, const gecc_fault_t* inject, int n_inject,
                       float* rowpart, float* colpart, const DetectArgs* det, bool pdl, cudaStream_t stream, const TlArgs* tla) {
  using C = Cfg<KIND>;
  using S = Smem<KIND>;
  CUtensorMap tmA, tmB, tmAp, tmBp, tmAlo, tmBlo, tmAplo, tmBplo;
  int rc;
  const int nsw = 128 / C::ELT;  // elements per 128-byte swizzle row
  // MN-major operand: 16-bit elements take the plain 128B swizzle, 32-bit elements the 32-byte-atom variant
  const CUtensorMapSwizzle swzMN = KIND == GECC_BF16 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B;
  auto map_a = [&](CUtensorMap* tm, const void* ptr) {  // A: n x k row-major (K-major boxes) or A^T: k x n (MN-major boxes)
    return trans_a ? make_tmap(tm, KIND, ptr, n, k, lda, nsw, C::BK, swzMN) : make_tmap(tm, KIND, ptr, k, n, lda, C::BK, BM, CU_TENSOR_MAP_SWIZZLE_128B);
  };
  auto map_b = [&](CUtensorMap* tm, const void* ptr) {  // B: k x m row-major (MN-major boxes) or B^T: m x k (K-major boxes)
    return trans_b ? make_tmap(tm, KIND, ptr, k, m, ldb, C::BK, BM, CU_TENSOR_MAP_SWIZZLE_128B) : make_tmap(tm, KIND, ptr, m, k, ldb, nsw, C::BK, swzMN);
  };
  if ((rc = map_a(&tmA, A))) return rc;
  if ((rc = map_b(&tmB, B))) return rc;
  tmAp = tmA; tmBp = tmB; tmAlo = tmA; tmBlo = tmB; tmAplo = tmA; tmBplo = tmB;
  // parity operands, K-major [rows x k]: the two global parity rows of each side (8 rows with limbs, one box), or -- tile-local
  // grid -- the stacked panel parity (8 rows per panel of 128 lines), fetched in boxes of 128 rows like rows of A
  const int64_t par_rows_a = tla ? tla->rows_a : GECC_PAR_ROWS, par_rows_b = tla ? tla->rows_b : GECC_PAR_ROWS;
  const int par_box = tla ? BM : GECC_PAR_ROWS;
  if (protect) {
    if ((rc = make_tmap(&tmAp, KIND, A_par, k, par_rows_a, k, C::BK, par_box))) return rc;
    if ((rc = make_tmap(&tmBp, KIND, B_par, k, par_rows_b, k, C::BK, par_box))) return rc;
  }
  if (KIND == GECC_F32) {
    if ((rc = map_a(&tmAlo, A_lo))) return rc;
    if ((rc = map_b(&tmBlo, B_lo))) return rc;
    tmAplo = tmAlo; tmBplo = tmBlo;
    if (protect) {
      if ((rc = make_tmap(&tmAplo, KIND, A_par_lo, k, par_rows_a, k, C::BK, par_box))) return rc;
      if ((rc = make_tmap(&tmBplo, KIND, B_par_lo, k, par_rows_b, k, C::BK, par_box))) return rc;
    }
  }
  const int sms = num_sms();
  if (sms < 2) return GECC_ECUDA;
  const int pairs_max = sms / 2;
  GemmParams p;
  p.n = (int)n; p.k = (int)k; p.m = (int)m;
  p.mbp = (int)((n + 2 * BM - 1) / (2 * BM));
  p.nbp = (int)((m + BN - 1) / BN);
  p.protect = protect ? 1 : 0;
  p.a_mn = trans_a ? 1 : 0;
  p.b_mn = trans_b ? 0 : 1;
  // Tail balancing: the data units left over after the last full round of the pairs are computed as two half-width tiles
  // each when that fills at most one more round (3.46 rounds become 3.5 instead of 4 at 4096^2 on 74 pairs).
  p.n_data_units = p.mbp * p.nbp;
  p.tl = tla ? 1 : 0;
  p.tl_rows_a = tla ? (int)tla->rows_a : 0; p.tl_rows_b = tla ? (int)tla->rows_b : 0;
  p.tl_rb = tla ? (p.tl_rows_a + 2 * BM - 1) / (2 * BM) : 0;
  p.tl_cb = tla ? (p.tl_rows_b + BN - 1) / BN : 0;
  p.PcL = tla ? tla->PcL : nullptr; p.PrL = tla ? tla->PrL : nullptr;
  p.ldpcl = tla ? tla->ldpcl : 0; p.ldprl = tla ? tla->ldprl : 0;
  const int units = p.n_data_units + p.tl_rb * p.nbp + p.mbp * p.tl_cb, rem = units % pairs_max;
  p.n_split = (rem > 0 && 2 * rem <= pairs_max) ? rem : 0;
  p.n_full = units - p.n_split;
  // operands that fit in L2 beside the C being written (4096^2 bf16: 64 MB) keep the plain column-block-major order (one
  // band: measured 120 MB instead of 133 MB of DRAM reads per 4096^3 product); larger ones take bands of 8
  const bool fits_l2 = (double)(n * k + k * m) * C::ELT <= 64.0 * 1024 * 1024;
  p.gh = (fits_l2 || p.mbp < 8) ? p.mbp : 8;
  p.num_items = p.n_full + 2 * p.n_split + ((protect && !tla) ? p.nbp + p.mbp + 1 : 0);
  p.C = Cout; p.ldc = ldc; p.P_r = P_r; p.P_c = P_c; p.P_g = P_g;
  p.rowpart = rowpart; p.colpart = colpart;
  p.inject = inject; p.n_inject = inject ? n_inject : 0;
  p.detect = 0; p.st = nullptr; p.counters = nullptr; p.arrive = nullptr; p.report = nullptr; p.lineacc = nullptr;
  p.nrb128 = (int)((n + kSumRows - 1) / kSumRows); p.ncb128 = (int)((m + kSumCols - 1) / kSumCols);
  p.ts.have_tau = 0; p.ts.sumsq_a = p.ts.sumsq_b = nullptr; p.ts.noise_c = noise_coeff(KIND, (double)k); p.ts.single = 0;
  for (int q = 0; q < 4; ++q) p.ts.tau[q] = 0.0;
  if (protect && det) {
    p.st = det->st;  // the product always says whether it left syndromes or partial sums only
    p.detect = det->detect ? 1 : 0;
    p.counters = det->counters; p.arrive = det->arrive; p.report = det->report; p.lineacc = det->lineacc;
    p.ts.have_tau = det->tau ? 1 : 0;
    for (int q = 0; q < 4; ++q) p.ts.tau[q] = det->tau ? det->tau[q] : 0.0;
    p.ts.sumsq_a = det->sumsq_a; p.ts.sumsq_b = det->sumsq_b; p.ts.single = det->single ? 1 : 0;
    p.fb.dtype = KIND; p.fb.n = (int)n; p.fb.m = (int)m;
    p.fb.rowpart = rowpart; p.fb.colpart = colpart; p.fb.P_r = P_r; p.fb.P_c = P_c;
    p.fb.syn = det->syn; p.fb.rflag = det->flags; p.fb.qflag = det->flags + ((n + 15) & ~15ll);
  }
  // the attribute is per device: set it on every launch (a host-side table lookup, no device work)
  if (cudaFuncSetAttribute(gecc_gemm_kernel<KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::TOTAL) != cudaSuccess) return GECC_ECUDA;
  const int pairs = p.num_items < pairs_max ? p.num_items : pairs_max;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(2 * pairs);
  cfg.blockDim = dim3(NUM_THREADS);
  cfg.dynamicSmemBytes = S::TOTAL;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;  // overlap this kernel's prologue with the encoder's tail
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = pdl ? 1 : 0;
  if (cudaLaunchKernelEx(&cfg, gecc_gemm_kernel<KIND>, tmA, tmB, tmAp, tmBp, tmAlo, tmBlo, tmAplo, tmBplo, p) != cudaSuccess) return GECC_ECUDA;
  return GECC_OK;
}

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

int gemm_dispatch(bool protect, int dtype, int64_t n, int64_t k, int64_t m, bool trans_a, bool trans_b, const void* A, int64_t lda, const void* A_par, const float* A_lo,
                  const float* A_par_lo, const void* B, int64_t ldb, const void* B_par, const float* B_lo, const float* B_par_lo, float* C,
                  int64_t ldc, float* P_r, float* P_c, float* P_g, const gecc_fault_t* inject, int n_inject, float* rowpart, float* colpart,
                  const DetectArgs* det, bool pdl, cudaStream_t stream, const TlArgs* tla) {
  if (dtype != GECC_BF16 && dtype != GECC_F32) return GECC_EUNSUPPORTED;
  if (!A || !B || !C || n <= 0 || k <= 0 || m <= 0 || n > (1 << 30) || k > (1 << 30) || m > (1 << 30)) return GECC_EINVAL;
  const int epr = dtype == GECC_BF16 ? 8 : 4;  // elements per 16 bytes
  if (lda < (trans_a ? n : k) || ldb < (trans_b ? k : m) || ldc < m || lda % epr || ldb % epr || ldc % 4 || m % 4 || k % epr) return GECC_EINVAL;
  if ((trans_a && n % epr) || (trans_b && k % epr)) return GECC_EINVAL;
  if (!aligned16(A) || !aligned16(B) || !aligned16(C)) return GECC_EINVAL;
  if (dtype == GECC_F32 && (!A_lo || !B_lo || !aligned16(A_lo) || !aligned16(B_lo))) return GECC_EINVAL;
  if (protect) {
    if (!A_par || !B_par || !rowpart || !colpart || !aligned16(A_par) || !aligned16(B_par)) return GECC_EINVAL;
    if (tla) {
      if (!tla->PcL || !tla->PrL || !aligned16(tla->PcL) || !aligned16(tla->PrL) || tla->ldpcl < m || tla->ldprl < tla->rows_b || tla->ldpcl % 4 || tla->ldprl % 4 ||
          tla->rows_a <= 0 || tla->rows_b <= 0 || !det || det->detect)
        return GECC_EINVAL;
    } else if (!P_r || !P_c || !P_g || !aligned16(P_r) || !aligned16(P_c) || !aligned16(P_g)) return GECC_EINVAL;
    if (dtype == GECC_F32 && (!A_par_lo || !B_par_lo)) return GECC_EINVAL;
    if (n_inject < 0 || (n_inject > 0 && !inject)) return GECC_EINVAL;
  }
  if (dtype == GECC_BF16)
    return launch_gemm<GECC_BF16>(protect, n, k, m, trans_a, trans_b, A, lda, A_par, A_lo, A_par_lo, B, ldb, B_par, B_lo, B_par_lo, C, ldc, P_r, P_c, P_g, inject,
                                  n_inject, rowpart, colpart, det, pdl, stream, tla);
  return launch_gemm<GECC_F32>(protect, n, k, m, trans_a, trans_b, A, lda, A_par, A_lo, A_par_lo, B, ldb, B_par, B_lo, B_par_lo, C, ldc, P_r, P_c, P_g, inject,
                               n_inject, rowpart, colpart, det, pdl, stream, tla);
}

}  // namespace gecc
