// Detection and correction and its completion for input faults (readings R5-R9) as ONE
// cooperative kernel: every phase runs on the whole grid, separated by grid barriers, so a fault-free product costs one
// launch, one pass over the per-tile partial sums and one barrier.
//
//   phase 1  syndromes   r1, r2, q1, q2 = sum minus parity from the partial sums the product's epilogue
//                        left in the workspace, compared with the thresholds of their own line -> flag sets E_r, E_t
//                        (PAPER.md:215-217).  Nothing flagged: block 0 writes CLEAN and everyone leaves.
//   phase 2  decide      block 0.  |E_r| = s, |E_t| = t -> min(s,t) >= 3: "needs to be recalculated";
//                        otherwise WLOG s <= t: locate the <= 2 faulty rows, estimate the errors from the
//                        column syndromes (s = 1: PAPER.md:223, s = 2: the 2x2 system of PAPER.md:227 with the right-hand
//                        side "sum minus parity"), classify whole-line faults (an input fault) vs points.
//   phase 3  verify      Level-X.  Column checks of A / row checks of B recomputed by the encoder's reductions and compared
//                        with the fp64 parity stored at encode time; locates (i, l, e) / (l, j, e).
//   phase 4  repair      patches A / B, recomputes the rows / columns of C the faults touched from the patched operands
//                        ("mark the compromised data for recomputation") and carries the change into the
//                        syndromes; then decides again on what is left (points only).
//   phase 5  patch       applies the plan to C in place (c_true = c - e) and writes the report.
#include <cuda_bf16.h>
#include <cstdio>
#include <cuda_runtime.h>

#include "encode_core.cuh"
#include "fold.cuh"
#include "gecc_internal.h"
#include "sm100_ptx.cuh"

namespace gecc {

using ptx::griddep_wait;
using ptx::griddep_launch_dependents;

constexpr int DT = 256;  // threads per block of the decoder

struct Scratch {
  int i[DT / 32];
  unsigned long long u[DT / 32];
  double d[DT / 32][4];
  int cnt;
  int idx[8];
  int flag;
};

struct DecodeParams {
  int dtype, level, n, k, m;
  int trans_a, trans_b;  // storage of the operands: A^T (k x n), B^T (m x k)
  float* C;
  int64_t ldc;
  FoldBufs fb;       // partial sums, parity symbols of C, syndromes, flags
  ThresholdSpec ts;  // used only when the product did not fold its sums itself (otherwise the thresholds are in the state)
  void* A;
  int64_t lda;
  float* A_lo;
  const double* A_par64;
  void* B;
  int64_t ldb;
  float* B_lo;
  const double* B_par64;
  gecc_report_t* report;
  unsigned int* counters;
  double* encpart;    // encoder scratch (chunk partials of the verification pass over A)
  double* encpart_b;  // the same for a transposed B (stored m x k: the column-direction reduction)
  double* recomp;   // partials of the row recomputation / a contiguous column of B
  int* votes;
  uint8_t* lists;
  DecodeState* st;
  int enc_chunk_rows;    // rows per partial of the verification pass over A: the encoder's own choice for this shape
  int enc_chunk_rows_b;  // the same for B^T
  double G;        // residual allowance per unit of removed footprint
  int single;      // GECC_SINGLE_CHECKSUM
  float* P_r_w;    // the parity blocks of C_bar, writable: a faulty parity symbol is repaired in place
  float* P_c_w;
  const float* P_g;  // global parity block [GECC_PAR_ROWS x GECC_PR_LD] or null
  unsigned long long* stamps;  // phase boundary timestamps (block 0), diagnostic
};


// Grid barrier of the cooperative launch (all blocks are co-resident): arrivals are counted on a word that only grows
// during one launch; `target` is the arrival count that releases this barrier.  The last block to leave the kernel
// clears the word again.  Release: every thread fences its writes before the block arrives; acquire: the polling thread
// fences after it sees the count (which also drops stale L1 lines), then releases the block.
__device__ __forceinline__ void grid_barrier(unsigned int* ctr, unsigned int& target) {
  target += gridDim.x;
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    atomicAdd(ctr, 1u);
    // relaxed polls (an acquire load would invalidate this SM's L1 on every iteration, which also serves the local memory
    // of a co-resident block that is still working), one fence once the count is seen
    unsigned int seen;
    for (;;) {
      asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(ctr) : "memory");
      if (seen >= target) break;
      __nanosleep(100);
    }
    __threadfence();
  }
  __syncthreads();
}


__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}

__device__ int block_sum(int v, Scratch& sc) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) sc.i[threadIdx.x >> 5] = v;
  __syncthreads();
  int t = 0;
  for (int w = 0; w < DT / 32; ++w) t += sc.i[w];
  return t;
}
__device__ unsigned long long block_max(unsigned long long v, Scratch& sc) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long w = __shfl_xor_sync(0xffffffffu, v, o);
    v = w > v ? w : v;
  }
  __syncthreads();
  if ((threadIdx.x & 31) == 0) sc.u[threadIdx.x >> 5] = v;
  __syncthreads();
  unsigned long long t = 0;
  for (int w = 0; w < DT / 32; ++w) t = sc.u[w] > t ? sc.u[w] : t;
  return t;
}
// Sum of four doubles per thread over the block, fixed tree; the result is valid in every thread.
__device__ void block_sum4(double (&v)[4], Scratch& sc) {
#pragma unroll
  for (int q = 0; q < 4; ++q)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0)
#pragma unroll
    for (int q = 0; q < 4; ++q) sc.d[threadIdx.x >> 5][q] = v[q];
  __syncthreads();
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    double t = 0.0;
    for (int w = 0; w < DT / 32; ++w) t += sc.d[w][q];
    v[q] = t;
  }
}

__device__ void sort_found(gecc_found_t* f, int n) {
  for (int a = 0; a < n; ++a)
    for (int b = a + 1; b < n; ++b) {
      const bool less = f[b].kind < f[a].kind || (f[b].kind == f[a].kind && (f[b].row < f[a].row || (f[b].row == f[a].row && f[b].col < f[a].col)));
      if (less) { const gecc_found_t t = f[a]; f[a] = f[b]; f[b] = t; }
    }
}

// Compact view of the flagged lines of one side, ascending by index: idx[e], plain / weighted syndrome a1[e], a2[e] and the
// thresholds of the line's own checks t1[e] = tau_plain + tolx, t2[e] = tau_weighted + tolx.
struct FlagList {
  int* idx;
  double* a1;
  double* a2;
  double* t1;
  double* t2;
  int cnt;
};

// Warp w of the block owns the contiguous slice [wlo, whi) of [0, cnt), a multiple of 32 long, and walks it 32 entries at
// a time (lane <-> entry: coalesced); slices in warp order, rounds in order, lanes in order = ascending entries.
__device__ __forceinline__ void warp_slice(int cnt, int& wlo, int& whi) {
  const int cw = (((cnt + DT / 32 - 1) / (DT / 32)) + 31) & ~31;
  wlo = min(cnt, (int)(threadIdx.x >> 5) * cw);
  whi = min(cnt, wlo + cw);
}

// Builds the list of flagged lines from the byte flags.  One block; the list comes out sorted (see warp_slice).
__device__ void compact_flagged(const uint8_t* flg, int len, const double* v1, const double* v2, const double* x1, const double* x2, double tau1,
                                double tau2, FlagList& L, bool with_values, Scratch& sc) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int wlo, whi;
  warp_slice(len, wlo, whi);
  int c = 0;  // flagged lines of this warp's slice (same in every lane)
  for (int i0 = wlo; i0 < whi; i0 += 128) {
    uint8_t f[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { const int i = i0 + 32 * u + lane; f[u] = i < whi ? __ldcg(flg + i) : (uint8_t)0; }
#pragma unroll
    for (int u = 0; u < 4; ++u) c += __popc(__ballot_sync(0xffffffffu, f[u] != 0));
  }
  __syncthreads();
  if (lane == 0) sc.i[w] = c;
  __syncthreads();
  int pos = 0, total = 0;
  for (int ww = 0; ww < DT / 32; ++ww) { if (ww < w) pos += sc.i[ww]; total += sc.i[ww]; }
  if (c > 0) {
    for (int i0 = wlo; i0 < whi; i0 += 128) {
      uint8_t f[4];
      double a1[4], a2[4], t1[4], t2[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) { const int i = i0 + 32 * u + lane; f[u] = i < whi ? __ldcg(flg + i) : (uint8_t)0; }
      if (with_values) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int i = min(i0 + 32 * u + lane, len - 1);
          a1[u] = __ldcg(v1 + i); a2[u] = __ldcg(v2 + i); t1[u] = __ldcg(x1 + i); t2[u] = __ldcg(x2 + i);
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const unsigned b = __ballot_sync(0xffffffffu, f[u] != 0);
        if (f[u]) {
          const int o = pos + __popc(b & ((1u << lane) - 1u));
          L.idx[o] = i0 + 32 * u + lane;
          if (with_values) { L.a1[o] = a1[u]; L.a2[o] = a2[u]; L.t1[o] = tau1 + t1[u]; L.t2[o] = tau2 + t2[u]; }
        }
        pos += __popc(b);
      }
    }
  }
  L.cnt = total;
  __threadfence_block();
  __syncthreads();
}

// The same list from the entries the flagging blocks left in the decoder state (cnt <= 8 of them, unordered): every
// thread ranks its entry among the others, so the list comes out sorted without a search of the flags.
__device__ void collect_early(const DecodeState::Early* E, int cnt, FlagList& L, bool with_values, Scratch& sc) {
  __syncthreads();
  if ((int)threadIdx.x < cnt) {
    int id[8];
#pragma unroll
    for (int a = 0; a < 8; ++a) id[a] = __ldcg(&E->idx[a]);
    const int e = threadIdx.x;
    double v1 = 0.0, v2 = 0.0, w1 = 0.0, w2 = 0.0;
    if (with_values) { v1 = __ldcg(&E->a1[e]); v2 = __ldcg(&E->a2[e]); w1 = __ldcg(&E->t1[e]); w2 = __ldcg(&E->t2[e]); }
    int mine = 0, rank = 0;
#pragma unroll
    for (int a = 0; a < 8; ++a) if (a == e) mine = id[a];
#pragma unroll
    for (int a = 0; a < 8; ++a) rank += (a < cnt && id[a] < mine) ? 1 : 0;
    L.idx[rank] = mine;
    if (with_values) { L.a1[rank] = v1; L.a2[rank] = v2; L.t1[rank] = w1; L.t2[rank] = w2; }
  }
  L.cnt = cnt;
  __threadfence_block();
  __syncthreads();
}

// Visits the entries of a list: f(e, valid, a1, a2, t1, t2) is called by whole warps (valid = false past the end), four
// rounds' values loaded at a time.
template <typename F>
__device__ __forceinline__ void list_visit(const FlagList& L, F f) {
  const int lane = threadIdx.x & 31;
  int wlo, whi;
  warp_slice(L.cnt, wlo, whi);
  for (int e0 = wlo; e0 < whi; e0 += 128) {
    double a1[4], a2[4], t1[4], t2[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int e = min(e0 + 32 * u + lane, L.cnt - 1);
      a1[u] = L.a1[e]; a2[u] = L.a2[e]; t1[u] = L.t1[e]; t2[u] = L.t2[e];
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (e0 + 32 * u >= whi) break;  // warp-uniform
      const int e = e0 + 32 * u + lane;
      f(e, e < whi, a1[u], a2[u], t1[u], t2[u]);
    }
  }
}

// First (up to) four entries with pred, in entry order, and how many satisfy it.  One block.
template <typename Pred>
__device__ int list_first4(const FlagList& L, Pred pred, Scratch& sc, int (&out)[4]) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  int c = 0, mine[4] = {-1, -1, -1, -1};  // per warp, identical in every lane
  list_visit(L, [&](int e, bool valid, double a1, double a2, double t1, double t2) {
    unsigned b = __ballot_sync(0xffffffffu, valid && pred(e, a1, a2, t1, t2));
    const int base = e - lane;
    const int nb = __popc(b);
    for (int r = c; r < 4 && b; ++r) {  // only the first four of the warp are kept
      mine[r] = base + __ffs(b) - 1;
      b &= b - 1;
    }
    c += nb;
  });
  __syncthreads();
  if (lane == 0) {
    sc.i[w] = c;
    for (int r = 0; r < 4; ++r) sc.d[w][r] = (double)mine[r];
  }
  __syncthreads();
  int total = 0, have = 0;
  for (int a = 0; a < 4; ++a) out[a] = -1;
  for (int ww = 0; ww < DT / 32; ++ww) {
    const int cw = sc.i[ww];
    for (int r = 0; r < 4 && r < cw && have < 4; ++r) out[have++] = (int)sc.d[ww][r];
    total += cw;
  }
  __syncthreads();
  return total;
}

// Number of entries with pred.
template <typename Pred>
__device__ int list_count(const FlagList& L, Pred pred, Scratch& sc) {
  int c = 0;
  list_visit(L, [&](int e, bool valid, double a1, double a2, double t1, double t2) { c += (valid && pred(e, a1, a2, t1, t2)) ? 1 : 0; });
  return block_sum(c, sc);
}

// ---------------------------------------------------------------------------------------------------------------
// phase 2 / second decision.  One block.  post_repair = 0: Level-P on the syndromes as computed.  post_repair = 1:
// re-flags the updated syndromes and accepts CLEAN or point errors only.
// Every comparison uses the threshold of its own line: tau + tolx[line].  The flagged lines of both sides are compacted
// into sorted lists first, so every later pass touches flagged lines only, from contiguous arrays.
// ---------------------------------------------------------------------------------------------------------------
#ifdef GECC_FINE_STAMPS
#define DSTAMP()                                                                     \
  do {                                                                               \
    __syncthreads();                                                                 \
    if (threadIdx.x == 0 && bufs.stamps[0] + 1 < (unsigned long long)kMaxPhaseStamps) { \
      bufs.stamps[bufs.stamps[0] + 1] = globaltimer_ns();                            \
      bufs.stamps[0] += 1;                                                           \
    }                                                                                \
  } while (0)
#else
#define DSTAMP() do { } while (0)
#endif

// Shared-memory storage for the two lists of a decision about few lines (<= 8 per side): no global round trips.
struct SmallLists {
  int idx[2][8];
  double a1[2][8], a2[2][8], t1[2][8], t2[2][8];
};
__device__ __forceinline__ FlagList small_list(SmallLists* sm, int w) {
  FlagList L;
  L.idx = sm->idx[w]; L.a1 = sm->a1[w]; L.a2 = sm->a2[w]; L.t1 = sm->t1[w]; L.t2 = sm->t2[w]; L.cnt = 0;
  return L;
}

// One check (c = 0 plain, 1 weighted) of line idx of the parity block of C_bar: P_r[idx][c] (is_row) / P_c[c][idx].
__device__ __forceinline__ double parity_symbol(int dtype, const float* P_r, const float* P_c, int m, bool is_row, int64_t idx, int c) {
  const int nl = dtype == GECC_BF16 ? 3 : 1;
  double v = 0.0;
  for (int l = 0; l < nl; ++l) v += (double)__ldcg(is_row ? P_r + idx * GECC_PR_LD + 3 * c + l : P_c + (int64_t)(3 * c + l) * m + idx);
  return v;
}

struct DecideBufs {
  int dtype, single;
  const float* P_r;  // for the global checks of Eq. (4)
  const float* P_c;
  const float* P_g;  // null: no global checks
  SmallLists* small;
  unsigned long long* stamps;
  uint8_t* rflag;  // [align16(n)]
  uint8_t* qflag;  // [align16(m)]
  int* votes;      // [max(n, m)]
  FlagList rows, cols;
};

__device__ __noinline__ void decide(DecodeState* st, const double* syn, const double* tolx, DecideBufs bufs, int n, int m, int level, int post_repair, int s_in,
                       int t_in, Scratch& sc) {
  const double* r1 = syn; const double* r2 = syn + n; const double* q1 = syn + 2 * (int64_t)n; const double* q2 = syn + 2 * (int64_t)n + m;
  const double* xr1 = tolx; const double* xr2 = tolx + n; const double* xq1 = tolx + 2 * (int64_t)n; const double* xq2 = tolx + 2 * (int64_t)n + m;
  const double t_r1 = st->tau[0], t_r2 = st->tau[1], t_q1 = st->tau[2], t_q2 = st->tau[3];
  const int s = s_in, t = t_in;  // flagged rows, flagged columns (counted by the grid)
  __syncthreads();
#ifdef GECC_DEBUG_PRINT
  if (threadIdx.x == 0) {
    printf("decide post=%d s=%d t=%d tau %g %g %g %g\n", post_repair, s, t, t_r1, t_r2, t_q1, t_q2);
    for (int sd = 0; sd < 2; ++sd)
      for (int e = 0; e < 8 && e < (sd == 0 ? s : t); ++e)
        printf("  side %d line %d a1 %g a2 %g t1 %g t2 %g\n", sd, st->el[sd].idx[e], st->el[sd].a1[e], st->el[sd].a2[e], st->el[sd].t1[e], st->el[sd].t2[e]);
  }
#endif

  // ---- decision; every thread computes the same scalars ----
  int verdict = GECC_UNCORRECTABLE;
  int nS = 0, S[2] = {-1, -1}, whole[2] = {0, 0};
  int npts = 0, pt_s[kMaxPoints], pt_l[kMaxPoints];
  double pt_x[kMaxPoints];
  int hidden_n = 0, hidden_s[2], hidden_l[2];
  double hidden_x[2];
  const bool rows_short = s <= t;
  // oriented views: "short" side holds the <= 2 faulty lines, "long" side supplies the syndromes used to correct
  const double* s1 = rows_short ? r1 : q1; const double* s2 = rows_short ? r2 : q2;
  const double* xs1 = rows_short ? xr1 : xq1; const double* xs2 = rows_short ? xr2 : xq2;
  const int n_short = rows_short ? n : m, n_long = rows_short ? m : n;
  const double tau_s1_ = rows_short ? t_r1 : t_q1, tol_s_ = rows_short ? t_r2 : t_q2;
  auto tau_s1 = [&](int i) { return tau_s1_ + __ldcg(xs1 + i); };
  auto tol_s = [&](int i) { return tol_s_ + __ldcg(xs2 + i); };
  auto S1v = [&](int i) { return __ldcg(s1 + i); };
  auto S2v = [&](int i) { return __ldcg(s2 + i); };

  bool ok = true;
  if (s == 0 && t == 0) { verdict = GECC_CLEAN; ok = false; }
  else if (s >= 3 && t >= 3) ok = false;  // min(s,t) >= 3
  else if (bufs.single && !(s == 1 && t == 1)) ok = false;  // single checksum: one bad row crossing one bad column, nothing else

  DSTAMP();
  FlagList SL = rows_short ? bufs.rows : bufs.cols, LL = rows_short ? bufs.cols : bufs.rows;
  int Sflag[2] = {-1, -1};
  int nSflag = 0;
  if (ok) {
    const int cnt_short = rows_short ? s : t, cnt_long = rows_short ? t : s;
    if (cnt_short <= 8) { SL = small_list(bufs.small, 0); collect_early(&st->el[rows_short ? 0 : 1], cnt_short, SL, false, sc); }
    else compact_flagged(rows_short ? bufs.rflag : bufs.qflag, n_short, nullptr, nullptr, nullptr, nullptr, 0.0, 0.0, SL, false, sc);
    if (cnt_long <= 8) { LL = small_list(bufs.small, 1); collect_early(&st->el[rows_short ? 1 : 0], cnt_long, LL, true, sc); }
    else
      compact_flagged(rows_short ? bufs.qflag : bufs.rflag, n_long, rows_short ? q1 : r1, rows_short ? q2 : r2, rows_short ? xq1 : xr1,
                      rows_short ? xq2 : xr2, rows_short ? t_q1 : t_r1, rows_short ? t_q2 : t_r2, LL, true, sc);
    DSTAMP();
    nSflag = SL.cnt;
    if (nSflag > 0) Sflag[0] = SL.idx[0];
    if (nSflag > 1) Sflag[1] = SL.idx[1];
    nS = nSflag; S[0] = Sflag[0]; S[1] = Sflag[1];
    // A flagged long-side line is explained by S if |S| = 2 (Theorem 2) or S = {s} and its two syndromes
    // are in the ratio of the weight of s (one error in line s).
    const bool single = bufs.single != 0;
    auto explained = [&](double l1, double l2, double tl2, int cnt, int a0) { return cnt == 2 || (cnt == 1 && (single || fabs(l2 - (double)(a0 + 1) * l1) <= tl2)); };
    const int nU = list_count(LL, [&](int, double l1, double l2, double, double tl2) { return !explained(l1, l2, tl2, nS, S[0]); }, sc);
    DSTAMP();
    if (nU > 0) {
      // Input faults leave their own side's syndromes silent (reading R7): locate the line by the weighted ratio.
      int* votes = bufs.votes;
      for (int i = threadIdx.x; i < n_short; i += DT) votes[i] = 0;
      if (threadIdx.x == 0) { sc.flag = 0; sc.cnt = 0; }
      __syncthreads();
      {
        // votes of one thread's contiguous entries mostly name the same line: count runs, one atomic per run
        int run_c = -1, run_n = 0;
        auto flush = [&]() {
          if (run_n > 0 && atomicAdd(&votes[run_c], run_n) == 0) {  // first votes for this line: remember it
            const int pslot = atomicAdd(&sc.cnt, 1);
            if (pslot < 8) sc.idx[pslot] = run_c;
          }
        };
        list_visit(LL, [&](int, bool valid, double l1, double l2, double tl1, double tl2) {
          if (!valid || explained(l1, l2, tl2, nS, S[0])) return;
          const double elig = tl1 > tl2 ? tl1 : tl2;  // ratio resolvable under the weighted noise
          if (!(fabs(l1) > elig)) return;              // too weak to vote
          const double ratio = rint(l2 / l1);
          const bool good = ratio >= 1.0 && ratio <= (double)n_short && fabs(l2 - ratio * l1) <= tl2;
          if (good) {
            const int cand = (int)ratio - 1;
            if (cand != run_c) { flush(); run_c = cand; run_n = 0; }
            ++run_n;
          } else atomicExch(&sc.flag, 1);
        });
        flush();
      }
      __threadfence_block();
      __syncthreads();
      DSTAMP();
      const bool all_valid = sc.flag == 0;
      const int distinct = sc.cnt;
      int cand[8];
      for (int a = 0; a < 8; ++a) cand[a] = a < distinct ? sc.idx[a] : -1;
      __syncthreads();
      if (nS == 0) {
        if (!all_valid || distinct == 0 || distinct > 2) ok = false;
        else {
          nS = distinct;
          S[0] = distinct == 2 ? min(cand[0], cand[1]) : cand[0];
          S[1] = distinct == 2 ? max(cand[0], cand[1]) : -1;
        }
      } else {
        unsigned long long key = 0;
        if (distinct <= 8) {
          for (int a = 0; a < distinct; ++a)
            if (cand[a] != S[0]) {
              const unsigned long long kk = ((unsigned long long)votes[cand[a]] << 32) | (unsigned long long)(0x7FFFFFFF - cand[a]);  // mode, ties -> smallest
              key = kk > key ? kk : key;
            }
        } else {
          for (int i = threadIdx.x; i < n_short; i += DT)
            if (i != S[0] && votes[i] > 0) {
              const unsigned long long kk = ((unsigned long long)votes[i] << 32) | (unsigned long long)(0x7FFFFFFF - i);
              key = kk > key ? kk : key;
            }
          key = block_max(key, sc);
        }
        if (key == 0) ok = false;
        else {
          const int best = 0x7FFFFFFF - (int)(key & 0xFFFFFFFFull);
          const int a = S[0];
          S[0] = a < best ? a : best; S[1] = a < best ? best : a; nS = 2;
        }
      }
      if (ok && list_count(LL, [&](int, double l1, double l2, double, double tl2) { return !explained(l1, l2, tl2, nS, S[0]); }, sc) > 0) ok = false;
    }
    if (ok && nS == 0) ok = false;
    // single checksum: the two plain syndromes must agree on the magnitude (the weighted ones are not consulted)
    if (ok && single && !(fabs(S1v(S[0]) - LL.a1[0]) <= tau_s1(S[0]) + LL.t1[0])) ok = false;
    DSTAMP();
  }

  if (ok) {
    const int nl = LL.cnt;
    const double w1 = (double)(S[0] + 1), w2 = (double)(S[1] + 1);
    // |S| = 2: x2 = (l2 - w1 l1) / (w2 - w1), x1 = l1 - x2.  The weighted syndrome's noise enters divided by (w2 - w1).
    auto xhat = [&](int idx, int e) -> double {
      if (nS == 1) return LL.a1[e];
      const double x2 = (LL.a2[e] - w1 * LL.a1[e]) / (w2 - w1);
      return idx == 0 ? LL.a1[e] - x2 : x2;
    };
    auto tau_loc = [&](int e) -> double {
      if (nS == 1) return LL.t1[e];
      const double amp = 2.0 * LL.t2[e] / fabs(w2 - w1);
      return amp > LL.t1[e] ? amp : LL.t1[e];
    };
    // Two flagged rows and two flagged columns: within the two-error budget the errors sit on one diagonal of the 2x2
    // block.  In exact arithmetic the 2x2 solve below finds which; under fp32 noise its weighted right-hand side is
    // divided by (w2 - w1), so first test the two diagonals against all eight syndromes: plain sums must match pairwise,
    // weighted ones within their own threshold.  Exactly one consistent diagonal decides; none -> general solve
    // (more than two errors in the block, still E(2,2), Theorem 1); both -> indistinguishable under the noise.
    bool decided = false;
    if (nS == 2 && nSflag == 2 && nl == 2) {
      const int a = S[0], b = S[1];
      auto diag_ok = [&](int ea, int eb) {  // error of line a in long entry ea, error of line b in long entry eb
        const int ca = LL.idx[ea], cb = LL.idx[eb];
        return fabs(S1v(a) - LL.a1[ea]) <= tau_s1(a) + LL.t1[ea] && fabs(S1v(b) - LL.a1[eb]) <= tau_s1(b) + LL.t1[eb] &&
               fabs(LL.a2[ea] - (double)(a + 1) * LL.a1[ea]) <= LL.t2[ea] && fabs(LL.a2[eb] - (double)(b + 1) * LL.a1[eb]) <= LL.t2[eb] &&
               fabs(S2v(a) - (double)(ca + 1) * S1v(a)) <= tol_s(a) && fabs(S2v(b) - (double)(cb + 1) * S1v(b)) <= tol_s(b);
      };
      const bool h1 = diag_ok(0, 1), h2 = diag_ok(1, 0);
      if (h1 != h2) {
        const int ea = h1 ? 0 : 1, eb = h1 ? 1 : 0;
        pt_s[0] = a; pt_l[0] = LL.idx[ea]; pt_x[0] = LL.a1[ea];
        pt_s[1] = b; pt_l[1] = LL.idx[eb]; pt_x[1] = LL.a1[eb];
        npts = 2;
        decided = true;
      } else if (h1 && h2) ok = false;
    }
    for (int idx = 0; idx < nS && ok && !decided; ++idx) {
      const int sl = S[idx];
      const bool in_flag = (sl == Sflag[0] && nSflag > 0) || (sl == Sflag[1] && nSflag > 1);
      int g[4];
      const int ncols = list_first4(LL, [&](int, double l1, double l2, double tl1, double tl2) {
        double x = l1, tl = tl1;
        if (nS == 2) {
          const double x2 = (l2 - w1 * l1) / (w2 - w1);
          x = idx == 0 ? l1 - x2 : x2;
          const double amp = 2.0 * tl2 / fabs(w2 - w1);
          tl = amp > tl1 ? amp : tl1;
        }
        return fabs(x) > tl;
      }, sc, g);
      // a single error explaining the line's OWN two syndromes: their ratio is an integer weight
      int hidden_at = -1;
      if (in_flag && ncols >= 3) {
        const double v1 = S1v(sl), v2 = S2v(sl);
        if (fabs(v1) > tau_s1(sl)) {
          const double ratio = rint(v2 / v1);
          if (ratio >= 1.0 && ratio <= (double)n_long && fabs(v2 - ratio * v1) <= tol_s(sl)) hidden_at = (int)ratio - 1;
        }
      }
      if (!in_flag) whole[idx] = 1;  // located by the ratio only: an input fault
      else if (ncols >= 3 && hidden_at >= 0) {
        // three or more bad symbols in a line whose own syndromes point at one column: an input fault shifted the whole
        // line consistently and one C error hides in it
        whole[idx] = 1;
        hidden_s[hidden_n] = sl; hidden_l[hidden_n] = hidden_at; hidden_x[hidden_n] = S1v(sl); ++hidden_n;
      } else if (ncols > kMaxPointsPerLine) {
        // E(s,t), t large, the errors known to sit in this line: every t* is corrected by the long-side syndromes
        // (Theorem 2); too many to list, so reported and corrected as a whole line
        whole[idx] = 1;
      } else if (ncols == 0) ok = false;  // flagged line with nothing locatable (e.g. a parity-symbol fault, R11)
      else {
        for (int a = 0; a < ncols && npts < kMaxPoints; ++a) {
          const int e = g[a];
          double x = xhat(idx, e);
          if (nS == 2 && !(fabs(xhat(1 - idx, e)) > tau_loc(e))) x = LL.a1[e];  // the other line is clean here: plain syndrome
          pt_s[npts] = sl; pt_l[npts] = LL.idx[e]; pt_x[npts] = x; ++npts;
        }
      }
    }
    // One whole line and a single point in the other line: the 2x2 solve divides the weighted syndrome's noise by
    // (w2 - w1), which is 1 for adjacent lines.  The point's own line holds nothing else, so its plain short-side syndrome
    // IS the point's value; the whole line then takes the rest of each long-side plain syndrome (see the patch).
    if (ok && nS == 2 && whole[0] != whole[1]) {
      const int pl = whole[0] ? 1 : 0;
      int cntp = 0, which = -1;
      for (int a = 0; a < npts; ++a)
        if (pt_s[a] == S[pl]) { ++cntp; which = a; }
      if (cntp == 1 && fabs(S1v(S[pl])) > tau_s1(S[pl])) pt_x[which] = S1v(S[pl]);
    }
    if (ok) verdict = GECC_CORRECTED;
    DSTAMP();
  }
  if (post_repair && verdict == GECC_CORRECTED && (whole[0] || whole[1])) verdict = GECC_UNCORRECTABLE;

  // Nothing locatable in C, one flagged line on one side, nothing on the other, only ONE of its two checks off: a local
  // parity symbol of C_bar itself may be faulty.  The parity columns P_r / rows P_c are codewords too, checked by the
  // global parity P_g (Eq. 4): sum_i w_d(i) P_r[i][c] - P_g[d][c] must show the same error delta at the
  // line's weight: delta (d = 0) and (i + 1) delta (d = 1).  Then C is intact and the symbol is what gets corrected.
  int par_kind = -1, par_line = -1, par_c = -1;
  double par_delta = 0.0;
  if (!ok && verdict == GECC_UNCORRECTABLE && !post_repair && !bufs.single && bufs.P_g && s + t == 1) {
    const bool is_row = s == 1;
    const DecodeState::Early& E = st->el[is_row ? 0 : 1];
    const int idx = __ldcg(&E.idx[0]);
    const double a1 = __ldcg(&E.a1[0]), a2 = __ldcg(&E.a2[0]), tl1 = __ldcg(&E.t1[0]), tl2 = __ldcg(&E.t2[0]);
    const bool off1 = !(fabs(a1) <= tl1), off2 = !(fabs(a2) <= tl2);
    if (off1 != off2) {
      const int c = off1 ? 0 : 1;
      const double delta = -(c == 0 ? a1 : a2), tl = c == 0 ? tl1 : tl2;
      const int len = is_row ? n : m;
      double v4[4] = {0.0, 0.0, 0.0, 0.0};
      for (int64_t i = threadIdx.x; i < len; i += DT) {
        const double pv = parity_symbol(bufs.dtype, bufs.P_r, bufs.P_c, m, is_row, i, c);
        v4[0] += pv;
        v4[1] += (double)(i + 1) * pv;
      }
      block_sum4(v4, sc);
      const int nl = bufs.dtype == GECC_BF16 ? 3 : 1;
      double g[2];
      for (int d = 0; d < 2; ++d) {
        double pg = 0.0;  // P_g[d][c] for the row side, P_g[c][d] for the column side (limb products)
        for (int l = 0; l < nl; ++l)
          for (int l2 = 0; l2 < nl; ++l2)
            pg += (double)__ldcg(bufs.P_g + (3 * (is_row ? d : c) + l) * GECC_PR_LD + 3 * (is_row ? c : d) + l2);
        g[d] = v4[d] - pg;
      }
      const double tau_c = is_row ? (c == 0 ? t_r1 : t_r2) : (c == 0 ? t_q1 : t_q2);
      const double tg0 = tau_c * sqrt((double)len), tg1 = tg0 * sqrt((len + 1.0) * (2.0 * len + 1.0) / 6.0);
      // the global check must CONFIRM the error (stand out of its own tolerance), not merely fail to contradict it
      if (fabs(delta) > 4.0 * tg0 && fabs(g[0] - delta) <= tg0 + tl && fabs(g[1] - (double)(idx + 1) * delta) <= tg1 + (double)(idx + 1) * tl) {
        par_kind = is_row ? GECC_KIND_PR : GECC_KIND_PC; par_line = idx; par_c = c; par_delta = delta;
        verdict = GECC_CORRECTED;
      }
    }
  }

  __syncthreads();
  if (threadIdx.x == 0) {
    if (!post_repair) {
      st->n_row_flags0 = s;
      st->n_col_flags0 = t;
    }
    st->verdict = verdict;
    st->rows_short = rows_short ? 1 : 0;
    int nf = 0;
    gecc_found_t* f = st->found;
    if (post_repair) {
      if (verdict == GECC_UNCORRECTABLE) nf = 0;
      else {
        for (int a = 0; a < st->n_fa && nf < GECC_MAX_FOUND; ++a) f[nf++] = gecc_found_t{GECC_KIND_A, st->fa[a].row, st->fa[a].col, 0, st->fa[a].e};
        for (int a = 0; a < st->n_fb && nf < GECC_MAX_FOUND; ++a) f[nf++] = gecc_found_t{GECC_KIND_B, st->fb[a].row, st->fb[a].col, 0, st->fb[a].e};
        verdict = GECC_CORRECTED;
        st->verdict = verdict;
      }
    }
    st->par_kind = par_kind; st->par_line = par_line; st->par_c = par_c; st->par_delta = par_delta;
    if (par_kind >= 0) {
      st->nS = 0; st->n_points = 0; st->whole_line[0] = st->whole_line[1] = 0;
      f[nf++] = par_kind == GECC_KIND_PR ? gecc_found_t{GECC_KIND_PR, par_line, par_c, 0, par_delta} : gecc_found_t{GECC_KIND_PC, par_c, par_line, 0, par_delta};
    } else if (verdict == GECC_CORRECTED) {
      st->nS = nS; st->S[0] = S[0]; st->S[1] = S[1]; st->whole_line[0] = whole[0]; st->whole_line[1] = whole[1];
      st->n_points = npts;
      for (int a = 0; a < npts; ++a) { st->pt_s[a] = pt_s[a]; st->pt_l[a] = pt_l[a]; st->pt_x[a] = pt_x[a]; }
      for (int a = 0; a < nS; ++a)
        if (whole[a] && nf < GECC_MAX_FOUND)
          f[nf++] = rows_short ? gecc_found_t{GECC_KIND_ROW, S[a], -1, 0, 0.0} : gecc_found_t{GECC_KIND_COL, -1, S[a], 0, 0.0};
      for (int a = 0; a < npts && nf < GECC_MAX_FOUND; ++a)
        f[nf++] = rows_short ? gecc_found_t{GECC_KIND_C, pt_s[a], pt_l[a], 0, pt_x[a]} : gecc_found_t{GECC_KIND_C, pt_l[a], pt_s[a], 0, pt_x[a]};
      for (int a = 0; a < hidden_n && nf < GECC_MAX_FOUND; ++a)
        f[nf++] = rows_short ? gecc_found_t{GECC_KIND_C, hidden_s[a], hidden_l[a], 0, hidden_x[a]} : gecc_found_t{GECC_KIND_C, hidden_l[a], hidden_s[a], 0, hidden_x[a]};
      sort_found(f, nf);
    } else {
      st->nS = 0; st->n_points = 0; st->whole_line[0] = st->whole_line[1] = 0;
    }
    st->n_found = nf;
    if (!post_repair) {
      st->need_verify = (level >= 1 && (verdict == GECC_UNCORRECTABLE || (verdict == GECC_CORRECTED && (whole[0] || whole[1])))) ? 1 : 0;
      st->repaired = 0;
      st->n_fa = st->n_fb = 0;
    }
    __threadfence();
  }
}

// ---------------------------------------------------------------------------------------------------------------
// The same decision for the patterns that make up almost every call -- at most two flagged rows and two flagged columns,
// all of them explained by point errors: (1,1) one symbol, (1,2) / (2,1) two symbols in one line, (2,2) two symbols on
// a diagonal -- taken by ONE thread straight from the (at most four) noted lines, no lists, no block-wide passes.
// Same tests, same order, same outcome as decide(); anything else (input faults, refusals, single-checksum mode, more
// lines) returns false and goes through decide().  Thread 0 of block 0.
// ---------------------------------------------------------------------------------------------------------------
struct NotedLine { int idx; double a1, a2, t1, t2; };

__device__ __noinline__ bool decide_small(DecodeState* st, int post_repair, int s, int t, int single) {
  if (single || s < 1 || t < 1 || s > 2 || t > 2) return false;
  NotedLine R[2], Q[2];
  for (int e = 0; e < 2; ++e) {
    R[e].idx = -1; Q[e].idx = -1;
    if (e < s) { const DecodeState::Early& E = st->el[0]; R[e].idx = __ldcg(&E.idx[e]); R[e].a1 = __ldcg(&E.a1[e]); R[e].a2 = __ldcg(&E.a2[e]); R[e].t1 = __ldcg(&E.t1[e]); R[e].t2 = __ldcg(&E.t2[e]); }
    if (e < t) { const DecodeState::Early& E = st->el[1]; Q[e].idx = __ldcg(&E.idx[e]); Q[e].a1 = __ldcg(&E.a1[e]); Q[e].a2 = __ldcg(&E.a2[e]); Q[e].t1 = __ldcg(&E.t1[e]); Q[e].t2 = __ldcg(&E.t2[e]); }
  }
  if (s == 2 && R[1].idx < R[0].idx) { const NotedLine x = R[0]; R[0] = R[1]; R[1] = x; }
  if (t == 2 && Q[1].idx < Q[0].idx) { const NotedLine x = Q[0]; Q[0] = Q[1]; Q[1] = x; }
  const bool rows_short = s <= t;
  const NotedLine* S = rows_short ? R : Q;   // short side: the lines that hold the errors
  const NotedLine* L = rows_short ? Q : R;   // long side: its syndromes give the magnitudes
  const int nS = rows_short ? s : t, nL = rows_short ? t : s;
  int npts = 0, pt_s[2], pt_l[2];
  double pt_x[2];
  if (nS == 1) {
    // every flagged long-side line must be explained by the one short line: its two syndromes in the ratio of that line's weight
    for (int e = 0; e < nL; ++e)
      if (!(fabs(L[e].a2 - (double)(S[0].idx + 1) * L[e].a1) <= L[e].t2)) return false;
    for (int e = 0; e < nL; ++e)
      if (fabs(L[e].a1) > L[e].t1) { pt_s[npts] = S[0].idx; pt_l[npts] = L[e].idx; pt_x[npts] = L[e].a1; ++npts; }
    if (npts == 0) return false;
  } else {
    if (nL != 2) return false;
    auto diag_ok = [&](int ea, int eb) {  // error of short line 0 in long entry ea, of short line 1 in long entry eb
      return fabs(S[0].a1 - L[ea].a1) <= S[0].t1 + L[ea].t1 && fabs(S[1].a1 - L[eb].a1) <= S[1].t1 + L[eb].t1 &&
             fabs(L[ea].a2 - (double)(S[0].idx + 1) * L[ea].a1) <= L[ea].t2 && fabs(L[eb].a2 - (double)(S[1].idx + 1) * L[eb].a1) <= L[eb].t2 &&
             fabs(S[0].a2 - (double)(L[ea].idx + 1) * S[0].a1) <= S[0].t2 && fabs(S[1].a2 - (double)(L[eb].idx + 1) * S[1].a1) <= S[1].t2;
    };
    const bool h1 = diag_ok(0, 1), h2 = diag_ok(1, 0);
    if (h1 == h2) return false;
    const int ea = h1 ? 0 : 1, eb = h1 ? 1 : 0;
    pt_s[0] = S[0].idx; pt_l[0] = L[ea].idx; pt_x[0] = L[ea].a1;
    pt_s[1] = S[1].idx; pt_l[1] = L[eb].idx; pt_x[1] = L[eb].a1;
    npts = 2;
  }
  // the plan and the report entries, as decide() leaves them
  if (!post_repair) { st->n_row_flags0 = s; st->n_col_flags0 = t; }
  st->verdict = GECC_CORRECTED;
  st->rows_short = rows_short ? 1 : 0;
  st->par_kind = -1; st->par_line = -1; st->par_c = -1; st->par_delta = 0.0;
  st->nS = nS; st->S[0] = S[0].idx; st->S[1] = nS > 1 ? S[1].idx : -1; st->whole_line[0] = 0; st->whole_line[1] = 0;
  st->n_points = npts;
  int nf = 0;
  gecc_found_t* f = st->found;
  if (post_repair) {
    for (int a = 0; a < st->n_fa && nf < GECC_MAX_FOUND; ++a) f[nf++] = gecc_found_t{GECC_KIND_A, st->fa[a].row, st->fa[a].col, 0, st->fa[a].e};
    for (int b = 0; b < st->n_fb && nf < GECC_MAX_FOUND; ++b) f[nf++] = gecc_found_t{GECC_KIND_B, st->fb[b].row, st->fb[b].col, 0, st->fb[b].e};
  }
  for (int a = 0; a < npts; ++a) {
    st->pt_s[a] = pt_s[a]; st->pt_l[a] = pt_l[a]; st->pt_x[a] = pt_x[a];
    if (nf < GECC_MAX_FOUND) f[nf++] = rows_short ? gecc_found_t{GECC_KIND_C, pt_s[a], pt_l[a], 0, pt_x[a]} : gecc_found_t{GECC_KIND_C, pt_l[a], pt_s[a], 0, pt_x[a]};
  }
  sort_found(f, nf);
  st->n_found = nf;
  if (!post_repair) { st->need_verify = 0; st->repaired = 0; st->n_fa = st->n_fb = 0; }
  __threadfence();
  return true;
}

// Level-X: the lines of A / B whose recomputed checks differ from the stored ones were collected by the whole grid; a
// single corrupted symbol per line is located by the ratio of its two differences.  Every block evaluates the (at most
// 2 x kMaxInputFaults) candidates itself, so no barrier separates this from the repair.  One thread per block.
// rel_tol bounds the rounding of the difference of two passes: bf16 symbols are summed in groups of 8 in fp32 with 6-bit
// weights (error <= 2^-24 x 56 (|e| + |a|) in the one group that changed), fp32 symbols in fp64 throughout.
struct Faults {
  int ok, repaired, nfa, nfb, ncb;
  InputFault fa[kMaxInputFaults], fb[kMaxInputFaults];
  DecodeState::Cand cb[kMaxInputFaults];
};
__device__ void verify_compare(const DecodeState* st, int dtype, int n, int m, double sigma_a, double sigma_b, Faults& F) {
  const double rel_tol = dtype == GECC_BF16 ? 1e-5 : 1e-11;
  F.ok = 1; F.nfa = 0; F.nfb = 0; F.ncb = 0;
  for (int side = 0; side < 2; ++side) {
    const int cnt = __ldcg(side == 0 ? &st->cnt_a : &st->cnt_b);
    const DecodeState::Cand* src = side == 0 ? st->ca : st->cb;
    const int nline = side == 0 ? n : m;  // number of symbols each check spans
    const double sigma = side == 0 ? sigma_a : sigma_b;
    if (cnt > kMaxInputFaults) { F.ok = 0; continue; }
    DecodeState::Cand cd[kMaxInputFaults];
    for (int a = 0; a < cnt; ++a) { cd[a].l = __ldcg(&src[a].l); cd[a].d1 = __ldcg(&src[a].d1); cd[a].d2 = __ldcg(&src[a].d2); }
    for (int a = 0; a < cnt; ++a)  // ascending by line: the grid filled the slots in no particular order
      for (int b = a + 1; b < cnt; ++b)
        if (cd[b].l < cd[a].l) { const DecodeState::Cand x = cd[a]; cd[a] = cd[b]; cd[b] = x; }
    for (int a = 0; a < cnt; ++a) {
      const int l = cd[a].l;
      const double d1 = cd[a].d1, d2 = cd[a].d2;
      const double ratio = rint(d2 / d1);
      const double tol = rel_tol * (fabs(d1) + 8.0 * sigma) * (dtype == GECC_BF16 ? 1.0 : (double)nline);
      if (!(fabs(d1) > 0.0) || !(ratio >= 1.0 && ratio <= (double)nline) || !(fabs(d2 - ratio * d1) <= tol)) { F.ok = 0; break; }
      InputFault f;
      if (side == 0) { f.row = (int)ratio - 1; f.col = l; } else { f.row = l; f.col = (int)ratio - 1; }
      f.e = d1;
      if (side == 0) F.fa[F.nfa++] = f; else { F.cb[F.ncb++] = cd[a]; F.fb[F.nfb++] = f; }
    }
  }
  if (!F.ok) { F.nfa = F.nfb = 0; }
  F.repaired = F.ok && (F.nfa + F.nfb > 0);
}
// Block 0 publishes the outcome in the decoder state (read by the second decision and the report).
__device__ void publish_faults(DecodeState* st, const Faults& F) {
  st->verify_ok_a = st->verify_ok_b = F.ok;
  st->n_fa = F.nfa; st->n_fb = F.nfb;
  for (int a = 0; a < F.nfa; ++a) st->fa[a] = F.fa[a];
  for (int b = 0; b < F.nfb; ++b) st->fb[b] = F.fb[b];
  if (!F.ok) {
    st->verdict = GECC_UNCORRECTABLE_INPUT;
    st->n_found = 0; st->nS = 0; st->n_points = 0; st->whole_line[0] = st->whole_line[1] = 0;
  }
  st->repaired = F.repaired;  // repaired: the Level-P plan is dropped; otherwise (memory intact: transient fault) it is kept
  __threadfence();
}

template <typename T>
__device__ __forceinline__ float load_sym(const T* p);
template <>
__device__ __forceinline__ float load_sym<__nv_bfloat16>(const __nv_bfloat16* p) { return __bfloat162float(*p); }
template <>
__device__ __forceinline__ float load_sym<float>(const float* p) { return *p; }

template <typename T>
__device__ __forceinline__ void patch_sym(T* X, float* X_lo, int64_t idx, double e);
template <>
__device__ __forceinline__ void patch_sym<__nv_bfloat16>(__nv_bfloat16* X, float*, int64_t idx, double e) {
  X[idx] = __double2bfloat16((double)__bfloat162float(X[idx]) - e);
}
template <>
__device__ __forceinline__ void patch_sym<float>(float* X, float* X_lo, int64_t idx, double e) {
  const float v = (float)((double)X[idx] - e);
  X[idx] = v;
  if (X_lo) X_lo[idx] = v - tf32_trunc(v);
}

// Products of two symbols: exact in fp32 for bf16 x bf16 (16 significant bits); fp32 x fp32 goes through fp64.
template <typename T>
__device__ __forceinline__ void load_vec(const T* src, float (&x)[Vec<T>::V]) {
  if (sizeof(T) == 2) {
    const uint4 q = __ldcg(reinterpret_cast<const uint4*>(src));
    const uint32_t ww[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
    for (int i2 = 0; i2 < Vec<T>::V / 2; ++i2) { x[2 * i2] = __uint_as_float(ww[i2] << 16); x[2 * i2 + 1] = __uint_as_float(ww[i2] & 0xFFFF0000u); }
  } else {
    const float4 q = __ldcg(reinterpret_cast<const float4*>(src));
    x[0] = q.x; x[1] = q.y; x[2] = q.z; x[3] = q.w;
  }
}

// 16-byte load through L2 (the operands were patched by this kernel: not the read-only path).  volatile keeps a run of
// these together, as ld_stream does.
__device__ __forceinline__ uint4 ld_cg16(const void* p) {
  uint4 u;
  asm volatile("ld.global.cg.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(u.x), "=r"(u.y), "=r"(u.z), "=r"(u.w) : "l"(p));
  return u;
}

// One warp: partial[c] = sum over rows r of chunk `chunk` of w[r wstride] x[r][c] for the 32 V columns of strip `strip`.
// Eight products at a time are summed in fp32 (bf16 symbols) and folded into fp64; fp32 symbols are multiplied in fp64.
// All eight 16-byte loads of a group are in flight before the first use (join_loads, encode_core.cuh); rows past the end
// re-read the last row with weight zero.
template <typename T>
__device__ __forceinline__ void wcolsum_warp_item(const T* __restrict__ X, int64_t rows, int64_t cols, int64_t ld, const T* __restrict__ w,
                                                  int64_t wstride, double* __restrict__ partial, int strip, int chunk) {
  constexpr int V = Vec<T>::V;
  const int lane = threadIdx.x & 31;
  const int64_t c0 = ((int64_t)strip * 32 + lane) * V;
  if (c0 >= cols) return;
  double S[V];
#pragma unroll
  for (int v = 0; v < V; ++v) S[v] = 0.0;
  const int64_t rbase = (int64_t)chunk * kRecompRows;
  const uint32_t rz = (uint32_t)((uint64_t)rows >> 40);
#pragma unroll 2
  for (int g = 0; g < kRecompRows / 8; ++g) {
    uint4 raw[8];
    float wr[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int64_t r = rbase + 8 * g + u, rc = r < rows ? r : rows - 1;
      raw[u] = ld_cg16(X + rc * ld + c0);
      wr[u] = load_sym<T>(w + rc * wstride);
      if (r >= rows) wr[u] = 0.f;
    }
    join_loads(raw, rz);
    if (sizeof(T) == 2) {
      float f[V];
#pragma unroll
      for (int v = 0; v < V; ++v) f[v] = 0.f;
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        float x[V];
        Vec<T>::unpack(raw[u], x);
#pragma unroll
        for (int v = 0; v < V; ++v) f[v] = fmaf(wr[u], x[v], f[v]);
      }
#pragma unroll
      for (int v = 0; v < V; ++v) S[v] += (double)f[v];
    } else {
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        float x[V];
        Vec<T>::unpack(raw[u], x);
#pragma unroll
        for (int v = 0; v < V; ++v) S[v] += (double)wr[u] * (double)x[v];
      }
    }
  }
#pragma unroll
  for (int v = 0; v < V; ++v) partial[(int64_t)chunk * cols + c0 + v] = S[v];
}

// One warp: dot product of a storage row with the vector wv (same symbol type, contiguous); valid in every lane.
template <typename T>
__device__ __forceinline__ double wdot_warp(const T* __restrict__ row, const T* __restrict__ wv, int64_t cols) {
  constexpr int V = Vec<T>::V;
  const int lane = threadIdx.x & 31;
  const int64_t nvec = cols / V;
  const uint32_t rz = (uint32_t)((uint64_t)cols >> 40);
  double S = 0.0;
  for (int64_t v0 = lane; v0 < nvec; v0 += 32 * 8) {
    uint4 rx[8], ry[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int64_t vi = v0 + 32 * u, vc = vi < nvec ? vi : nvec - 1;
      rx[u] = ld_cg16(row + vc * V);
      ry[u] = ld_cg16(wv + vc * V);
    }
    join_loads(rx, rz);
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      if (v0 + 32 * u >= nvec) continue;
      float x[V], y[V];
      Vec<T>::unpack(rx[u], x);
      Vec<T>::unpack(ry[u], y);
      if (sizeof(T) == 2) {
        float f = 0.f;
#pragma unroll
        for (int v = 0; v < V; ++v) f = fmaf(x[v], y[v], f);
        S += (double)f;
      } else {
#pragma unroll
        for (int v = 0; v < V; ++v) S += (double)x[v] * (double)y[v];
      }
    }
  }
  return warp_sum(S);
}

// Block 0, threads 0..GECC_MAX_FOUND-1: one located symbol per thread (loads in parallel, not one after the other).
__device__ __noinline__ void write_report_block0(const DecodeParams& p, int verdict, int n_found, int s0, int t0, const double* sh_max, const Thresholds& th) {
  gecc_report_t* r = p.report;
  if (threadIdx.x < GECC_MAX_FOUND) {
    gecc_found_t f = gecc_found_t{-1, -1, -1, 0, 0.0};
    if ((int)threadIdx.x < n_found) f = p.st->found[threadIdx.x];
    r->found[threadIdx.x] = f;
  }
  if (threadIdx.x == 0) {
    r->verdict = verdict;
    r->n_found = n_found;
    r->n_row_flags = s0;
    r->n_col_flags = t0;
    for (int q = 0; q < 4; ++q) { r->max_abs_syndrome[q] = sh_max[q]; r->tau[q] = th.tau[q]; }
  }
}

// ================= phase 5: c_true = c - e by block 0, and the report =================
// Whole-line faults are corrected along the whole line (reading R6), points only where located (reading R5).
__device__ __noinline__ void apply_plan_block0(const DecodeParams& p, int s0, int t0, const double* sh_max, const Thresholds& th) {
  DecodeState* st = p.st;
  const int n = p.n, m = p.m;
  double* syn = p.fb.syn;

    __syncthreads();
    const int verdict = __ldcg(&st->verdict);
    if (verdict == GECC_CORRECTED && __ldcg(&st->par_kind) >= 0) {  // a parity symbol of C_bar, not C: p_true = p - delta (first limb)
      if (threadIdx.x == 0) {
        const int line = __ldcg(&st->par_line), c = __ldcg(&st->par_c);
        float* sym = __ldcg(&st->par_kind) == GECC_KIND_PR ? p.P_r_w + (int64_t)line * GECC_PR_LD + 3 * c : p.P_c_w + (int64_t)(3 * c) * m + line;
        *sym = (float)((double)__ldcg(sym) - __ldcg(&st->par_delta));
      }
    } else if (verdict == GECC_CORRECTED) {
      const bool rows_short = __ldcg(&st->rows_short) != 0;
      const double* l1 = rows_short ? syn + 2 * (int64_t)n : syn;
      const double* l2 = rows_short ? syn + 2 * (int64_t)n + m : syn + n;
      const int n_long = rows_short ? m : n;
      const int nS = __ldcg(&st->nS);
      const int S0 = __ldcg(&st->S[0]), S1i = __ldcg(&st->S[1]);
      const int wl0 = __ldcg(&st->whole_line[0]), wl1 = __ldcg(&st->whole_line[1]);
      const double w1 = (double)(S0 + 1), w2 = (double)(S1i + 1);
      const int npts = __ldcg(&st->n_points);
      if (wl0 || wl1) {
        for (int64_t g = threadIdx.x; g < n_long; g += DT) {
          for (int idx = 0; idx < nS; ++idx) {
            if (!(idx == 0 ? wl0 : wl1)) continue;
            const int sl = idx == 0 ? S0 : S1i;
            double x;
            if (nS == 1) x = __ldcg(l1 + g);
            else if ((wl0 != 0) != (wl1 != 0)) {  // the other line holds located points only: the rest of the plain syndrome is this line's
              x = __ldcg(l1 + g);
              for (int a = 0; a < npts; ++a)
                if (__ldcg(&st->pt_l[a]) == g && __ldcg(&st->pt_s[a]) != sl) x -= __ldcg(&st->pt_x[a]);
            } else { const double y1 = __ldcg(l1 + g), x2 = (__ldcg(l2 + g) - w1 * y1) / (w2 - w1); x = idx == 0 ? y1 - x2 : x2; }
            const int64_t off = rows_short ? (int64_t)sl * p.ldc + g : g * p.ldc + sl;
            p.C[off] = (float)((double)__ldcg(p.C + off) - x);
          }
        }
      }
      if ((int)threadIdx.x < npts) {
        const int g = threadIdx.x;
        const int sl = __ldcg(&st->pt_s[g]), ll = __ldcg(&st->pt_l[g]);
        bool in_whole = (wl0 && S0 == sl) || (wl1 && nS > 1 && S1i == sl);  // already corrected along its line
        const int pi = rows_short ? sl : ll, pj = rows_short ? ll : sl;
        if (__ldcg(&st->repaired)) {  // a symbol of a recomputed line that was set aside: its recomputed value was kept
          const int nk = min(__ldcg(&st->n_keep), kMaxKeep);
          for (int q = 0; q < nk; ++q) {
            const int kr = __ldcg(&st->keep[q].is_row), kl = __ldcg(&st->keep[q].line), kt = __ldcg(&st->keep[q].t);
            if ((kr && kl == pi && kt == pj) || (!kr && kl == pj && kt == pi)) {
              p.C[(int64_t)pi * p.ldc + pj] = (float)__ldcg(&st->keep[q].v);
              in_whole = true;
              break;
            }
          }
        }
        if (!in_whole) {
          const int64_t off = (int64_t)pi * p.ldc + pj;
          p.C[off] = (float)((double)__ldcg(p.C + off) - __ldcg(&st->pt_x[g]));
        }
      }
      // A located symbol corrected by its syndrome inherits the syndrome's noise (sigma of a plain syndrome: tau / kappa,
      // the rounding of a whole line of C).  Where that exceeds the repair accuracy (large k; 3xTF32) and the operands are
      // at hand (level X), the located symbols are RECOMPUTED instead: c_ij = sum_l a_il b_lj in fp64 ("mark the
      // compromised data for recomputation").  The reported magnitude stays the syndrome's estimate.
      const double sigma_long = th.tau[rows_short ? 2 : 0] / kKappa;
      if (p.level >= 1 && p.A && p.B && th.sigma_c2 > 0.0 && sigma_long > kRepairAccuracy * sqrt(th.sigma_c2)) {
        __shared__ double red[DT / 32];
        const bool ta = p.trans_a != 0, tb = p.trans_b != 0;
        for (int g = 0; g < npts; ++g) {
          const int sl = __ldcg(&st->pt_s[g]), ll = __ldcg(&st->pt_l[g]);
          const int64_t pi = rows_short ? sl : ll, pj = rows_short ? ll : sl;
          double acc = 0.0;
          for (int64_t l = threadIdx.x; l < p.k; l += DT) {
            const int64_t ia = ta ? l * p.lda + pi : pi * p.lda + l, ib = tb ? pj * p.ldb + l : l * p.ldb + pj;
            const double a = p.dtype == GECC_BF16 ? (double)__bfloat162float(reinterpret_cast<const __nv_bfloat16*>(p.A)[ia]) : (double)reinterpret_cast<const float*>(p.A)[ia];
            const double b = p.dtype == GECC_BF16 ? (double)__bfloat162float(reinterpret_cast<const __nv_bfloat16*>(p.B)[ib]) : (double)reinterpret_cast<const float*>(p.B)[ib];
            acc += a * b;
          }
          acc = warp_sum(acc);
          __syncthreads();
          if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
          __syncthreads();
          if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int w = 0; w < DT / 32; ++w) tot += red[w];
            p.C[pi * p.ldc + pj] = (float)tot;
          }
        }
      }
    }
    write_report_block0(p, verdict, __ldcg(&st->n_found), s0, t0, sh_max, th);
  }

template <typename T>
__global__ void __launch_bounds__(DT, 2) decode_kernel(const __grid_constant__ DecodeParams p) {
  unsigned int bar_target = 0;
  __shared__ EncSmem<T> esm;
  __shared__ Scratch sc;
  __shared__ Thresholds th;
  __shared__ Faults flt;
  __shared__ int sh_s, sh_t, sh_go;
  __shared__ int sh_elc[2], sh_elbase[2];  // flagged lines this block met (rows, columns), their first slot in the state's lists
  __shared__ DecodeState::Early sh_el[2];
  __shared__ unsigned long long sh_bm[4];  // block maxima of |syndrome| (bit patterns of non-negative doubles)
  __shared__ double sh_max[4];
  __shared__ SmallLists sh_lists;          // the decision's lists of flagged lines while they are short (<= 8 per side)

  const int n = p.n, m = p.m, k = p.k;
  DecodeState* st = p.st;
  double* syn = p.fb.syn;
  double* tolx = syn + 2 * ((int64_t)n + m);  // extra tolerance per line, same order as syn
  const int64_t gthreads = (int64_t)gridDim.x * DT, gtid = (int64_t)blockIdx.x * DT + threadIdx.x;
  const int gwarps = gridDim.x * (DT / 32), gwarp = blockIdx.x * (DT / 32) + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;

  // Programmatic dependent launch: the product that precedes this kernel in the stream has completed from here on.  The next
  // kernel in the stream, if launched as a programmatic dependent (the encoder of the next product), may take its places as
  // this grid's blocks leave: it waits for this grid's completion before it reads anything.  (The trigger fires once every
  // block of this grid is resident, so the grid barrier below cannot be starved by the newcomers.)
  griddep_wait();
  griddep_launch_dependents();

  auto stamp = [&]() {  // block 0, thread 0: slot 0 holds the number of stamps that follow
    if (blockIdx.x == 0 && threadIdx.x == 0 && p.stamps[0] + 1 < (unsigned long long)kMaxPhaseStamps) {
      p.stamps[p.stamps[0] + 1] = globaltimer_ns();
      p.stamps[0] += 1;
    }
  };
#ifdef GECC_FINE_STAMPS
#define FSTAMP() stamp()
#else
#define FSTAMP() do { } while (0)
#endif
  // syn_status 1: the product itself folded its partial sums (syndromes, flags, counts, early lists, thresholds are in the
  // workspace) -- this kernel starts at the decision.  Written before this launch, cleared by the last block to leave.
  const bool ready = __ldcg(&st->syn_status) == 1;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    ws_enter(p.counters, "gecc_decode_correct");
    p.stamps[0] = 0;
  }
  stamp();
  if (threadIdx.x == 0) {
    if (ready) {
      for (int q = 0; q < 4; ++q) th.tau[q] = __ldcg(&st->tau[q]);
      th.sigma_a = __ldcg(&st->sigma_a); th.sigma_b = __ldcg(&st->sigma_b); th.sigma_c2 = __ldcg(&st->sigma_c2);
      th.single = p.single;
    } else make_thresholds(p.ts, n, k, m, th);
  }
  __syncthreads();
  DecideBufs dbufs;
  {
    dbufs.stamps = p.stamps;
    dbufs.rflag = p.fb.rflag;
    dbufs.qflag = p.fb.qflag;
    dbufs.votes = p.votes;
    uint8_t* q = p.lists;  // doubles first (8-byte aligned), then the index arrays
    auto take_d = [&](int64_t len) { double* r = reinterpret_cast<double*>(q); q += len * sizeof(double); return r; };
    dbufs.rows.a1 = take_d(n); dbufs.rows.a2 = take_d(n); dbufs.rows.t1 = take_d(n); dbufs.rows.t2 = take_d(n);
    dbufs.cols.a1 = take_d(m); dbufs.cols.a2 = take_d(m); dbufs.cols.t1 = take_d(m); dbufs.cols.t2 = take_d(m);
    dbufs.rows.idx = reinterpret_cast<int*>(q); q += (int64_t)n * sizeof(int);
    dbufs.cols.idx = reinterpret_cast<int*>(q);
    dbufs.rows.cnt = dbufs.cols.cnt = 0;
    dbufs.small = &sh_lists;
    dbufs.dtype = p.dtype; dbufs.single = p.single; dbufs.P_r = p.fb.P_r; dbufs.P_c = p.fb.P_c; dbufs.P_g = p.P_g;
  }

  // A flagged line is noted in shared memory (the first 8 per side and block); once the block knows how many it has, it
  // reserves that many slots in the grid-wide count and copies those that fall among the first 8 into the decoder state.
  auto note_flagged = [&](int side, int idx, double a, double b, double t1, double t2) {
    const int ls = atomicAdd(&sh_elc[side], 1);
    if (ls < 8) { sh_el[side].idx[ls] = idx; sh_el[side].a1[ls] = a; sh_el[side].a2[ls] = b; sh_el[side].t1[ls] = t1; sh_el[side].t2[ls] = t2; }
  };
  auto publish_flagged = [&](unsigned int* ctr_s, unsigned int* ctr_t) {  // sh_elc holds the block's flagged rows / columns
    __syncthreads();
    if (threadIdx.x == 0) {
      sh_elbase[0] = sh_elc[0] ? (int)atomicAdd(ctr_s, (unsigned int)sh_elc[0]) : 0;
      sh_elbase[1] = sh_elc[1] ? (int)atomicAdd(ctr_t, (unsigned int)sh_elc[1]) : 0;
    }
    __syncthreads();
    if (threadIdx.x < 16) {
      const int side = threadIdx.x >> 3, e = threadIdx.x & 7, slot = sh_elbase[side] + e;
      if (e < min(sh_elc[side], 8) && slot < 8) {
        DecodeState::Early& E = st->el[side];
        E.idx[slot] = sh_el[side].idx[e]; E.a1[slot] = sh_el[side].a1[e]; E.a2[slot] = sh_el[side].a2[e];
        E.t1[slot] = sh_el[side].t1[e]; E.t2[slot] = sh_el[side].t2[e];
      }
    }
    __threadfence();
  };
  if (threadIdx.x < 2) sh_elc[threadIdx.x] = 0;
  if (threadIdx.x < 4) sh_bm[threadIdx.x] = 0ull;
  __syncthreads();

  // ================= phase 1: syndromes and flags (only when the product did not fold them itself) =================
  // Four threads per line; sum minus parity, see fold.cuh.
  if (!ready) {
    const int64_t lines = (int64_t)n + m;
    double mx[4] = {0.0, 0.0, 0.0, 0.0};
    for (int64_t q0 = gtid >> 2; q0 < ((lines + 63) & ~63ll); q0 += gthreads >> 2) {  // whole quads stay together
      const int qd = threadIdx.x & 3;
      const bool is_row = q0 < n, live = q0 < lines;
      const int64_t idx = is_row ? q0 : q0 - n;
      const FoldResult r = fold_line<4>(p.fb, th, is_row, live ? idx : 0, live, qd);
      if (live && qd == 0) {
        if (r.flagged) note_flagged(is_row ? 0 : 1, (int)idx, r.a, r.b, r.t1, r.t2);
        const int o = is_row ? 0 : 2;
        mx[o] = fmax(mx[o], abs_for_max(r.a)); mx[o + 1] = fmax(mx[o + 1], abs_for_max(r.b));
      }
    }
    // block maxima: warp shuffles, then one shared-memory atomic per warp and value (order-independent)
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      unsigned long long v = (unsigned long long)__double_as_longlong(mx[q]);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) { const unsigned long long w2 = __shfl_xor_sync(0xffffffffu, v, o); v = w2 > v ? w2 : v; }
      if (lane == 0 && v) atomicMax(&sh_bm[q], v);
    }
    publish_flagged(p.counters + kCtrDecS, p.counters + kCtrDecT);
    if (threadIdx.x < 4 && sh_bm[threadIdx.x]) atomicMax(reinterpret_cast<unsigned long long*>(p.counters + kCtrDecMax) + threadIdx.x, sh_bm[threadIdx.x]);
    grid_barrier(p.counters + kCtrDecBar, bar_target); stamp();
  }

  if (threadIdx.x == 0) {
    if (ready) {
      sh_s = __ldcg(&st->n_row_flags0);
      sh_t = __ldcg(&st->n_col_flags0);
#pragma unroll
      for (int q = 0; q < 4; ++q) sh_max[q] = __ldcg(&st->maxabs[q]);
    } else {
      sh_s = (int)__ldcg(p.counters + kCtrDecS);
      sh_t = (int)__ldcg(p.counters + kCtrDecT);
      const unsigned long long* gmax = reinterpret_cast<const unsigned long long*>(p.counters + kCtrDecMax);
#pragma unroll
      for (int q = 0; q < 4; ++q) sh_max[q] = __longlong_as_double((long long)__ldcg(gmax + q));
    }
  }
  __syncthreads();
  const int s0 = sh_s, t0 = sh_t;

  auto write_report = [&](int verdict, int n_found) { write_report_block0(p, verdict, n_found, s0, t0, sh_max, th); };

  // Every block passes here on its way out, after its last barrier and its last read of the shared words: the last one to
  // leave clears them for the next launch.
  auto leave = [&]() {
    if (threadIdx.x == 0) {
      __threadfence();
      if (atomicAdd(p.counters + kCtrDecExit, 1u) == gridDim.x - 1) {
        p.counters[kCtrDecBar] = 0; p.counters[kCtrDecS] = 0; p.counters[kCtrDecT] = 0; p.counters[kCtrDecWork] = 0;
        p.counters[kCtrDecS2] = 0; p.counters[kCtrDecT2] = 0; p.counters[kCtrDecGo] = 0;
        unsigned long long* gmax = reinterpret_cast<unsigned long long*>(p.counters + kCtrDecMax);
        for (int q = 0; q < 4; ++q) gmax[q] = 0;
        st->syn_status = 0;
        // scratch of the verification and the repair (no barrier separates a launch's start from their first use)
        st->cnt_a = 0; st->cnt_b = 0; st->n_keep = 0;
        for (int s2 = 0; s2 < 2 * kMaxInputFaults; ++s2) { st->acc[s2][0] = 0.0; st->acc[s2][1] = 0.0; st->accad[s2] = 0.0; }
        p.counters[kCtrDecExit] = 0;
        __threadfence();
        atomicExch(p.counters + kCtrBusy, 0u);  // the workspace is free again
      }
    }
  };

  if (s0 == 0 && t0 == 0) {  // nothing flagged: CLEAN (PAPER.md:215-219 with both sets empty)
    if (blockIdx.x == 0) {
      if (threadIdx.x == 0) { st->verdict = GECC_CLEAN; st->n_found = 0; }
      write_report(GECC_CLEAN, 0);
    }
    leave();
    return;
  }

  const T* A = reinterpret_cast<const T*>(p.A);
  const T* B = reinterpret_cast<const T*>(p.B);
  const bool ta = p.trans_a != 0, tb = p.trans_b != 0;
  // symbol (i, l) of A / (l, j) of B in the operand's storage
  auto ia = [&](int64_t i, int64_t l) -> int64_t { return ta ? l * p.lda + i : i * p.lda + l; };
  auto ib = [&](int64_t l, int64_t j) -> int64_t { return tb ? j * p.ldb + l : l * p.ldb + j; };

  auto apply_plan_and_report = [&]() { apply_plan_block0(p, s0, t0, sh_max, th); };

  // ================= phase 2: decision without verification (few flagged lines, or level 0) =================
  // Block 0 decides alone; the other blocks only learn whether the operands have to be verified (Level X with a
  // whole-line fault or a refusal) -- if not, block 0 patches C, writes the report, and everyone leaves.
  const bool spec = p.level >= 1 && (s0 > 8 || t0 > 8) && gridDim.x > 1;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    for (int q = 0; q < 4; ++q) st->tau[q] = th.tau[q];
    st->sigma_a = th.sigma_a; st->sigma_b = th.sigma_b; st->sigma_c2 = th.sigma_c2;
  }
  __syncthreads();
  bool have_plan = false;
  if (!spec) {
    int need_verify;
    if (blockIdx.x == 0) {
      FSTAMP();
      if (threadIdx.x == 0) sh_go = decide_small(st, 0, s0, t0, p.single) ? 1 : 0;
      __syncthreads();
      if (!sh_go) decide(st, syn, tolx, dbufs, n, m, p.level, 0, s0, t0, sc);
      __syncthreads();
      FSTAMP();
      need_verify = __ldcg(&st->need_verify);
      if (!need_verify) apply_plan_and_report();
      FSTAMP();
      __syncthreads();
      if (threadIdx.x == 0) {
        __threadfence();
        atomicExch(p.counters + kCtrDecGo, 1u + (unsigned int)need_verify);
      }
    } else {
      if (threadIdx.x == 0) {
        unsigned int go;
        for (;;) {
          asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(go) : "l"(p.counters + kCtrDecGo) : "memory");
          if (go) break;
          __nanosleep(200);
        }
        __threadfence();
        sh_go = (int)go;
      }
      __syncthreads();
      need_verify = sh_go - 1;
    }
    stamp();
    if (!need_verify) { leave(); return; }
    have_plan = true;
  }

  // ================= phase 3: input verification (Level X) =================
  // The encoder's reductions over A and B; unchanged lines reproduce the stored checks bit for bit, so any difference marks
  // a faulty line.  With many flagged lines (what an input fault looks like) this comes BEFORE any decision: the Level-P
  // plan is only needed, and only then computed, if the operands turn out intact.
  auto candidate = [&](bool of_a, int line, double d1, double d2) {
    if (!(d1 == 0.0) || !(d2 == 0.0)) {
      const int slot = atomicAdd(of_a ? &st->cnt_a : &st->cnt_b, 1);
      if (slot < kMaxInputFaults) {
        DecodeState::Cand& c = of_a ? st->ca[slot] : st->cb[slot];
        c.l = line; c.d1 = d1; c.d2 = d2;
      }
    }
  };
  {
    constexpr int V = Vec<T>::V;
    // Both checks of both operands run along k.  An operand whose storage has k as its column index (A, or B^T stored
    // m x k) is reduced over its storage rows, exactly as encode_colsum_kernel did; one whose rows are the lines l (B, or
    // A^T stored k x n) is summed along each storage row, as encode_rowsum_kernel did.
    const int strips = (k + 32 * V - 1) / (32 * V);
    const int rows_a = n, rows_b = m;
    const int chunks_a = ta ? 0 : (rows_a + p.enc_chunk_rows - 1) / p.enc_chunk_rows;
    const int chunks_b = tb ? (rows_b + p.enc_chunk_rows_b - 1) / p.enc_chunk_rows_b : 0;
    const int items_a = strips * chunks_a, items_b = strips * chunks_b;
    for (int item0 = (int)blockIdx.x; item0 < items_a + items_b; item0 += (int)gridDim.x) {
      const bool of_a = item0 < items_a;
      const int item = of_a ? item0 : item0 - items_a;
      const int strip = item % strips, chunk = item / strips;
      const T* X = of_a ? A : B;
      const int rows = of_a ? rows_a : rows_b, chunks = of_a ? chunks_a : chunks_b, chunk_rows = of_a ? p.enc_chunk_rows : p.enc_chunk_rows_b;
      double* part = of_a ? p.encpart : p.encpart_b;
      const double* par = of_a ? p.A_par64 : p.B_par64;
      colsum_item<T>(X, rows, k, of_a ? p.lda : p.ldb, nullptr, part, strip, chunk, chunk_rows, esm);
      // the last chunk of a strip to finish folds the strip's columns (the encoder's own arrival counters, idle now; the
      // strips of B^T count on the slots after those of A)
      if (arrive_last(p.counters + kCtrEncStrip + (of_a ? 0 : strips) + strip, chunks, esm.last)) {
        const int t = threadIdx.x;
        const int64_t c = (int64_t)strip * 32 * V + t;
        if (t < 32 * V && c < k) {
          double s1, s2;
          colsum_combine(part, chunks, chunk_rows, k, c, s1, s2);
          candidate(of_a, (int)c, s1 - par[c], s2 - par[k + c]);
        }
      }
    }
    // storage rows are handed out four at a time from a counter, so blocks that had fewer items above take more here:
    // first the k rows of A^T (if A is stored transposed), then the k rows of B (if it is not)
    const int nrow_a = ta ? k : 0, nrow_b = tb ? 0 : k;
    for (;;) {
      int r0 = 0;
      if (lane == 0) r0 = (int)atomicAdd(p.counters + kCtrDecWork, 4u);
      r0 = __shfl_sync(0xffffffffu, r0, 0);
      if (r0 >= nrow_a + nrow_b) break;
      for (int rr = r0; rr < r0 + 4 && rr < nrow_a + nrow_b; ++rr) {
        const bool of_a = rr < nrow_a;
        const int64_t r = of_a ? rr : rr - nrow_a;
        double S1, S2;
        float q = 0.f;
        if (of_a) rowsum_warp<T>(A + r * p.lda, n, nullptr, S1, S2, q);
        else rowsum_warp<T>(B + r * p.ldb, m, nullptr, S1, S2, q);
        const double* par = of_a ? p.A_par64 : p.B_par64;
        if (lane == 0) candidate(of_a, (int)r, S1 - par[r], S2 - par[k + r]);
      }
    }
    __threadfence();
  }
  grid_barrier(p.counters + kCtrDecBar, bar_target); stamp();
  // every block evaluates the (at most 2 x kMaxInputFaults) candidate lines itself: no barrier before the repair
  if (threadIdx.x == 0) verify_compare(st, p.dtype, n, m, th.sigma_a, th.sigma_b, flt);
  __syncthreads();
  FSTAMP();

  if (!flt.ok || !flt.repaired) {
    // a line of A or B with more than one bad symbol: UNCORRECTABLE_INPUT, nothing is patched; or the operands are intact
    // (a transient fault in the product's read of them): the Level-P result stands
    if (blockIdx.x == 0) {
      if (flt.ok && !have_plan) decide(st, syn, tolx, dbufs, n, m, p.level, 0, s0, t0, sc);
      __syncthreads();
      if (threadIdx.x == 0) {
        if (!flt.ok && !have_plan) { st->n_row_flags0 = s0; st->n_col_flags0 = t0; st->rows_short = 1; }
        publish_faults(st, flt);
      }
      apply_plan_and_report();
    }
    stamp();
    leave();
    return;
  }

  // ================= phase 4: repair =================
  // (A + E_A)(B + E_B) = A B + E_A (B + E_B) + A E_B: row i of C carries e b~_l* for an A fault (i, l, e) (b~: the faulty
  // B), column j carries e' a_*l' for a B fault (l', j, e') (a: the clean A).  Every line that carried a footprint is
  // settled symbol by symbol, in one of two ways (the same for the whole repair, from the faults' magnitudes):
  //   subtract   the exact footprint is subtracted from what the symbol holds.  What stays behind is the rounding the
  //              tensor cores did at the footprint's magnitude, about (k / 16) 2^-24 |d| (one truncation per MMA step); taken
  //              when that is below kRepairAccuracy x RMS(C).  Reads one line of the other operand per fault.
  //   recompute  ("mark the compromised data for recomputation") the line is recomputed from the patched
  //              operands; each recomputed symbol is compared with (what it held - the footprint): if rounding explains
  //              the difference the exact value is written, else the footprint alone is removed and the symbol is left
  //              for the second decision (a point error in this very line; its exact value is kept for the final patch).
  // The syndromes follow every change and the settled lines' own syndromes are taken from scratch (sum of the line minus
  // its exact parity), so the second decision sees no residue of a footprint and keeps the plain thresholds.
  T* Aw = reinterpret_cast<T*>(p.A);
  T* Bw = reinterpret_cast<T*>(p.B);
  const int nfa = flt.nfa, nfb = flt.nfb;
  double* q1 = syn + 2 * (int64_t)n; double* q2 = q1 + m;
  double* r1 = syn; double* r2 = syn + n;
  const double G = p.G;
  bool recompute = false;
  const double rho = (double)k / 16.0 * (p.dtype == GECC_F32 ? 3.0 : 1.0) * 5.9604644775390625e-08;  // truncation per unit of footprint
  {
    const double steps16 = rho, u24 = 1.0;
    const double budget = kRepairAccuracy * sqrt(th.sigma_c2);
    for (int a = 0; a < nfa; ++a) recompute |= !(steps16 * u24 * fabs(flt.fa[a].e) * 4.0 * th.sigma_b <= budget);
    for (int b = 0; b < nfb; ++b) recompute |= !(steps16 * u24 * fabs(flt.fb[b].e) * 4.0 * th.sigma_a <= budget);
    for (int a = 0; a < nfa; ++a)  // an A and a B fault sharing l: the symbol where their lines cross carried e e'
      for (int b = 0; b < nfb; ++b)
        if (flt.fa[a].col == flt.fb[b].row) recompute |= !(steps16 * u24 * fabs(flt.fa[a].e * flt.fb[b].e) <= budget);
    if (!(th.sigma_c2 > 0.0)) recompute = true;  // caller's thresholds without sums of squares: no scale known
  }
  // the lines to settle: rows of C that carried an A fault's footprint, then columns that carried a B fault's
  int nsteps = 0, step_kind[2 * kMaxInputFaults], step_line[2 * kMaxInputFaults];
  for (int a = 0; a < nfa; ++a) {
    bool done = false;
    for (int a2 = 0; a2 < a; ++a2) done |= flt.fa[a2].row == flt.fa[a].row;
    if (!done) { step_kind[nsteps] = 0; step_line[nsteps++] = flt.fa[a].row; }
  }
  for (int b = 0; b < nfb; ++b) {
    bool done = false;
    for (int b2 = 0; b2 < b; ++b2) done |= flt.fb[b2].col == flt.fb[b].col;
    if (!done) { step_kind[nsteps] = 1; step_line[nsteps++] = flt.fb[b].col; }
  }
  // One line settled by subtraction, few flagged lines on its own side: the lines of the other side are flagged again by
  // the threads that settle their symbols and the line's own side keeps its flags (only the settled line is judged again),
  // so the separate pass over all lines and its barrier are not needed.
  const bool fast = !recompute && nsteps == 1 && (step_kind[0] == 0 ? s0 : t0) <= 8;
  // The operands are patched (a_true = a - e) by block 0: before the lines are recomputed from them, or, when footprints
  // are only subtracted, at the very end -- until then every block reads them as the product saw them.
  auto patch_operands = [&]() {
    if (threadIdx.x == 0) {
      for (int a = 0; a < nfa; ++a) patch_sym<T>(Aw, p.A_lo, ia(flt.fa[a].row, flt.fa[a].col), flt.fa[a].e);
      for (int b = 0; b < nfb; ++b) patch_sym<T>(Bw, p.B_lo, ib(flt.fb[b].row, flt.fb[b].col), flt.fb[b].e);
      __threadfence();
    }
  };
  const bool patched = recompute;  // operands already clean while the lines are settled
  // symbol (i, l) of A / (l, j) of B as the product saw it (faulty) and as it should be (clean), whatever memory holds now
  auto a_clean = [&](int64_t i, int64_t l) -> double {
    double v = (double)load_sym<T>(Aw + ia(i, l));
    if (!patched) for (int a = 0; a < nfa; ++a) if (flt.fa[a].row == i && flt.fa[a].col == l) v -= flt.fa[a].e;
    return v;
  };
  auto b_seen = [&](int64_t l, int64_t j) -> double {
    double v = (double)load_sym<T>(Bw + ib(l, j));
    if (patched) for (int b = 0; b < nfb; ++b) if (flt.fb[b].row == l && flt.fb[b].col == j) v += flt.fb[b].e;
    return v;
  };
  if (recompute) {
    if (blockIdx.x == 0) patch_operands();
    grid_barrier(p.counters + kCtrDecBar, bar_target); stamp();  // the operands are patched
  }
  {
    constexpr int V = Vec<T>::V;
    T* wv = reinterpret_cast<T*>(p.recomp);
    const double sym_floor = 2.0 * fmax(th.tau[0] / sqrt((double)m), th.tau[2] / sqrt((double)n));
    FSTAMP();
    if (fast) {
      __syncthreads();
      if (threadIdx.x < 2) sh_elc[threadIdx.x] = 0;
      __syncthreads();
    }
    for (int sidx = 0; sidx < nsteps; ++sidx) {
      if (sidx > 0) { __threadfence(); grid_barrier(p.counters + kCtrDecBar, bar_target); stamp(); }  // the previous line is settled (p.recomp is reused)
      const int line = step_line[sidx];
      const bool is_row = step_kind[sidx] == 0;          // row `line` of C from A[line, :] and B; else column from A and B[:, line]
      const T* X = is_row ? Bw : Aw;                       // the operand that is read in full
      const int64_t ldx = is_row ? p.ldb : p.lda;
      const bool x_l_rows = is_row ? !tb : ta;            // storage of X: k rows (l) x len columns
      const int len = is_row ? m : n;                      // symbols of the line
      const T* w = is_row ? Aw + ia(line, 0) : Bw + ib(0, line);
      const int64_t wstride = is_row ? (ta ? p.lda : 1) : (tb ? 1 : p.ldb);
      const int64_t cstride = is_row ? 1 : p.ldc;
      float* cline = is_row ? p.C + (int64_t)line * p.ldc : p.C + line;
      // this thread's share of the line's own sums: of what the line holds now (recompute: its syndromes are taken from
      // scratch against the exact parity) or of the changes made to it (subtract: the syndromes are updated), and of |footprint|
      double S1 = 0.0, S2 = 0.0, SA = 0.0;
      auto settle = [&](int t, double v) {
        float* cp = cline + t * cstride;
        const double old = (double)__ldcg(cp);
        // the footprints this symbol still carries (D) and their magnitudes (ad)
        double D = 0.0, ad = 0.0;
        if (is_row) {
          for (int a = 0; a < nfa; ++a) {
            if (flt.fa[a].row != line) continue;
            const double term = flt.fa[a].e * b_seen(flt.fa[a].col, t);  // b~: B as the product saw it
            D += term; ad += fabs(term);
          }
          for (int b = 0; b < nfb; ++b) {
            if (flt.fb[b].col != t) continue;
            const double term = flt.fb[b].e * a_clean(line, flt.fb[b].row);
            D += term; ad += fabs(term);
          }
        } else {
          bool row_done = false;  // a symbol of a row that was settled in an earlier step carries nothing any more
          for (int s2 = 0; s2 < sidx; ++s2) row_done |= step_kind[s2] == 0 && step_line[s2] == t;
          if (!row_done)
            for (int b = 0; b < nfb; ++b) {
              if (flt.fb[b].col != line) continue;
              const double term = flt.fb[b].e * a_clean(t, flt.fb[b].row);
              D += term; ad += fabs(term);
            }
        }
        float cnew;
        if (!recompute) cnew = (float)(old - D);
        else if (fabs((double)(float)v + D - old) <= G * ad + sym_floor) cnew = (float)v;  // rounding explains the difference: take the exact value
        else {
          cnew = (float)(old - D);  // something else sits here: remove the footprints only, keep the exact value for later
          const int slot = atomicAdd(&st->n_keep, 1);
          if (slot < kMaxKeep) { st->keep[slot].is_row = is_row ? 1 : 0; st->keep[slot].line = line; st->keep[slot].t = t; st->keep[slot].v = v; }
        }
        *cp = cnew;
        const double cfin = (double)cnew, delta = cfin - old, wl = (double)(line + 1);
        if (fast) {  // the crossing line's syndromes follow the change and its flag is taken again at once
          const int64_t o1 = is_row ? 2 * (int64_t)n + t : t, o2 = is_row ? 2 * (int64_t)n + m + t : (int64_t)n + t;
          const double a2 = __ldcg(syn + o1) + delta, b2 = __ldcg(syn + o2) + wl * delta;
          const double t1 = th.tau[is_row ? 2 : 0] + __ldcg(tolx + o1), t2 = th.tau[is_row ? 3 : 1] + __ldcg(tolx + o2);
          syn[o1] = a2; syn[o2] = b2;
          const bool fl = !(fabs(a2) <= t1) || !(fabs(b2) <= t2);
          (is_row ? dbufs.qflag : dbufs.rflag)[t] = fl;
          if (fl) note_flagged(is_row ? 1 : 0, t, a2, b2, t1, t2);
        } else if (is_row) { q1[t] = __ldcg(q1 + t) + delta; q2[t] = __ldcg(q2 + t) + wl * delta; }
        else {
          int own = -1;  // row t was itself settled: its sums are kept in the step's accumulators
          for (int s2 = 0; s2 < sidx; ++s2)
            if (step_kind[s2] == 0 && step_line[s2] == t) own = s2;
          if (own >= 0) { atomicAdd(&st->acc[own][0], delta); atomicAdd(&st->acc[own][1], wl * delta); }
          else { r1[t] = __ldcg(r1 + t) + delta; r2[t] = __ldcg(r2 + t) + wl * delta; }
        }
        S1 += recompute ? cfin : delta;
        S2 += (double)(t + 1) * (recompute ? cfin : delta);
        SA += ad;
      };
      if (!recompute) {
        for (int64_t t = gtid; t < len; t += gthreads) settle((int)t, 0.0);
        FSTAMP();
      } else if (x_l_rows) {
        // line = sum_l w[l] X[l][.]: the reduction over storage rows with weights (partials per kRecompRows rows, then summed)
        const int strips = (len + 32 * V - 1) / (32 * V), chunks = (k + kRecompRows - 1) / kRecompRows;
        for (int item = gwarp; item < strips * chunks; item += gwarps)
          wcolsum_warp_item<T>(X, k, len, ldx, w, wstride, p.recomp, item % strips, item / strips);
        __threadfence();
        grid_barrier(p.counters + kCtrDecBar, bar_target); stamp();
        // 32 consecutive symbols per block and turn: warp q sums its eighth of the chunk partials, warp 0 settles
        double (*red)[32] = reinterpret_cast<double (*)[32]>(&esm.part[0][0][0][0]);
        const int per = (chunks + 7) / 8, wq = threadIdx.x >> 5;
        for (int grp = blockIdx.x; grp * 32 < len; grp += gridDim.x) {
          const int t = grp * 32 + lane;
          double ssum = 0.0;
          if (t < len) {
            const int ch_end = min(chunks, (wq + 1) * per);
            for (int ch = wq * per; ch < ch_end; ch += 8) {
              double v8[8];
#pragma unroll
              for (int u = 0; u < 8; ++u) v8[u] = ch + u < ch_end ? __ldcg(p.recomp + (int64_t)(ch + u) * len + t) : 0.0;
#pragma unroll
              for (int u = 0; u < 8; ++u) ssum += v8[u];
            }
          }
          red[wq][lane] = ssum;
          __syncthreads();
          if (wq == 0 && t < len) {
            double tot = 0.0;
#pragma unroll
            for (int q = 0; q < DT / 32; ++q) tot += red[q][lane];
            settle(t, tot);
          }
          __syncthreads();
        }
      } else {
        // line[t] = w . X[t][:] (l runs along the storage rows of X): w is first gathered into a contiguous vector
        for (int64_t l2 = gtid; l2 < k; l2 += gthreads) wv[l2] = w[l2 * wstride];
        __threadfence();
        grid_barrier(p.counters + kCtrDecBar, bar_target); stamp();
        for (int64_t t = gwarp; t < len; t += gwarps) {
          const double sdot = wdot_warp<T>(X + t * ldx, wv, k);
          if (lane == 0) settle((int)t, sdot);
        }
      }
      // The line's own parity.  recompute: exact, row i: A[i, :] . B_P; column j: A_P . B[:, j],
      // by the last block.  subtract: the parity symbol the product computed carries the fault's shift e B_P[l] (row) /
      // e' A_P[l'] (column): par = minus that shift, so that (old syndrome + changes - par) is the updated syndrome.
      double p0 = 0.0, p1 = 0.0;
      if (blockIdx.x == gridDim.x - 1) {
        const double* par = is_row ? p.B_par64 : p.A_par64;
        if (recompute) {
          for (int l0 = threadIdx.x; l0 < k; l0 += 4 * DT) {
            double wl[4], a0[4], a1[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
              const int l = min(l0 + u * DT, k - 1);
              wl[u] = l0 + u * DT < k ? (double)load_sym<T>(w + l * wstride) : 0.0;
              a0[u] = par[l]; a1[u] = par[k + l];
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) { p0 += wl[u] * a0[u]; p1 += wl[u] * a1[u]; }
          }
        } else if (threadIdx.x == 0) {
          if (is_row) { for (int a = 0; a < nfa; ++a) if (flt.fa[a].row == line) { p0 -= flt.fa[a].e * par[flt.fa[a].col]; p1 -= flt.fa[a].e * par[k + flt.fa[a].col]; } }
          else { for (int b = 0; b < nfb; ++b) if (flt.fb[b].col == line) { p0 -= flt.fb[b].e * par[flt.fb[b].row]; p1 -= flt.fb[b].e * par[k + flt.fb[b].row]; } }
        }
      }
      {
        double v4[4] = {S1, S2, p0, p1};
        block_sum4(v4, sc);
        if (threadIdx.x == 0) {
          if (v4[0] != 0.0 || v4[1] != 0.0) { atomicAdd(&st->acc[sidx][0], v4[0]); atomicAdd(&st->acc[sidx][1], v4[1]); }
          if (blockIdx.x == gridDim.x - 1) { st->par[sidx][0] = v4[2]; st->par[sidx][1] = v4[3]; }
        }
        const double saw = warp_sum(SA);
        if (lane == 0 && saw != 0.0) atomicAdd(&st->accad[sidx], saw);
      }
      FSTAMP();
    }
    if (fast) publish_flagged(p.counters + kCtrDecS2, p.counters + kCtrDecT2);
    __threadfence();
    grid_barrier(p.counters + kCtrDecBar, bar_target); stamp();
    if (fast) {
      if (blockIdx.x == 0) {
        const bool is_row = step_kind[0] == 0;
        const int idx = step_line[0], side = is_row ? 0 : 1;
        if (threadIdx.x == 0) {
          // the settled line's own syndromes, updated (see the pass over all lines below for the allowance)
          const int64_t o1 = is_row ? idx : 2 * (int64_t)n + idx, o2 = is_row ? (int64_t)n + idx : 2 * (int64_t)n + m + idx;
          const double a = __ldcg(syn + o1) + __ldcg(&st->acc[0][0]) - __ldcg(&st->par[0][0]);
          const double b = __ldcg(syn + o2) + __ldcg(&st->acc[0][1]) - __ldcg(&st->par[0][1]);
          const double len = is_row ? (double)m : (double)n;
          const double adn = 2.0 * __ldcg(&st->accad[0]) / sqrt(len);
          const double x1 = __ldcg(tolx + o1) + rho * (fabs(__ldcg(&st->par[0][0])) + adn);
          const double x2 = __ldcg(tolx + o2) + rho * (fabs(__ldcg(&st->par[0][1])) + sqrt((len + 1.0) * (2.0 * len + 1.0) / 6.0) * adn);
          syn[o1] = a; syn[o2] = b; tolx[o1] = x1; tolx[o2] = x2;
          const double t1 = th.tau[is_row ? 0 : 2] + x1, t2 = th.tau[is_row ? 1 : 3] + x2;
          const bool fl = !(fabs(a) <= t1) || !(fabs(b) <= t2);
          (is_row ? dbufs.rflag : dbufs.qflag)[idx] = fl;
          // its side's list of flagged lines (from the first pass, still valid for every other line): the settled line is
          // taken out, or put in / brought up to date
          DecodeState::Early& E = st->el[side];
          int cnt = is_row ? s0 : t0, at = -1;
          for (int e = 0; e < cnt; ++e) if (E.idx[e] == idx) at = e;
          if (at >= 0 && !fl) { --cnt; E.idx[at] = E.idx[cnt]; E.a1[at] = E.a1[cnt]; E.a2[at] = E.a2[cnt]; E.t1[at] = E.t1[cnt]; E.t2[at] = E.t2[cnt]; }
          else if (fl) {
            if (at < 0) at = cnt++;
            if (at < 8) { E.idx[at] = idx; E.a1[at] = a; E.a2[at] = b; E.t1[at] = t1; E.t2[at] = t2; }
          }
          sh_go = cnt;
          publish_faults(st, flt);
          const int other0 = (int)__ldcg(p.counters + (is_row ? kCtrDecT2 : kCtrDecS2));
          if (cnt == 0 && other0 == 0) {
            // nothing is flagged any more: the input faults were all there was.  Verdict and report entries at once.
            int nf = 0;
            gecc_found_t* f = st->found;
            for (int a2 = 0; a2 < nfa && nf < GECC_MAX_FOUND; ++a2) f[nf++] = gecc_found_t{GECC_KIND_A, flt.fa[a2].row, flt.fa[a2].col, 0, flt.fa[a2].e};
            for (int b2 = 0; b2 < nfb && nf < GECC_MAX_FOUND; ++b2) f[nf++] = gecc_found_t{GECC_KIND_B, flt.fb[b2].row, flt.fb[b2].col, 0, flt.fb[b2].e};
            sort_found(f, nf);
            st->verdict = GECC_CORRECTED; st->rows_short = 1; st->n_found = nf; st->par_kind = -1;
            st->nS = 0; st->n_points = 0; st->whole_line[0] = st->whole_line[1] = 0;
            sh_go = -1 - nf;
          } else if (decide_small(st, 1, is_row ? cnt : other0, is_row ? other0 : cnt, p.single)) sh_go = -100;
        }
        __syncthreads();
        FSTAMP();
        if (sh_go <= -1 && sh_go > -100) {  // all clear
          patch_operands();
          write_report(GECC_CORRECTED, -1 - sh_go);
        } else {
          if (sh_go != -100) {
            const int own_side = sh_go, other = (int)__ldcg(p.counters + (is_row ? kCtrDecT2 : kCtrDecS2));
            decide(st, syn, tolx, dbufs, n, m, p.level, 1, is_row ? own_side : other, is_row ? other : own_side, sc);
          }
          FSTAMP();
          if (__ldcg(&st->verdict) == GECC_CORRECTED) patch_operands();
          FSTAMP();
          apply_plan_and_report();
        }
      }
      stamp();
      leave();
      return;
    }
    // Every line is flagged again, by the whole grid.  The settled lines' own syndromes are taken from scratch: the sum of
    // what the line now holds minus its exact parity, with the plain thresholds.
    {
      __syncthreads();
      if (threadIdx.x < 2) sh_elc[threadIdx.x] = 0;
      __syncthreads();
      for (int64_t ln = gtid; ln < (int64_t)n + m; ln += gthreads) {
        const bool is_row = ln < n;
        const int idx = (int)(is_row ? ln : ln - n);
        const int64_t o1 = is_row ? idx : 2 * (int64_t)n + idx, o2 = is_row ? (int64_t)n + idx : 2 * (int64_t)n + m + idx;
        int own = -1;
        for (int s2 = 0; s2 < nsteps; ++s2)
          if ((step_kind[s2] == 0) == is_row && step_line[s2] == idx) own = s2;
        double a, b, x1, x2;
        if (own >= 0) {
          a = __ldcg(&st->acc[own][0]) - __ldcg(&st->par[own][0]);
          b = __ldcg(&st->acc[own][1]) - __ldcg(&st->par[own][1]);
          if (recompute) {  // recomputed symbols are exact and so is the parity they are compared with: plain thresholds
            x1 = 0.0; x2 = 0.0;
          } else {
            // updated, not recomputed: what the line held (symbols and parity symbol alike) was rounded by the tensor cores
            // at the footprint's magnitude.  The line keeps the energy-scaled tolerance it had and gets an allowance for
            // that rounding: rho per unit of the parity symbol's shift and of the footprints (these add in quadrature).
            a += __ldcg(syn + o1); b += __ldcg(syn + o2);
            const double len = is_row ? (double)m : (double)n;
            const double adn = 2.0 * __ldcg(&st->accad[own]) / sqrt(len);
            x1 = __ldcg(tolx + o1) + rho * (fabs(__ldcg(&st->par[own][0])) + adn);
            x2 = __ldcg(tolx + o2) + rho * (fabs(__ldcg(&st->par[own][1])) + sqrt((len + 1.0) * (2.0 * len + 1.0) / 6.0) * adn);
          }
          syn[o1] = a; syn[o2] = b; tolx[o1] = x1; tolx[o2] = x2;
        } else {
          a = __ldcg(syn + o1); b = __ldcg(syn + o2); x1 = __ldcg(tolx + o1); x2 = __ldcg(tolx + o2);
        }
        const double t1 = th.tau[is_row ? 0 : 2] + x1, t2 = th.tau[is_row ? 1 : 3] + x2;
        const bool fl = !(fabs(a) <= t1) || !(fabs(b) <= t2);
        (is_row ? dbufs.rflag : dbufs.qflag)[idx] = fl;
        if (fl) note_flagged(is_row ? 0 : 1, idx, a, b, t1, t2);
      }
      FSTAMP();
      publish_flagged(p.counters + kCtrDecS2, p.counters + kCtrDecT2);
      FSTAMP();
    }
    grid_barrier(p.counters + kCtrDecBar, bar_target); stamp();
    // second decision, patch and report: block 0 alone (only CLEAN or point errors are accepted now)
    if (blockIdx.x == 0) {
      if (threadIdx.x == 0) publish_faults(st, flt);
      __syncthreads();
      FSTAMP();
      decide(st, syn, tolx, dbufs, n, m, p.level, 1, (int)__ldcg(p.counters + kCtrDecS2), (int)__ldcg(p.counters + kCtrDecT2), sc);
      FSTAMP();
      if (!patched && __ldcg(&st->verdict) == GECC_CORRECTED) patch_operands();
      FSTAMP();
      apply_plan_and_report();
    }
  }
  stamp();
  leave();
}

int decode_dispatch(int dtype, int64_t n, int64_t k, int64_t m, float* C, int64_t ldc, float* P_r, float* P_c, const float* P_g, const double* tau,
                    const double* sumsq_a, const double* sumsq_b, int level, int trans_a, int trans_b, void* A, int64_t lda, float* A_lo, const double* A_par64,
                    void* B, int64_t ldb, float* B_lo, const double* B_par64, gecc_report_t* report, uint8_t* ws, const WsLayout& L, cudaStream_t stream) {
  DecodeParams p;
  p.trans_a = trans_a; p.trans_b = trans_b;
  p.single = (level & GECC_SINGLE_CHECKSUM) ? 1 : 0;
  level = p.single ? 0 : (level & GECC_LEVEL_X);  // single-checksum mode decodes C_bar alone
  p.P_r_w = P_r; p.P_c_w = P_c; p.P_g = P_g;
  p.dtype = dtype; p.level = level; p.n = (int)n; p.k = (int)k; p.m = (int)m;
  p.C = C; p.ldc = ldc;
  p.fb.dtype = dtype; p.fb.n = (int)n; p.fb.m = (int)m;
  p.fb.rowpart = reinterpret_cast<const float*>(ws + L.rowpart);
  p.fb.colpart = reinterpret_cast<const float*>(ws + L.colpart);
  p.fb.P_r = P_r; p.fb.P_c = P_c;
  p.fb.syn = reinterpret_cast<double*>(ws + L.syn);
  p.fb.rflag = ws + L.flags;
  p.fb.qflag = ws + L.flags + ((n + 15) & ~15ll);
  p.ts.have_tau = tau != nullptr;
  for (int q = 0; q < 4; ++q) p.ts.tau[q] = tau ? tau[q] : 0.0;
  p.ts.sumsq_a = sumsq_a; p.ts.sumsq_b = sumsq_b;
  p.ts.noise_c = noise_coeff(dtype, (double)k);
  p.ts.single = p.single;
  p.A = A; p.lda = lda; p.A_lo = A_lo; p.A_par64 = A_par64;
  p.B = B; p.ldb = ldb; p.B_lo = B_lo; p.B_par64 = B_par64;
  p.report = report;
  p.counters = reinterpret_cast<unsigned int*>(ws);
  // scratch shared with the encoder: chunk partials of the verification pass over A ([chunks(n)][2][k]) and of the row
  // recomputation ([chunks(k)][m]); both fit the region ws_layout() reserved for the larger of the two operands
  p.encpart = reinterpret_cast<double*>(ws + enc_layout(n, k).encpart);
  p.recomp = reinterpret_cast<double*>(ws + L.recomp);
  p.votes = reinterpret_cast<int*>(ws + L.votes);
  p.lists = ws + L.lists;
  p.st = reinterpret_cast<DecodeState*>(ws + L.state);
  {
    const int64_t strips = (k + (dtype == GECC_BF16 ? 256 : 128) - 1) / (dtype == GECC_BF16 ? 256 : 128);
    if (level >= 1 && (trans_b ? 2 : 1) * strips > 512) return GECC_EUNSUPPORTED;  // arrival counters of the verification pass
    p.enc_chunk_rows = enc_chunk_rows(n, strips, num_sms());
    p.enc_chunk_rows_b = enc_chunk_rows(m, strips, num_sms());
  }
  p.encpart_b = reinterpret_cast<double*>(ws + L.encpart_b);
  p.G = 4.0 * kKappa * p.ts.noise_c * 5.9604644775390625e-08;
  p.stamps = reinterpret_cast<unsigned long long*>(ws + L.timing);

  const int sms = num_sms();
  if (sms <= 0) return GECC_ECUDA;
  int per_sm = 0;
  const void* fn = dtype == GECC_BF16 ? (const void*)decode_kernel<__nv_bfloat16> : (const void*)decode_kernel<float>;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, DT, 0) != cudaSuccess || per_sm < 1) return GECC_ECUDA;
  int grid = sms * (per_sm > 2 ? 2 : per_sm);
  if (grid > kMaxDecodeBlocks) grid = kMaxDecodeBlocks;
  // Cooperative (the blocks meet at grid barriers: they must be co-resident) and, after the product, a programmatic
  // dependent: the blocks may take their places while the product's last tiles drain; they wait for its completion
  // before they read anything (griddepcontrol.wait at the top of the kernel).
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(DT);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = stream;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeCooperative;
  attr[0].val.cooperative = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 2;
  void* args[] = {(void*)&p};
  if (cudaLaunchKernelExC(&cfg, fn, args) != cudaSuccess) {
    (void)cudaGetLastError();
    cfg.numAttrs = 1;  // cooperative only
    if (cudaLaunchKernelExC(&cfg, fn, args) != cudaSuccess) return GECC_ECUDA;
  }
  return GECC_OK;
}

}  // namespace gecc
