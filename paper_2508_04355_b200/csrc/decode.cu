// Correction step and its completion for input faults (readings R5-R9).
//
//   decide_kernel  : one block.  |E_r| = s, |E_t| = t -> min(s,t) >= 3: "needs to be recalculated";
//                    otherwise WLOG s <= t: locate the <= 2 faulty rows, estimate the errors from the
//                    column syndromes (s = 1: PAPER.md:223, s = 2: the 2x2 system of PAPER.md:227 with the right-hand
//                    side "sum minus parity"), classify whole-line faults (an input fault) vs points.
//   verify_compare : Level-X.  Column checks of A / row checks of B recomputed by the encoder kernels against the
//                    fp64 parity stored at encode time; locates (i, l, e) / (l, j, e).
//   repair_a / _b  : removes the exact rank-1 footprint of each located input fault from C and from the syndromes and
//                    patches the operand.
//   patch_kernel   : applies the plan to C in place (c_true = c - e) and writes the report.
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "gecc_internal.h"

namespace gecc {

constexpr int DT = 1024;  // threads of the decision block

struct Scratch {
  int i[32];
  unsigned long long u[32];
  int cnt;
  int idx[8];
  int flag;
};

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
// Collect (ascending) up to 4 indices i < len with pred(i); returns how many satisfied pred.
template <typename Pred>
__device__ int block_gather(int len, Pred pred, Scratch& sc, int (&out)[4]) {
  __syncthreads();
  if (threadIdx.x == 0) sc.cnt = 0;
  __syncthreads();
  for (int i = threadIdx.x; i < len; i += DT)
    if (pred(i)) {
      const int p = atomicAdd(&sc.cnt, 1);
      if (p < 8) sc.idx[p] = i;
    }
  __syncthreads();
  const int c = sc.cnt;
  int tmp[8];
  const int cc = c < 8 ? c : 8;
  for (int a = 0; a < cc; ++a) tmp[a] = sc.idx[a];
  for (int a = 0; a < cc; ++a)
    for (int b = a + 1; b < cc; ++b)
      if (tmp[b] < tmp[a]) { const int x = tmp[a]; tmp[a] = tmp[b]; tmp[b] = x; }
  for (int a = 0; a < 4; ++a) out[a] = a < cc ? tmp[a] : -1;
  __syncthreads();
  return c;
}

__device__ void sort_found(gecc_found_t* f, int n) {
  for (int a = 0; a < n; ++a)
    for (int b = a + 1; b < n; ++b) {
      const bool less = f[b].kind < f[a].kind || (f[b].kind == f[a].kind && (f[b].row < f[a].row || (f[b].row == f[a].row && f[b].col < f[a].col)));
      if (less) { const gecc_found_t t = f[a]; f[a] = f[b]; f[b] = t; }
    }
}

// post_repair = 0: Level-P on the syndromes as computed.  post_repair = 1: runs only if input faults were repaired;
// re-flags the updated syndromes and accepts CLEAN or point errors only.
// Every comparison uses the threshold of its own line: tau + tolx[line] (tolx: see syndrome_kernel).
__global__ void __launch_bounds__(DT) decide_kernel(DecodeState* st, double* syn, const double* tolx, uint8_t* flags, int* votes, int n, int m, int level,
                                                    int post_repair) {
  __shared__ Scratch sc;
  if (post_repair && !st->repaired) return;
  const double* r1 = syn; const double* r2 = syn + n; const double* q1 = syn + 2 * (int64_t)n; const double* q2 = syn + 2 * (int64_t)n + m;
  const double* xr1 = tolx; const double* xr2 = tolx + n; const double* xq1 = tolx + 2 * (int64_t)n; const double* xq2 = tolx + 2 * (int64_t)n + m;
  uint8_t* rflag = flags; uint8_t* qflag = flags + n;
  const double t_r1 = st->tau[0], t_r2 = st->tau[1], t_q1 = st->tau[2], t_q2 = st->tau[3];
  int s, t;
  if (post_repair) {
    int c = 0;
    for (int i = threadIdx.x; i < n; i += DT) { const bool f = !(fabs(r1[i]) <= t_r1 + xr1[i]) || !(fabs(r2[i]) <= t_r2 + xr2[i]); rflag[i] = f; c += f; }
    s = block_sum(c, sc);
    c = 0;
    for (int j = threadIdx.x; j < m; j += DT) { const bool f = !(fabs(q1[j]) <= t_q1 + xq1[j]) || !(fabs(q2[j]) <= t_q2 + xq2[j]); qflag[j] = f; c += f; }
    t = block_sum(c, sc);
  } else {
    s = st->n_row_flags;
    t = st->n_col_flags;
  }
  __syncthreads();

  // ---- decision; every thread computes the same scalars ----
  int verdict = GECC_UNCORRECTABLE;
  int nS = 0, S[2] = {-1, -1}, whole[2] = {0, 0};
  int npts = 0, pt_s[4], pt_l[4];
  double pt_x[4];
  int hidden_n = 0, hidden_s[2], hidden_l[2];
  double hidden_x[2];
  const bool rows_short = s <= t;
  // oriented views: "short" side holds the <= 2 faulty lines, "long" side supplies the syndromes used to correct
  const double* s1 = rows_short ? r1 : q1; const double* s2 = rows_short ? r2 : q2;
  const double* l1 = rows_short ? q1 : r1; const double* l2 = rows_short ? q2 : r2;
  const double* xs1 = rows_short ? xr1 : xq1; const double* xs2 = rows_short ? xr2 : xq2;
  const double* xl1 = rows_short ? xq1 : xr1; const double* xl2 = rows_short ? xq2 : xr2;
  const uint8_t* sflag = rows_short ? rflag : qflag; const uint8_t* lflag = rows_short ? qflag : rflag;
  const int n_short = rows_short ? n : m, n_long = rows_short ? m : n;
  const double tau_s1_ = rows_short ? t_r1 : t_q1, tol_s_ = rows_short ? t_r2 : t_q2;
  const double tau_l1_ = rows_short ? t_q1 : t_r1, tol_l_ = rows_short ? t_q2 : t_r2;
  auto tau_s1 = [&](int i) { return tau_s1_ + xs1[i]; };
  auto tol_s = [&](int i) { return tol_s_ + xs2[i]; };
  auto tau_l1 = [&](int j) { return tau_l1_ + xl1[j]; };
  auto tol_l = [&](int j) { return tol_l_ + xl2[j]; };

  bool ok = true;
  if (s == 0 && t == 0) { verdict = GECC_CLEAN; ok = false; }
  else if (s >= 3 && t >= 3) ok = false;  // min(s,t) >= 3

  int Sflag[2] = {-1, -1};
  int nSflag = 0;
  if (ok) {
    int g[4];
    nSflag = block_gather(n_short, [&](int i) { return sflag[i] != 0; }, sc, g);
    Sflag[0] = g[0]; Sflag[1] = g[1];
    nS = nSflag; S[0] = g[0]; S[1] = g[1];
    // A flagged long-side line j is explained by S if |S| = 2 (Theorem 2) or S = {s} and its two syndromes
    // are in the ratio of the weight of s (one error in line s).
    auto explained = [&](int j, int cnt, int a0) { return cnt == 2 || (cnt == 1 && fabs(l2[j] - (double)(a0 + 1) * l1[j]) <= tol_l(j)); };
    int c = 0;
    for (int j = threadIdx.x; j < n_long; j += DT) c += (lflag[j] && !explained(j, nS, S[0])) ? 1 : 0;
    const int nU = block_sum(c, sc);
    if (nU > 0) {
      // Input faults leave their own side's syndromes silent (reading R7): locate the line by the weighted ratio.
      for (int i = threadIdx.x; i < n_short; i += DT) votes[i] = 0;
      if (threadIdx.x == 0) sc.flag = 0;
      __syncthreads();
      for (int j = threadIdx.x; j < n_long; j += DT) {
        if (!lflag[j] || explained(j, nS, S[0])) continue;
        const double elig = tau_l1(j) > tol_l(j) ? tau_l1(j) : tol_l(j);  // ratio resolvable under the weighted noise
        if (!(fabs(l1[j]) > elig)) continue;                              // too weak to vote
        const double ratio = rint(l2[j] / l1[j]);
        const bool valid = ratio >= 1.0 && ratio <= (double)n_short && fabs(l2[j] - ratio * l1[j]) <= tol_l(j);
        if (valid) atomicAdd(&votes[(int)ratio - 1], 1);
        else atomicExch(&sc.flag, 1);
      }
      __syncthreads();
      const bool all_valid = sc.flag == 0;
      if (nS == 0) {
        int g2[4];
        const int distinct = block_gather(n_short, [&](int i) { return votes[i] > 0; }, sc, g2);
        if (!all_valid || distinct == 0 || distinct > 2) ok = false;
        else { nS = distinct; S[0] = g2[0]; S[1] = g2[1]; }
      } else {
        unsigned long long key = 0;
        for (int i = threadIdx.x; i < n_short; i += DT)
          if (i != S[0] && votes[i] > 0) {
            const unsigned long long kk = ((unsigned long long)votes[i] << 32) | (unsigned long long)(0x7FFFFFFF - i);  // mode, ties -> smallest
            key = kk > key ? kk : key;
          }
        key = block_max(key, sc);
        if (key == 0) ok = false;
        else {
          const int best = 0x7FFFFFFF - (int)(key & 0xFFFFFFFFull);
          const int a = S[0];
          S[0] = a < best ? a : best; S[1] = a < best ? best : a; nS = 2;
        }
      }
      if (ok) {
        c = 0;
        for (int j = threadIdx.x; j < n_long; j += DT) c += (lflag[j] && !explained(j, nS, S[0])) ? 1 : 0;
        if (block_sum(c, sc) > 0) ok = false;
      }
    }
    if (ok && nS == 0) ok = false;
  }

  if (ok) {
    const double w1 = (double)(S[0] + 1), w2 = (double)(S[1] + 1);
    // |S| = 2: x2 = (l2 - w1 l1) / (w2 - w1), x1 = l1 - x2.  The weighted syndrome's noise enters divided by (w2 - w1).
    auto xhat = [&](int idx, int j) -> double {
      if (nS == 1) return l1[j];
      const double x2 = (l2[j] - w1 * l1[j]) / (w2 - w1);
      return idx == 0 ? l1[j] - x2 : x2;
    };
    auto tau_loc = [&](int j) -> double {
      if (nS == 1) return tau_l1(j);
      const double amp = 2.0 * tol_l(j) / fabs(w2 - w1);
      return amp > tau_l1(j) ? amp : tau_l1(j);
    };
    // Two flagged rows and two flagged columns: within the two-error budget the errors sit on one diagonal of the 2x2
    // block.  In exact arithmetic the 2x2 solve below finds which; under fp32 noise its weighted right-hand side is
    // divided by (w2 - w1), so first test the two diagonals against all eight syndromes: plain sums must match pairwise,
    // weighted ones within their own threshold.  Exactly one consistent diagonal decides; none -> general solve
    // (more than two errors in the block, still E(2,2), Theorem 1); both -> indistinguishable under the noise.
    bool decided = false;
    const int n_long_flagged = rows_short ? t : s;
    if (nS == 2 && nSflag == 2 && n_long_flagged == 2) {
      int gl[4];
      block_gather(n_long, [&](int j) { return lflag[j] != 0; }, sc, gl);
      const int a = S[0], b = S[1], c = gl[0], d = gl[1];
      auto diag_ok = [&](int ca, int cb) {  // error of line a in long line ca, error of line b in long line cb
        return fabs(s1[a] - l1[ca]) <= tau_s1(a) + tau_l1(ca) && fabs(s1[b] - l1[cb]) <= tau_s1(b) + tau_l1(cb) &&
               fabs(l2[ca] - (double)(a + 1) * l1[ca]) <= tol_l(ca) && fabs(l2[cb] - (double)(b + 1) * l1[cb]) <= tol_l(cb) &&
               fabs(s2[a] - (double)(ca + 1) * s1[a]) <= tol_s(a) && fabs(s2[b] - (double)(cb + 1) * s1[b]) <= tol_s(b);
      };
      const bool h1 = diag_ok(c, d), h2 = diag_ok(d, c);
      if (h1 != h2) {
        const int ca = h1 ? c : d, cb = h1 ? d : c;
        pt_s[0] = a; pt_l[0] = ca; pt_x[0] = l1[ca];
        pt_s[1] = b; pt_l[1] = cb; pt_x[1] = l1[cb];
        npts = 2;
        decided = true;
      } else if (h1 && h2) ok = false;
    }
    for (int idx = 0; idx < nS && ok && !decided; ++idx) {
      const int sl = S[idx];
      const bool in_flag = (sl == Sflag[0] && nSflag > 0) || (sl == Sflag[1] && nSflag > 1);
      int g[4];
      const int ncols = block_gather(n_long, [&](int j) { return lflag[j] && fabs(xhat(idx, j)) > tau_loc(j); }, sc, g);
      if (!in_flag) whole[idx] = 1;  // located by the ratio only: an input fault
      else if (ncols >= 3) {
        // three bad symbols in one line exceed the budget unless an input fault made them; the line's own syndrome
        // then comes from a point error hiding in it
        whole[idx] = 1;
        if (!(fabs(s1[sl]) > tau_s1(sl))) ok = false;
        else {
          const double ratio = rint(s2[sl] / s1[sl]);
          if (!(ratio >= 1.0 && ratio <= (double)n_long && fabs(s2[sl] - ratio * s1[sl]) <= tol_s(sl))) ok = false;
          else { hidden_s[hidden_n] = sl; hidden_l[hidden_n] = (int)ratio - 1; hidden_x[hidden_n] = s1[sl]; ++hidden_n; }
        }
      } else if (ncols == 0) ok = false;  // flagged line with nothing locatable (e.g. a parity-symbol fault, R11)
      else {
        for (int a = 0; a < ncols; ++a) {
          const int j = g[a];
          double x = xhat(idx, j);
          if (nS == 2 && !(fabs(xhat(1 - idx, j)) > tau_loc(j))) x = l1[j];  // the other line is clean here: plain syndrome
          pt_s[npts] = sl; pt_l[npts] = j; pt_x[npts] = x; ++npts;
        }
      }
    }
    if (ok) verdict = GECC_CORRECTED;
  }
  if (post_repair && verdict == GECC_CORRECTED && (whole[0] || whole[1])) verdict = GECC_UNCORRECTABLE;

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
    if (verdict == GECC_CORRECTED) {
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
    if (!post_repair)
      st->need_verify = (level >= 1 && (verdict == GECC_UNCORRECTABLE || (verdict == GECC_CORRECTED && (whole[0] || whole[1])))) ? 1 : 0;
  }
}

// Level-X: compare the recomputed checks with the stored ones.  Unchanged lines reproduce bit for bit, so any
// difference is a fault; a single corrupted symbol per line is located by the ratio of its two differences.
// rel_tol bounds the rounding of the difference of two passes: bf16 symbols are summed in groups of 8 in fp32 with 6-bit
// weights (error <= 2^-24 x 56 (|e| + |a|) in the one group that changed), fp32 symbols in fp64 throughout.
__global__ void __launch_bounds__(DT) verify_compare_kernel(DecodeState* st, int dtype, const double* verA, const double* parA, const double* verB,
                                                             const double* parB, int n, int k, int m) {
  __shared__ Scratch sc;
  if (!st->need_verify) return;
  const double rel_tol = dtype == GECC_BF16 ? 1e-5 : 1e-11;
  for (int side = 0; side < 2; ++side) {
    const double* ver = side == 0 ? verA : verB;
    const double* par = side == 0 ? parA : parB;
    const int nline = side == 0 ? n : m;  // number of symbols each check spans
    const double sigma = side == 0 ? st->sigma_a : st->sigma_b;
    int g[4];
    const int cnt = block_gather(k, [&](int l) { return !(ver[l] - par[l] == 0.0) || !(ver[k + l] - par[k + l] == 0.0); }, sc, g);
    if (threadIdx.x == 0) {
      int okk = cnt <= kMaxInputFaults;
      int nf = 0;
      for (int a = 0; a < cnt && okk; ++a) {
        const int l = g[a];
        const double d1 = ver[l] - par[l], d2 = ver[k + l] - par[k + l];
        const double ratio = rint(d2 / d1);
        const double tol = rel_tol * (fabs(d1) + 8.0 * sigma) * (dtype == GECC_BF16 ? 1.0 : (double)nline);
        if (!(fabs(d1) > 0.0) || !(ratio >= 1.0 && ratio <= (double)nline) || !(fabs(d2 - ratio * d1) <= tol)) { okk = 0; break; }
        InputFault f;
        if (side == 0) { f.row = (int)ratio - 1; f.col = l; } else { f.row = l; f.col = (int)ratio - 1; }
        f.e = d1;
        if (side == 0) st->fa[nf++] = f; else st->fb[nf++] = f;
      }
      if (side == 0) { st->verify_ok_a = okk; st->n_fa = okk ? nf : 0; } else { st->verify_ok_b = okk; st->n_fb = okk ? nf : 0; }
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    if (!(st->verify_ok_a && st->verify_ok_b)) {
      st->verdict = GECC_UNCORRECTABLE_INPUT;
      st->n_found = 0; st->nS = 0; st->n_points = 0; st->whole_line[0] = st->whole_line[1] = 0;
      st->repaired = 0;
    } else if (st->n_fa + st->n_fb > 0) {
      st->repaired = 1;  // the Level-P plan is dropped; repair, then decide again
    } else {
      st->repaired = 0;  // memory intact (transient fault): keep the Level-P result
    }
  }
}

template <typename T>
__device__ __forceinline__ double load_sym(const T* p);
template <>
__device__ __forceinline__ double load_sym<__nv_bfloat16>(const __nv_bfloat16* p) { return (double)__bfloat162float(*p); }
template <>
__device__ __forceinline__ double load_sym<float>(const float* p) { return (double)*p; }

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
  if (X_lo) X_lo[idx] = v - __uint_as_float(__float_as_uint(v) & 0xFFFFE000u);
}

// (A + E_A)(B + E_B) = A B + E_A (B + E_B) + A E_B: first remove e b~_l* from row i using the still-faulty B ...
template <typename T>
__global__ void repair_a_kernel(DecodeState* st, float* C, int64_t ldc, double* syn, double* tolx, double G, T* A, int64_t lda, float* A_lo, const T* B,
                                int64_t ldb, int n, int m, const double* verB, const double* parB, int k) {
  if (!st->repaired) return;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  double* q1 = syn + 2 * (int64_t)n; double* q2 = q1 + m;
  double* xq1 = tolx + 2 * (int64_t)n; double* xq2 = xq1 + m;
  const double Grow = G / sqrt((double)m);
  // Row i of C_bar moves by e b~_l* in its data part but by e B_P[l] (clean parity) in its parity part: if row l of B
  // is itself faulty the row checks of C see e times B's own check differences (the A x B cross term).
  if (j < st->n_fa) {
    const int i = st->fa[j].row, l = st->fa[j].col;
    atomicAdd(&syn[i], -st->fa[j].e * (verB[l] - parB[l]));
    atomicAdd(&syn[n + i], -st->fa[j].e * (verB[k + l] - parB[k + l]));
  }
  for (int a = 0; a < st->n_fa; ++a) {
    const int i = st->fa[a].row, l = st->fa[a].col;
    const double e = st->fa[a].e;
    // The symbol that carried the footprint d was accumulated (with truncation) and summed in fp32 at the footprint's
    // magnitude: what the exact subtraction leaves behind is bounded relative to |d|, not to the data.  G |d| is added
    // to the thresholds of the lines that summed it (the column directly, the row through G / sqrt(m) of its L1 norm).
    double ad = 0.0;
    if (j < m) {
      const double d = e * load_sym<T>(B + (int64_t)l * ldb + j);
      C[(int64_t)i * ldc + j] = (float)((double)C[(int64_t)i * ldc + j] - d);
      q1[j] -= d;
      q2[j] -= (double)(i + 1) * d;
      ad = fabs(d);
      xq1[j] += G * ad;
      xq2[j] += G * (double)(i + 1) * ad;
    }
    double a1 = ad, a2 = (double)(j + 1) * ad;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { a1 += __shfl_xor_sync(0xffffffffu, a1, o); a2 += __shfl_xor_sync(0xffffffffu, a2, o); }
    if ((threadIdx.x & 31) == 0 && a1 > 0.0) { atomicAdd(&tolx[i], Grow * a1); atomicAdd(&tolx[n + i], Grow * a2); }
  }
  if (j < st->n_fa) patch_sym<T>(A, A_lo, (int64_t)st->fa[j].row * lda + st->fa[j].col, st->fa[j].e);
}
// ... then e' a_*l from column j using the patched A.
template <typename T>
__global__ void repair_b_kernel(DecodeState* st, float* C, int64_t ldc, double* syn, double* tolx, double G, const T* A, int64_t lda, T* B, int64_t ldb,
                                float* B_lo, int n, int m) {
  if (!st->repaired) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  double* r1 = syn; double* r2 = syn + n;
  double* xr1 = tolx; double* xr2 = tolx + n;
  const double Gcol = G / sqrt((double)n);
  for (int a = 0; a < st->n_fb; ++a) {
    const int l = st->fb[a].row, j = st->fb[a].col;
    const double e = st->fb[a].e;
    double ad = 0.0;
    if (i < n) {
      const double d = e * load_sym<T>(A + (int64_t)i * lda + l);
      C[(int64_t)i * ldc + j] = (float)((double)C[(int64_t)i * ldc + j] - d);
      r1[i] -= d;
      r2[i] -= (double)(j + 1) * d;
      ad = fabs(d);
      xr1[i] += G * ad;
      xr2[i] += G * (double)(j + 1) * ad;
    }
    double a1 = ad, a2 = (double)(i + 1) * ad;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { a1 += __shfl_xor_sync(0xffffffffu, a1, o); a2 += __shfl_xor_sync(0xffffffffu, a2, o); }
    if ((threadIdx.x & 31) == 0 && a1 > 0.0) { atomicAdd(&tolx[2 * (int64_t)n + j], Gcol * a1); atomicAdd(&tolx[2 * (int64_t)n + m + j], Gcol * a2); }
  }
  if (i < st->n_fb) patch_sym<T>(B, B_lo, (int64_t)st->fb[i].row * ldb + st->fb[i].col, st->fb[i].e);
}

// A symbol of C that carried both an A-fault and a B-fault footprint held their product e_A e_B (the cross term, which
// can exceed the data by orders of magnitude) when the tensor cores rounded it: what is left after the exact repairs
// is that rounding error.  Such symbols (at most n_fa x n_fb of them) are recomputed from the patched operands, which is
// what "mark the compromised data for recomputation" asks for; the syndromes follow the change.
// One warp per (A fault, B fault) pair.
template <typename T>
__global__ void recompute_cross_kernel(DecodeState* st, float* C, int64_t ldc, double* syn, const T* A, int64_t lda, const T* B, int64_t ldb, int n, int m,
                                       int k) {
  if (!st->repaired) return;
  const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nfa = st->n_fa, nfb = st->n_fb;
  if (w >= nfa * nfb) return;
  const int i = st->fa[w / nfb].row, j = st->fb[w % nfb].col;
  if (st->fa[w / nfb].col != st->fb[w % nfb].row) return;  // no shared l: no cross term
  double acc = 0.0;
  for (int l = lane; l < k; l += 32) acc += load_sym<T>(A + (int64_t)i * lda + l) * load_sym<T>(B + (int64_t)l * ldb + j);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) {
    const float nv = (float)acc;
    const double delta = (double)nv - (double)C[(int64_t)i * ldc + j];
    C[(int64_t)i * ldc + j] = nv;
    atomicAdd(&syn[i], delta);
    atomicAdd(&syn[n + i], (double)(j + 1) * delta);
    atomicAdd(&syn[2 * (int64_t)n + j], delta);
    atomicAdd(&syn[2 * (int64_t)n + m + j], (double)(i + 1) * delta);
  }
}

// c_true = c - e.  Whole-line faults are corrected along the whole line (reading R6), points only
// where located (reading R5).  Block 0 also writes the report.
__global__ void patch_kernel(DecodeState* st, float* C, int64_t ldc, const double* syn, int n, int m, gecc_report_t* report) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  const bool apply = st->verdict == GECC_CORRECTED;
  if (apply) {
    const bool rows_short = st->rows_short != 0;
    const double* l1 = rows_short ? syn + 2 * (int64_t)n : syn;
    const double* l2 = rows_short ? syn + 2 * (int64_t)n + m : syn + n;
    const int n_long = rows_short ? m : n;
    const int nS = st->nS;
    const double w1 = (double)(st->S[0] + 1), w2 = (double)(st->S[1] + 1);
    if (g < n_long) {
      for (int idx = 0; idx < nS; ++idx) {
        if (!st->whole_line[idx]) continue;
        double x;
        if (nS == 1) x = l1[g];
        else { const double x2 = (l2[g] - w1 * l1[g]) / (w2 - w1); x = idx == 0 ? l1[g] - x2 : x2; }
        const int64_t off = rows_short ? (int64_t)st->S[idx] * ldc + g : (int64_t)g * ldc + st->S[idx];
        C[off] = (float)((double)C[off] - x);
      }
    }
    if (g < st->n_points) {
      const int sl = st->pt_s[g], ll = st->pt_l[g];
      bool in_whole = false;  // already corrected along its line
      for (int idx = 0; idx < nS; ++idx) in_whole |= st->whole_line[idx] && st->S[idx] == sl;
      if (!in_whole) {
        const int64_t off = rows_short ? (int64_t)sl * ldc + ll : (int64_t)ll * ldc + sl;
        C[off] = (float)((double)C[off] - st->pt_x[g]);
      }
    }
  }
  if (g == 0) {
    report->verdict = st->verdict;
    report->n_found = st->n_found;
    report->n_row_flags = st->n_row_flags0;
    report->n_col_flags = st->n_col_flags0;
    for (int q = 0; q < 4; ++q) {
      report->max_abs_syndrome[q] = __longlong_as_double((long long)st->maxabs_bits[q]);
      report->tau[q] = st->tau[q];
    }
    for (int a = 0; a < GECC_MAX_FOUND; ++a) report->found[a] = a < st->n_found ? st->found[a] : gecc_found_t{-1, -1, -1, 0, 0.0};
  }
}

// declared in syndrome.cu
__global__ void decode_init_kernel(DecodeState* st, int dtype, int64_t n, int64_t k, int64_t m, bool have_tau, double t0, double t1, double t2,
                                   double t3, const double* sumsq_a, const double* sumsq_b);
__global__ void syndrome_kernel(int dtype, int n, int m, int nb, int slabs, const float* __restrict__ rowpart, const float* __restrict__ colpart,
                                const float* __restrict__ P_r, const float* __restrict__ P_c, double* __restrict__ syn, uint8_t* __restrict__ flags,
                                DecodeState* st);

template <typename T>
static void launch_repairs(DecodeState* st, float* C, int64_t ldc, double* syn, double* tolx, double G, void* A, int64_t lda, float* A_lo, void* B,
                           int64_t ldb, float* B_lo, int n, int m, const double* verB, const double* parB, int k, cudaStream_t stream) {
  repair_a_kernel<T><<<(m + 255) / 256, 256, 0, stream>>>(st, C, ldc, syn, tolx, G, reinterpret_cast<T*>(A), lda, A_lo, reinterpret_cast<const T*>(B), ldb,
                                                         n, m, verB, parB, k);
  repair_b_kernel<T><<<(n + 255) / 256, 256, 0, stream>>>(st, C, ldc, syn, tolx, G, reinterpret_cast<const T*>(A), lda, reinterpret_cast<T*>(B), ldb, B_lo,
                                                         n, m);
  recompute_cross_kernel<T><<<1, 32 * kMaxInputFaults * kMaxInputFaults, 0, stream>>>(st, C, ldc, syn, reinterpret_cast<const T*>(A), lda,
                                                                                   reinterpret_cast<const T*>(B), ldb, n, m, k);
}

int decode_dispatch(int dtype, int64_t n, int64_t k, int64_t m, float* C, int64_t ldc, const float* P_r, const float* P_c, const double* tau,
                    const double* sumsq_a, const double* sumsq_b, int level, void* A, int64_t lda, float* A_lo, const double* A_par64, void* B,
                    int64_t ldb, float* B_lo, const double* B_par64, gecc_report_t* report, uint8_t* ws, const WsLayout& L, cudaStream_t stream) {
  DecodeState* st = reinterpret_cast<DecodeState*>(ws + L.state);
  double* syn = reinterpret_cast<double*>(ws + L.syn);
  double* tolx = syn + 2 * (n + m);  // per-line extra tolerance (syndrome_kernel, repair kernels)
  const double G = 4.0 * kKappa * noise_coeff(dtype, (double)k) * 5.9604644775390625e-08;  // residual allowance per unit of removed footprint
  uint8_t* flags = ws + L.flags;
  int* votes = reinterpret_cast<int*>(ws + L.votes);
  const int bn = block_n(dtype);
  const int nb = (int)((m + bn - 1) / bn), slabs = (int)(((n + 127) / 128) * 4);
  decode_init_kernel<<<1, 1, 0, stream>>>(st, dtype, n, k, m, tau != nullptr, tau ? tau[0] : 0.0, tau ? tau[1] : 0.0, tau ? tau[2] : 0.0,
                                          tau ? tau[3] : 0.0, sumsq_a, sumsq_b);
  syndrome_kernel<<<(unsigned)((n + m + 255) / 256), 256, 0, stream>>>(dtype, (int)n, (int)m, nb, slabs, reinterpret_cast<const float*>(ws + L.rowpart),
                                                                      reinterpret_cast<const float*>(ws + L.colpart), P_r, P_c, syn, flags, st);
  decide_kernel<<<1, DT, 0, stream>>>(st, syn, tolx, flags, votes, (int)n, (int)m, level, 0);
  if (level >= 1) {
    double* verA = reinterpret_cast<double*>(ws + L.ver64);
    double* verB = verA + 2 * k;
    double* encpart = reinterpret_cast<double*>(ws + L.encpart);
    int rc;
    if ((rc = encode_dispatch(dtype, true, A, n, k, lda, nullptr, nullptr, nullptr, verA, nullptr, encpart, nullptr, &st->need_verify, stream))) return rc;
    if ((rc = encode_dispatch(dtype, false, B, k, m, ldb, nullptr, nullptr, nullptr, verB, nullptr, encpart, nullptr, &st->need_verify, stream))) return rc;
    verify_compare_kernel<<<1, DT, 0, stream>>>(st, dtype, verA, A_par64, verB, B_par64, (int)n, (int)k, (int)m);
    if (dtype == GECC_BF16) launch_repairs<__nv_bfloat16>(st, C, ldc, syn, tolx, G, A, lda, A_lo, B, ldb, B_lo, (int)n, (int)m, verB, B_par64, (int)k, stream);
    else launch_repairs<float>(st, C, ldc, syn, tolx, G, A, lda, A_lo, B, ldb, B_lo, (int)n, (int)m, verB, B_par64, (int)k, stream);
    decide_kernel<<<1, DT, 0, stream>>>(st, syn, tolx, flags, votes, (int)n, (int)m, level, 1);
  }
  const int64_t mx = n > m ? n : m;
  patch_kernel<<<(unsigned)((mx + 255) / 256), 256, 0, stream>>>(st, C, ldc, syn, (int)n, (int)m, report);
  return cudaGetLastError() == cudaSuccess ? GECC_OK : GECC_ECUDA;
}

}  // namespace gecc
