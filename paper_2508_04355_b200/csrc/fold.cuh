// Detection step of PAPER.md:192-217 for ONE line (row or column of C): the line's partial sums (left by the product's
// epilogue or by the unfused pass) are folded in fp64, the parity symbols are subtracted (sum minus parity,
// PAPER.md:194-200), and the two syndromes are compared with the thresholds of the line -> flag.
//
// Shared by the two places that run it:
//   * the protected product itself (gemm_sm100.cu): the CTA that completes the last block of a 128-row / 128-column strip
//     folds the strip's lines at once, so a fault-free product needs no decoder pass at all;
//   * the decoder (decode.cu) after the unfused pass over a stored C (gecc_syndrome_unfused), where no product ran.
#pragma once
#include <cuda_runtime.h>

#include "gecc_internal.h"

namespace gecc {

// Thresholds (reading R4; stated in include/gecc.h).  tau_plain = kappa c(k) 2^-24 sqrt(k len) sigma_a sigma_b;
// the weighted syndromes scale with the RMS weight.  sigma_c2 = k sigma_a^2 sigma_b^2 is the expected energy of one symbol
// of C: a line whose measured energy exceeds it gets a proportionally larger threshold (rounding noise is relative).
struct Thresholds {
  double tau[4];  // r1, r2, q1, q2
  double sigma_a, sigma_b, sigma_c2;
  int single;     // single-checksum mode: a line is flagged by its plain check alone
};

struct ThresholdSpec {
  int have_tau;
  double tau[4];          // caller's thresholds (have_tau) ...
  const double* sumsq_a;  // ... or the sums of squares of the operands from the encoder (device)
  const double* sumsq_b;
  double noise_c;         // c(k) of the noise law (gecc_internal.h)
  int single;             // GECC_SINGLE_CHECKSUM
};

__device__ inline void make_thresholds(const ThresholdSpec& s, int n_, int k_, int m_, Thresholds& z) {
  const double n = n_, k = k_, m = m_;
  double sa = 0.0, sb = 0.0;
  if (s.sumsq_a) sa = sqrt(__ldcg(s.sumsq_a) / (n * k));
  if (s.sumsq_b) sb = sqrt(__ldcg(s.sumsq_b) / (k * m));
  z.sigma_a = sa;
  z.sigma_b = sb;
  z.sigma_c2 = k * sa * sa * sb * sb;
  z.single = s.single;
  if (s.have_tau) {
    for (int q = 0; q < 4; ++q) z.tau[q] = s.tau[q];
  } else {
    const double base = kKappa * s.noise_c * 5.9604644775390625e-08 * sa * sb;
    z.tau[0] = base * sqrt(k * m);
    z.tau[2] = base * sqrt(k * n);
    z.tau[1] = z.tau[0] * sqrt((m + 1) * (2 * m + 1) / 6.0);
    z.tau[3] = z.tau[2] * sqrt((n + 1) * (2 * n + 1) / 6.0);
  }
}

// Where the folded lines go (all in the workspace).
struct FoldBufs {
  int dtype, n, m;
  const float* rowpart;  // [ceil(m / kSumCols)][n][4]
  const float* colpart;  // [ceil(n / kSumRows)][m][4]
  const float* P_r;      // [n x GECC_PR_LD]
  const float* P_c;      // [GECC_PAR_ROWS x m]
  double* syn;           // r1[n], r2[n], q1[m], q2[m], then the same four again: extra tolerance per line
  uint8_t* rflag;        // [align16(n)]
  uint8_t* qflag;        // [align16(m)]
};

struct FoldResult {
  double a, b;     // plain / weighted syndrome
  double t1, t2;   // thresholds of this line (tau + extra tolerance)
  bool flagged;
};

// The line's parity symbols as the product emitted them (limbs).
__device__ __forceinline__ void load_parity(const FoldBufs& f, bool is_row, int64_t idx, float (&pv)[6]) {
  if (is_row) {
    const float4 lo4 = __ldcg(reinterpret_cast<const float4*>(f.P_r + idx * GECC_PR_LD));
    const float4 hi4 = __ldcg(reinterpret_cast<const float4*>(f.P_r + idx * GECC_PR_LD + 4));
    pv[0] = lo4.x; pv[1] = lo4.y; pv[2] = lo4.z; pv[3] = lo4.w; pv[4] = hi4.x; pv[5] = hi4.y;
  } else {
#pragma unroll
    for (int u = 0; u < 6; ++u) pv[u] = __ldcg(f.P_c + (int64_t)u * f.m + idx);
  }
}

// From the line's sums (a = sum c, b = sum (index + 1) c, en = sum c^2) and its parity symbols to syndromes, thresholds and
// flag; stores the syndromes, the extra tolerances and the flag byte.  One thread per line.
__device__ __forceinline__ FoldResult finish_line(const FoldBufs& f, const Thresholds& th, bool is_row, int64_t idx, double a, double b, double en,
                                                  const float (&pv)[6]) {
  const int n = f.n, m = f.m;
  double p1, p2;
  if (f.dtype == GECC_BF16) { p1 = (double)pv[0] + (double)pv[1] + (double)pv[2]; p2 = (double)pv[3] + (double)pv[4] + (double)pv[5]; }
  else { p1 = (double)pv[0]; p2 = (double)pv[3]; }
  a -= p1;  // sum minus parity
  b -= p2;
  const double len = is_row ? (double)m : (double)n;
  double fe = th.sigma_c2 > 0.0 ? sqrt(en / (len * th.sigma_c2)) : 1.0;
  fe = fe > 1.0 ? fe : 1.0;  // NaN-safe: a non-finite energy leaves fe = 1 and the non-finite syndrome flags the line
  const double t1 = th.tau[is_row ? 0 : 2], t2 = th.tau[is_row ? 1 : 3];
  const double x1 = t1 * (fe - 1.0), x2 = t2 * (fe - 1.0);
  const int64_t o1 = is_row ? idx : 2 * (int64_t)n + idx, o2 = is_row ? n + idx : 2 * (int64_t)n + m + idx;
  double* tolx = f.syn + 2 * ((int64_t)n + m);
  f.syn[o1] = a; f.syn[o2] = b;
  tolx[o1] = x1; tolx[o2] = x2;
  const bool fl = !(fabs(a) <= t1 + x1) || (!th.single && !(fabs(b) <= t2 + x2));
  (is_row ? f.rflag : f.qflag)[idx] = fl;
  FoldResult r;
  r.a = a; r.b = b; r.t1 = t1 + x1; r.t2 = t2 + x2; r.flagged = fl;
  return r;
}

// G threads (G = 1 or a power of two <= 32, consecutive lanes, all of them calling) fold line `idx` from the per-block
// partial sums; the result is valid in the group's first lane (qd == 0).  `live` = false: the group only takes part in the
// shuffles.
template <int G>
__device__ __forceinline__ FoldResult fold_line(const FoldBufs& f, const Thresholds& th, bool is_row, int64_t idx, bool live, int qd) {
  const int n = f.n, m = f.m;
  const int ncb = (m + kSumCols - 1) / kSumCols, nrb = (n + kSumRows - 1) / kSumRows;
  const int nparts = is_row ? ncb : nrb;
  const int blk = is_row ? kSumCols : kSumRows;
  const float* part = is_row ? f.rowpart : f.colpart;
  const int64_t stride = is_row ? n : m;
  double a = 0.0, b = 0.0, en = 0.0;
  // the line's parity symbols (limbs), requested before the partials so that both round trips overlap
  float pv[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  if (live && qd == 0) load_parity(f, is_row, idx, pv);
  if (live) {
    for (int t0 = qd; t0 < nparts; t0 += 8 * G) {  // eight independent loads in flight per thread
      float4 v[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int t = t0 + G * u;
        v[u] = t < nparts ? __ldcg(reinterpret_cast<const float4*>(part + ((int64_t)t * stride + idx) * 4)) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int t = t0 + G * u;
        a += (double)v[u].x;
        b += (double)(t * blk + 1) * (double)v[u].x + (double)v[u].y;  // weight of 0-based index x is x + 1
        en += (double)v[u].z;
      }
    }
  }
#pragma unroll
  for (int o = 1; o < G; o <<= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, o);
    b += __shfl_xor_sync(0xffffffffu, b, o);
    en += __shfl_xor_sync(0xffffffffu, en, o);
  }
  FoldResult r;
  r.a = 0.0; r.b = 0.0; r.t1 = 0.0; r.t2 = 0.0; r.flagged = false;
  if (live && qd == 0) r = finish_line(f, th, is_row, idx, a, b, en, pv);
  return r;
}

// |syndrome| for the report's maxima; non-finite values count as 1e300.
__device__ __forceinline__ double abs_for_max(double v) { return (fabs(v) <= 1e300) ? fabs(v) : 1e300; }

}  // namespace gecc
