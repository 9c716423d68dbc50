// Tile-local grid (a variant of Def. 1): one code M(P + 2, k, Q + 2) per block of P = 128 rows
// of A and Q = 128 columns of B, weights local to the panel (1..128).  Every 128 x 128 block of C is a codeword of its own:
// it corrects its own errors (min(s, t) <= 2 per block, Theorem 2), its thresholds do not grow with n or m,
// and the weights are exact in bf16.
//
//   tl_encode_kernel (A) A_PL[8 p + 3 c + l][col] = limb l of sum_{i in panel p} w_c(i) a_{i,col}     (PAPER.md:71-83 per panel)
//   tl_encode_kernel (B) B_PL[8 q + 3 c + l][row] = limb l of sum_{j in panel q} w_c(j) b_{row,j}     (PAPER.md:89-101 per panel)
//   (gemm_sm100.cu)      C = A B with the per-block detection sums in the epilogue, P_cL = A_PL B, P_rL = A B_PL^T as data-sized tiles
//   tl_decode_kernel     per block: syndromes = sums - parity, flags (215-217), the decoder of PAPER.md:219-231
//                        with the completions of DESIGN.md (R5-R8, R21) on the block's 128 + 128 lines, c_true = c - e in place
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "../../include/gecc.h"
#include "encode_core.cuh"
#include "fold.cuh"
#include "gecc_internal.h"
#include "sm100_ptx.cuh"

namespace gecc {

constexpr int kTlPanel = 128;             // must equal kSumRows and kSumCols: the product's epilogue sums per block of 128
constexpr int kTlRows = GECC_PAR_ROWS;    // rows of A_PL / B_PL per panel: 2 checks x 3 limbs (bf16), padded to 8
static_assert(kTlPanel == kSumRows && kTlPanel == kSumCols, "tile-local panels are the blocks of the detection sums");

__device__ __forceinline__ float tl_tf32_trunc(float x) { return __uint_as_float(__float_as_uint(x) & 0xFFFFE000u); }

// The two checks of one line of one panel, as the product consumes them (same limb layout as the global code's parity:
// bf16 rows 3 c + l; fp32: tf32 hi part in row 3 c, remainder in the lo plane).  base: row 8 * panel of the parity operand.
template <typename T>
__device__ __forceinline__ void tl_write_checks(T* par, float* par_lo, int64_t k, int64_t base_row, int64_t idx, double s1, double s2);
template <>
__device__ __forceinline__ void tl_write_checks<__nv_bfloat16>(__nv_bfloat16* par, float*, int64_t k, int64_t base_row, int64_t idx, double s1, double s2) {
  const double s[2] = {s1, s2};
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    double rem = s[c];
#pragma unroll
    for (int l = 0; l < 3; ++l) {
      const __nv_bfloat16 h = __double2bfloat16(rem);
      par[(base_row + 3 * c + l) * k + idx] = h;
      rem -= (double)__bfloat162float(h);
    }
  }
  par[(base_row + 6) * k + idx] = __float2bfloat16(0.f);
  par[(base_row + 7) * k + idx] = __float2bfloat16(0.f);
}
template <>
__device__ __forceinline__ void tl_write_checks<float>(float* par, float* par_lo, int64_t k, int64_t base_row, int64_t idx, double s1, double s2) {
  const double s[2] = {s1, s2};
#pragma unroll
  for (int r = 0; r < kTlRows; ++r) {
    float hi = 0.f, lo = 0.f;
    if (r == 0 || r == 3) {
      const float v = (float)s[r / 3];
      hi = tl_tf32_trunc(v);
      lo = v - hi;
    }
    par[(base_row + r) * k + idx] = hi;
    par_lo[(base_row + r) * k + idx] = lo;
  }
}

// One 16-byte vector of the operand as packed fp32 pairs (sm_100 FADD2 / FFMA2: two symbols per instruction, as in encode_core.cuh).
template <typename T>
struct TlVec;
template <>
struct TlVec<__nv_bfloat16> {
  static constexpr int V = 8, H = 4;
  __device__ static void pairs(const uint4& r, f32x2 (&xx)[4]) {
    xx[0] = bf16x2_widen(r.x); xx[1] = bf16x2_widen(r.y); xx[2] = bf16x2_widen(r.z); xx[3] = bf16x2_widen(r.w);
  }
};
template <>
struct TlVec<float> {
  static constexpr int V = 4, H = 2;
  __device__ static void pairs(const uint4& r, f32x2 (&xx)[2]) {
    xx[0] = pack2(__uint_as_float(r.x), __uint_as_float(r.y)); xx[1] = pack2(__uint_as_float(r.z), __uint_as_float(r.w));
  }
};
__device__ __forceinline__ void tl_store_lo(float* dst, const uint4& r) {  // 3xTF32: the low parts of four fp32 symbols, x - tf32(x)
  const float x0 = __uint_as_float(r.x), x1 = __uint_as_float(r.y), x2 = __uint_as_float(r.z), x3 = __uint_as_float(r.w);
  *reinterpret_cast<float4*>(dst) = make_float4(x0 - tl_tf32_trunc(x0), x1 - tl_tf32_trunc(x1), x2 - tl_tf32_trunc(x2), x3 - tl_tf32_trunc(x3));
}

// ---------------------------------------------------------------------------------------------------------------
// A side: sums over the 128 rows of each panel.  One block per (column strip of 32 x V columns, panel), 256 threads as (32, 8): thread
// (tx, ty) sums 16 rows of V columns (16-byte loads, all 16 in flight), the eight row groups are added through shared memory.
// ---------------------------------------------------------------------------------------------------------------
template <typename T>
struct TlEncSmem {
  float sh[8][2][TlVec<T>::V][33];   // A role: partial sums of the eight row groups
  float res[8][2][32];               // B role: the two checks of 8 panels x 32 rows
  float shq[8];
};

// Returns the block's sum of squares in thread 0.  Sums of 16 rows are kept in fp32 (bf16 symbols times weights <= 128 are exact
// products; the rounding of the additions, 2^-24 relative, is that of the limbs the checks are stored in), the eight row
// groups are added in fp64.
template <typename T>
__device__ __forceinline__ double tl_encode_a_block(const T* __restrict__ A, int64_t n, int64_t k, int64_t lda, float* __restrict__ A_lo, T* __restrict__ A_PL,
                                                    float* __restrict__ A_PL_lo, int bx, int by, TlEncSmem<T>& sm) {
  constexpr int V = TlVec<T>::V;
  constexpr int RG = 8, RPT = kTlPanel / RG, BATCH = 8;  // row groups, rows per thread, loads in flight per thread
  auto& sh = sm.sh;
  auto& shq = sm.shq;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const int64_t col = ((int64_t)bx * 32 + tx) * V;
  const int64_t r0 = (int64_t)by * kTlPanel + ty * RPT;
  constexpr int H = TlVec<T>::H;
  f32x2 s1[H], s2[H], q2[H];
#pragma unroll
  for (int i = 0; i < H; ++i) { s1[i] = pack2(0.f, 0.f); s2[i] = s1[i]; q2[i] = s1[i]; }
  if (col < k) {
#pragma unroll
    for (int b0 = 0; b0 < RPT; b0 += BATCH) {
      uint4 raw[BATCH];
#pragma unroll
      for (int rr = 0; rr < BATCH; ++rr) {
        raw[rr] = make_uint4(0u, 0u, 0u, 0u);
        ld_stream_if(raw[rr], A + (r0 + b0 + rr) * lda + col, r0 + b0 + rr < n);
      }
#pragma unroll
      for (int rr = 0; rr < BATCH; ++rr) {
        const float w = (float)(ty * RPT + b0 + rr + 1);  // weight of the 0-based row within its panel, plus one
        const f32x2 w2 = pack2(w, w);
        if (sizeof(T) == 4 && r0 + b0 + rr < n) tl_store_lo(A_lo + (r0 + b0 + rr) * lda + col, raw[rr]);
        f32x2 xx[H];
        TlVec<T>::pairs(raw[rr], xx);
#pragma unroll
        for (int i = 0; i < H; ++i) {
          s1[i] = add2(s1[i], xx[i]);
          s2[i] = fma2(w2, xx[i], s2[i]);
          q2[i] = fma2(xx[i], xx[i], q2[i]);
        }
      }
    }
  }
  float a1[V], a2[V];
  float sq = 0.f;
#pragma unroll
  for (int i = 0; i < H; ++i) {
    float lo, hi;
    unpack2(s1[i], a1[2 * i], a1[2 * i + 1]);
    unpack2(s2[i], a2[2 * i], a2[2 * i + 1]);
    unpack2(q2[i], lo, hi);
    sq += lo + hi;
  }
#pragma unroll
  for (int v = 0; v < V; ++v) { sh[ty][0][v][tx] = a1[v]; sh[ty][1][v][tx] = a2[v]; }
  for (int o = 16; o > 0; o >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, o);
  if (tx == 0) shq[ty] = sq;
  __syncthreads();
  // the V columns of each lane are spread over the row groups: thread (tx, ty) finishes column tx * V + ty
  for (int v = ty; v < V; v += RG) {
    double s1 = 0.0, s2 = 0.0;
#pragma unroll
    for (int g = 0; g < RG; ++g) { s1 += (double)sh[g][0][v][tx]; s2 += (double)sh[g][1][v][tx]; }
    if (col + v < k) tl_write_checks<T>(A_PL, A_PL_lo, k, (int64_t)by * kTlRows, col + v, s1, s2);
  }
  double t = 0.0;
  if (tx == 0 && ty == 0)
    for (int g = 0; g < RG; ++g) t += (double)shq[g];
  return t;
}

// ---------------------------------------------------------------------------------------------------------------
// B side: sums along each row over the 128 columns of each panel.  One block per (group of 32 rows, chunk of 8 panels), 256
// threads: warp w takes rows 4 w .. 4 w + 3; a 16-byte load per lane covers 128 / V ... lanes of one panel (bf16: 16 lanes, two
// panels per warp load; fp32: all 32 lanes, one panel), reduced by shuffles; the block writes its 32 rows of each parity row
// as one contiguous segment.
// ---------------------------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ double tl_encode_b_block(const T* __restrict__ B, int64_t k, int64_t m, int64_t ldb, float* __restrict__ B_lo, T* __restrict__ B_PL,
                                                    float* __restrict__ B_PL_lo, int bx, int by, TlEncSmem<T>& sm) {
  constexpr int V = TlVec<T>::V;
  constexpr int LPP = kTlPanel / V;   // lanes per panel: 16 (bf16) / 32 (fp32)
  constexpr int PPW = 32 / LPP;       // panels per warp load: 2 / 1
  constexpr int PCH = 8;              // panels per block
  auto& res = sm.res;
  auto& shq = sm.shq;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int64_t l0 = (int64_t)bx * 32;
  const int64_t p0 = (int64_t)by * PCH;
  const int64_t npanels = (m + kTlPanel - 1) / kTlPanel;
  const int sub = lane / LPP;                 // which of the warp load's panels this lane reads
  const int jl = (lane % LPP) * V;            // first column of the lane within its panel
  constexpr int H = TlVec<T>::H;
  f32x2 wv[H];  // weights of the lane's columns within their panel, plus one
#pragma unroll
  for (int i = 0; i < H; ++i) wv[i] = pack2((float)(jl + 2 * i + 1), (float)(jl + 2 * i + 2));
  f32x2 q2 = pack2(0.f, 0.f);
  for (int r2 = 0; r2 < 4; r2 += 2) {  // two rows at a time: eight loads per lane in flight
    uint4 raw[2][PCH / PPW];
#pragma unroll
    for (int rr = 0; rr < 2; ++rr) {
      const int64_t l = l0 + warp * 4 + r2 + rr;
#pragma unroll
      for (int it = 0; it < PCH / PPW; ++it) {
        const int64_t j = (p0 + it * PPW + sub) * kTlPanel + jl;
        raw[rr][it] = make_uint4(0u, 0u, 0u, 0u);
        ld_stream_if(raw[rr][it], B + l * ldb + j, l < k && j < m);
      }
    }
#pragma unroll
    for (int rr = 0; rr < 2; ++rr) {
      const int64_t l = l0 + warp * 4 + r2 + rr;
#pragma unroll
      for (int it = 0; it < PCH / PPW; ++it) {
        const int64_t j = (p0 + it * PPW + sub) * kTlPanel + jl;
        if (sizeof(T) == 4 && l < k && j < m) tl_store_lo(B_lo + l * ldb + j, raw[rr][it]);
        f32x2 xx[H];
        TlVec<T>::pairs(raw[rr][it], xx);
        f32x2 t1 = xx[0], t2 = mul2(wv[0], xx[0]);
        q2 = fma2(xx[0], xx[0], q2);
#pragma unroll
        for (int i = 1; i < H; ++i) {
          t1 = add2(t1, xx[i]);
          t2 = fma2(wv[i], xx[i], t2);
          q2 = fma2(xx[i], xx[i], q2);
        }
        float s1, s2, h1, h2;
        unpack2(t1, s1, h1);
        unpack2(t2, s2, h2);
        s1 += h1; s2 += h2;
#pragma unroll
        for (int o = LPP / 2; o > 0; o >>= 1) {
          s1 += __shfl_xor_sync(0xffffffffu, s1, o);
          s2 += __shfl_xor_sync(0xffffffffu, s2, o);
        }
        if (lane % LPP == 0) { res[it * PPW + sub][0][warp * 4 + r2 + rr] = s1; res[it * PPW + sub][1][warp * 4 + r2 + rr] = s2; }
      }
    }
  }
  float sq;
  {
    float lo, hi;
    unpack2(q2, lo, hi);
    sq = lo + hi;
  }
  for (int o = 16; o > 0; o >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, o);
  if (lane == 0) shq[warp] = sq;
  __syncthreads();
  {
    const int pl = threadIdx.x >> 5, li = threadIdx.x & 31;  // panel of the chunk, row of the group
    if (p0 + pl < npanels && l0 + li < k)
      tl_write_checks<T>(B_PL, B_PL_lo, k, (p0 + pl) * kTlRows, l0 + li, (double)res[pl][0][li], (double)res[pl][1][li]);
  }
  double t = 0.0;
  if (threadIdx.x == 0)
    for (int g = 0; g < 8; ++g) t += (double)shq[g];
  return t;
}

// Both operands in one launch: blocks [0, na) encode A (na = column strips x row panels), the rest encode B (groups of 32 rows
// x chunks of 8 column panels).  Sums of squares: per-block partials added to two accumulators in the workspace; the last
// block to arrive moves them to sumsq_a / sumsq_b and leaves accumulators and counter zero for the next call.
struct TlEncParams {
  const void* A; const void* B;
  int64_t n, k, m, lda, ldb;
  float* A_lo; float* B_lo;
  void* A_PL; void* B_PL;
  float* A_PL_lo; float* B_PL_lo;
  double* sumsq_a; double* sumsq_b;
  unsigned int* counters;
  int gxa, na, gxb, nb;
};
template <typename T>
__global__ void __launch_bounds__(256, sizeof(T) == 2 ? 3 : 2) tl_encode_kernel(const __grid_constant__ TlEncParams p) {
  __shared__ TlEncSmem<T> sm;
  const int b = blockIdx.x;
  const bool of_a = b < p.na;
  double t;
  if (of_a) t = tl_encode_a_block<T>(reinterpret_cast<const T*>(p.A), p.n, p.k, p.lda, p.A_lo, reinterpret_cast<T*>(p.A_PL), p.A_PL_lo, b % p.gxa, b / p.gxa, sm);
  else t = tl_encode_b_block<T>(reinterpret_cast<const T*>(p.B), p.k, p.m, p.ldb, p.B_lo, reinterpret_cast<T*>(p.B_PL), p.B_PL_lo, (b - p.na) % p.gxb, (b - p.na) / p.gxb, sm);
  ptx::griddep_launch_dependents();
  if (threadIdx.x == 0) {
    double* acc = reinterpret_cast<double*>(p.counters + kCtrTlSumsq);
    atomicAdd(acc + (of_a ? 0 : 1), t);
    __threadfence();
    if (atomicAdd(p.counters + kCtrTlArrive, 1u) == gridDim.x - 1u) {
      __threadfence();
      *p.sumsq_a = __ldcg(acc); *p.sumsq_b = __ldcg(acc + 1);
      acc[0] = 0.0; acc[1] = 0.0;
      p.counters[kCtrTlArrive] = 0;
    }
  }
}

int tl_encode_dispatch(int dtype, int64_t n, int64_t k, int64_t m, const void* A, int64_t lda, float* A_lo, void* A_PL, float* A_PL_lo, double* sumsq_a,
                       const void* B, int64_t ldb, float* B_lo, void* B_PL, float* B_PL_lo, double* sumsq_b, uint8_t* ws, cudaStream_t stream) {
  const int64_t np = (n + kTlPanel - 1) / kTlPanel, mp = (m + kTlPanel - 1) / kTlPanel;
  const int V = dtype == GECC_BF16 ? 8 : 4;
  TlEncParams p;
  p.A = A; p.B = B; p.n = n; p.k = k; p.m = m; p.lda = lda; p.ldb = ldb;
  p.A_lo = A_lo; p.B_lo = B_lo; p.A_PL = A_PL; p.B_PL = B_PL; p.A_PL_lo = A_PL_lo; p.B_PL_lo = B_PL_lo;
  p.sumsq_a = sumsq_a; p.sumsq_b = sumsq_b;
  p.counters = reinterpret_cast<unsigned int*>(ws);
  p.gxa = (int)((k + 32 * V - 1) / (32 * V));
  p.gxb = (int)((k + 31) / 32);
  const int64_t na = (int64_t)p.gxa * np, nb = (int64_t)p.gxb * ((mp + 7) / 8);
  if (na + nb > 0x7fffffffll) return GECC_EINVAL;
  p.na = (int)na; p.nb = (int)nb;
  if (dtype == GECC_BF16) tl_encode_kernel<__nv_bfloat16><<<(unsigned)(na + nb), 256, 0, stream>>>(p);
  else tl_encode_kernel<float><<<(unsigned)(na + nb), 256, 0, stream>>>(p);
  return cudaGetLastError() == cudaSuccess ? GECC_OK : GECC_ECUDA;
}

// ---------------------------------------------------------------------------------------------------------------
// Decoder.  One CTA of 256 threads per block of C at a time (thread t < 128: row t of the block, else column t - 128).
// Fault-free blocks cost two loads per thread.  A flagged block is decided by thread 0 alone -- 128 + 128 lines in shared
// memory, the steps of PAPER.md:215-231 in order -- and patched by the CTA.
// ---------------------------------------------------------------------------------------------------------------
struct TlState {  // in the workspace; zero when first used, left zero by the last CTA
  unsigned int done, n_found, row_flags, col_flags, any_uncorrectable, any_corrected, pad_[2];
  unsigned long long maxabs[4];
  gecc_found_t found[GECC_TL_MAX_FOUND];
};

struct TlDecodeParams {
  int dtype, n, k, m, nrb, ncb;
  const float* rowpart;  // [ncb][n][4]: per row, per block of 128 columns: sum, local-weighted sum (0-based), sum of squares
  const float* colpart;  // [nrb][m][4]
  const float* PrL; int64_t ldprl;
  const float* PcL; int64_t ldpcl;
  float* C; int64_t ldc;
  ThresholdSpec ts;
  TlState* st;
  unsigned int* counters;
  gecc_tl_report_t* report;
};

struct TlPlan {
  int verdict, rows_short, nS, S[2], whole[2];
  int npts, pt_s[kMaxPoints], pt_l[kMaxPoints];
  double pt_x[kMaxPoints];
  int nf;
  gecc_found_t found[2 + kMaxPoints + 2];
};

struct TlShared {
  double syn[4][kTlPanel];  // r1, r2, q1, q2 of the block
  double thr[4][kTlPanel];  // thresholds of each line (tau scaled by the line's energy, as in fold.cuh)
  int list[2][kTlPanel];   // flagged rows / flagged columns of the block, ascending (compacted by the whole CTA)
  int nlist[2];
  int wcnt[8];             // flagged lines per warp (warps 0..3: rows, 4..7: columns)
  double tau_full[4];      // thresholds of a full 128 x 128 block
  int votes[kTlPanel];
  TlPlan plan;
};

// The decision for one block, by one thread (completions R5-R8, R21 of DESIGN.md; the noise hardening of the
// global decoder's decide(): a long-side line votes only if its plain syndrome stands out of both thresholds, the 2 x 2 solve's
// estimates are located against max(tau_1, 2 tau_2 / |w2 - w1|), two rows crossing two columns are settled by the diagonal test).
__device__ __noinline__ void tl_decide(TlShared& sh, int br, int bc) {
  TlPlan& P = sh.plan;
  P.verdict = GECC_UNCORRECTABLE; P.nS = 0; P.S[0] = P.S[1] = -1; P.whole[0] = P.whole[1] = 0; P.npts = 0; P.nf = 0;
  const int* R = sh.list[0]; const int* Q = sh.list[1];
  const int nR = sh.nlist[0], nQ = sh.nlist[1];
  if (nR == 0 && nQ == 0) { P.verdict = GECC_CLEAN; return; }
  if (nR >= 3 && nQ >= 3) return;  // min(s, t) >= 3: PAPER.md:219
  const bool rows_short = nR <= nQ;
  P.rows_short = rows_short ? 1 : 0;
  const int so = rows_short ? 0 : 2, lo = rows_short ? 2 : 0;  // offsets of the short / long side in syn[] and thr[]
  const double* s1 = sh.syn[so]; const double* s2 = sh.syn[so + 1];
  const double* l1 = sh.syn[lo]; const double* l2 = sh.syn[lo + 1];
  const double* ts1 = sh.thr[so]; const double* ts2 = sh.thr[so + 1];
  const double* tl1 = sh.thr[lo]; const double* tl2 = sh.thr[lo + 1];
  const int n_short = rows_short ? br : bc, n_long = rows_short ? bc : br;
  const int* SF = rows_short ? R : Q; const int nSF = rows_short ? nR : nQ;
  const int* LF = rows_short ? Q : R; const int nLF = rows_short ? nQ : nR;
  int nS = nSF, S[2] = {nSF > 0 ? SF[0] : -1, nSF > 1 ? SF[1] : -1};
  auto explained = [&](int j) { return nS == 2 || (nS == 1 && fabs(l2[j] - (double)(S[0] + 1) * l1[j]) <= tl2[j]); };
  int nU = 0;
  for (int e = 0; e < nLF; ++e) if (!explained(LF[e])) ++nU;
  if (nU > 0) {
    // input faults leave their own side's syndromes silent (reading R7): the line is located by the weighted ratio
    for (int i = 0; i < n_short; ++i) sh.votes[i] = 0;
    bool all_valid = true;
    int distinct = 0, cand[3] = {-1, -1, -1};
    for (int e = 0; e < nLF; ++e) {
      const int j = LF[e];
      if (explained(j)) continue;
      const double elig = tl1[j] > tl2[j] ? tl1[j] : tl2[j];
      if (!(fabs(l1[j]) > elig)) continue;  // too weak to vote (non-finite values fall through to the ratio test and fail it)
      const double ratio = rint(l2[j] / l1[j]);
      if (ratio >= 1.0 && ratio <= (double)n_short && fabs(l2[j] - ratio * l1[j]) <= tl2[j]) {
        const int c = (int)ratio - 1;
        if (sh.votes[c]++ == 0) { if (distinct < 3) cand[distinct] = c; ++distinct; }
      } else all_valid = false;
    }
    if (nS == 0) {
      if (!all_valid || distinct == 0 || distinct > 2) return;
      nS = distinct;
      S[0] = distinct == 2 ? min(cand[0], cand[1]) : cand[0];
      S[1] = distinct == 2 ? max(cand[0], cand[1]) : -1;
    } else {
      int best = -1, bv = 0;
      for (int i = 0; i < n_short; ++i)
        if (i != S[0] && sh.votes[i] > bv) { bv = sh.votes[i]; best = i; }  // mode, ties -> smallest index
      if (best < 0) return;
      const int a = S[0];
      S[0] = a < best ? a : best; S[1] = a < best ? best : a; nS = 2;
    }
    for (int e = 0; e < nLF; ++e) if (!explained(LF[e])) return;
  }
  if (nS == 0) return;
  const double w1 = (double)(S[0] + 1), w2 = (double)(S[1] + 1);
  auto xhat = [&](int idx, int j) -> double {  // PAPER.md:223 (|S| = 1), the solve of PAPER.md:227 with the sign of R8 (|S| = 2)
    if (nS == 1) return l1[j];
    const double x2 = (l2[j] - w1 * l1[j]) / (w2 - w1);
    return idx == 0 ? l1[j] - x2 : x2;
  };
  auto tau_loc = [&](int j) -> double {
    if (nS == 1) return tl1[j];
    const double amp = 2.0 * tl2[j] / fabs(w2 - w1);
    return amp > tl1[j] ? amp : tl1[j];
  };
  int hidden_n = 0, hidden_s[2], hidden_l[2];
  double hidden_x[2];
  bool decided = false;
  if (nS == 2 && nSF == 2 && nLF == 2) {
    const int a = S[0], b = S[1];
    auto diag_ok = [&](int ja, int jb) {  // the error of line a in long-side line ja, the error of line b in jb
      return fabs(s1[a] - l1[ja]) <= ts1[a] + tl1[ja] && fabs(s1[b] - l1[jb]) <= ts1[b] + tl1[jb] &&
             fabs(l2[ja] - (double)(a + 1) * l1[ja]) <= tl2[ja] && fabs(l2[jb] - (double)(b + 1) * l1[jb]) <= tl2[jb] &&
             fabs(s2[a] - (double)(ja + 1) * s1[a]) <= ts2[a] && fabs(s2[b] - (double)(jb + 1) * s1[b]) <= ts2[b];
    };
    const bool h1 = diag_ok(LF[0], LF[1]), h2 = diag_ok(LF[1], LF[0]);
    if (h1 != h2) {
      const int ja = h1 ? LF[0] : LF[1], jb = h1 ? LF[1] : LF[0];
      P.pt_s[0] = a; P.pt_l[0] = ja; P.pt_x[0] = l1[ja];
      P.pt_s[1] = b; P.pt_l[1] = jb; P.pt_x[1] = l1[jb];
      P.npts = 2;
      decided = true;
    } else if (h1 && h2) return;
  }
  for (int idx = 0; idx < nS && !decided; ++idx) {
    const int sl = S[idx];
    const bool in_flag = (nSF > 0 && sl == SF[0]) || (nSF > 1 && sl == SF[1]);
    int g[kMaxPointsPerLine], ncols = 0;
    for (int e = 0; e < nLF; ++e) {  // reading R5: located only where the estimate stands out
      const int j = LF[e];
      if (fabs(xhat(idx, j)) > tau_loc(j)) { if (ncols < kMaxPointsPerLine) g[ncols] = j; ++ncols; }
    }
    int hidden_at = -1;
    if (in_flag && ncols >= 3) {  // a single error explaining the line's OWN two syndromes
      const double v1 = s1[sl], v2 = s2[sl];
      if (fabs(v1) > ts1[sl]) {
        const double ratio = rint(v2 / v1);
        if (ratio >= 1.0 && ratio <= (double)n_long && fabs(v2 - ratio * v1) <= ts2[sl]) hidden_at = (int)ratio - 1;
      }
    }
    if (!in_flag) P.whole[idx] = 1;  // located by the ratio only: an input fault, corrected along the line (R6)
    else if (ncols >= 3 && hidden_at >= 0) {
      P.whole[idx] = 1;
      hidden_s[hidden_n] = sl; hidden_l[hidden_n] = hidden_at; hidden_x[hidden_n] = s1[sl]; ++hidden_n;
    } else if (ncols > kMaxPointsPerLine) P.whole[idx] = 1;  // E(s, t), t large (Theorem 2; reading R21)
    else if (ncols == 0) return;                              // flagged line, nothing locatable (R11)
    else {
      for (int a = 0; a < ncols && P.npts < kMaxPoints; ++a) {
        const int j = g[a];
        double x = xhat(idx, j);
        if (nS == 2 && !(fabs(xhat(1 - idx, j)) > tau_loc(j))) x = l1[j];  // the other line is clean here: plain syndrome
        P.pt_s[P.npts] = sl; P.pt_l[P.npts] = j; P.pt_x[P.npts] = x; ++P.npts;
      }
    }
  }
  if (nS == 2 && P.whole[0] != P.whole[1]) {  // one whole line and a single point in the other: the point's own plain syndrome is its value
    const int pl = P.whole[0] ? 1 : 0;
    int cntp = 0, which = -1;
    for (int a = 0; a < P.npts; ++a)
      if (P.pt_s[a] == S[pl]) { ++cntp; which = a; }
    if (cntp == 1 && fabs(s1[S[pl]]) > ts1[S[pl]]) P.pt_x[which] = s1[S[pl]];
  }
  P.verdict = GECC_CORRECTED;
  P.nS = nS; P.S[0] = S[0]; P.S[1] = S[1];
  int nf = 0;
  for (int a = 0; a < nS; ++a)
    if (P.whole[a]) P.found[nf++] = rows_short ? gecc_found_t{GECC_KIND_ROW, S[a], -1, 0, 0.0} : gecc_found_t{GECC_KIND_COL, -1, S[a], 0, 0.0};
  for (int a = 0; a < P.npts; ++a)
    P.found[nf++] = rows_short ? gecc_found_t{GECC_KIND_C, P.pt_s[a], P.pt_l[a], 0, P.pt_x[a]} : gecc_found_t{GECC_KIND_C, P.pt_l[a], P.pt_s[a], 0, P.pt_x[a]};
  for (int a = 0; a < hidden_n; ++a) {
    const gecc_found_t f = rows_short ? gecc_found_t{GECC_KIND_C, hidden_s[a], hidden_l[a], 0, hidden_x[a]} : gecc_found_t{GECC_KIND_C, hidden_l[a], hidden_s[a], 0, hidden_x[a]};
    bool dup = false;  // the oracle's list is a set
    for (int b = 0; b < nf; ++b) dup = dup || (P.found[b].kind == f.kind && P.found[b].row == f.row && P.found[b].col == f.col);
    if (!dup) P.found[nf++] = f;
  }
  P.nf = nf;
}

__device__ __forceinline__ bool tl_found_less(const gecc_found_t& a, const gecc_found_t& b) {
  if (a.kind != b.kind) return a.kind < b.kind;
  if (a.row != b.row) return a.row < b.row;
  return a.col < b.col;
}

__global__ void __launch_bounds__(256) tl_decode_kernel(const __grid_constant__ TlDecodeParams p) {
  __shared__ TlShared sh;
  __shared__ unsigned long long shmax[4];
  __shared__ int shcnt[2];
  const int tid = threadIdx.x;
  const bool is_row = tid < kTlPanel;
  const int line = tid & (kTlPanel - 1);
  ptx::griddep_wait();  // launched as a programmatic dependent of the product
  if (blockIdx.x == 0 && tid == 0) ws_enter(p.counters, "gecc_tl_decode");
  if (tid < 4) shmax[tid] = 0ull;
  if (tid < 2) shcnt[tid] = 0;
  // thresholds of a full block and the operand statistics (fold.cuh: the formula of include/gecc.h with n, m -> 128), once per CTA:
  // double-precision square roots and divisions are long instruction sequences
  __shared__ double sh_stat[2];  // base = kappa c(k) 2^-24 sigma_a sigma_b; sigma_c2 = k sigma_a^2 sigma_b^2
  if (tid == 0) {
    double sa = 0.0, sb = 0.0;
    if (p.ts.sumsq_a) sa = sqrt(__ldcg(p.ts.sumsq_a) / ((double)p.n * p.k));
    if (p.ts.sumsq_b) sb = sqrt(__ldcg(p.ts.sumsq_b) / ((double)p.k * p.m));
    sh_stat[0] = kKappa * p.ts.noise_c * 5.9604644775390625e-08 * sa * sb;
    sh_stat[1] = (double)p.k * sa * sa * sb * sb;
  }
  __syncthreads();
  const double base = sh_stat[0], sigma_c2 = sh_stat[1];
  auto block_tau = [&](int br, int bc, double (&tau)[4]) {
    if (p.ts.have_tau) { for (int q = 0; q < 4; ++q) tau[q] = p.ts.tau[q]; return; }
    tau[0] = base * sqrt((double)p.k * bc);
    tau[2] = base * sqrt((double)p.k * br);
    tau[1] = tau[0] * sqrt((bc + 1.0) * (2.0 * bc + 1.0) / 6.0);
    tau[3] = tau[2] * sqrt((br + 1.0) * (2.0 * br + 1.0) / 6.0);
  };
  unsigned long long mx1 = 0ull, mx2 = 0ull;
  int my_flags = 0;
  __shared__ float sh_inv_c2;
  if (tid == 0) {
    double t4[4];
    block_tau(kTlPanel, kTlPanel, t4);
    for (int q = 0; q < 4; ++q) sh.tau_full[q] = t4[q];
    sh_inv_c2 = sigma_c2 > 0.0 ? (float)(1.0 / sigma_c2) : 0.f;
  }
  __syncthreads();
  const float inv_c2 = sh_inv_c2;
  const int nblocks = p.nrb * p.ncb;
  // the line's sums (left by the product's epilogue) and its parity limbs for block b; the next block's loads are in flight
  // while this one is worked on
  auto fetch = [&](int b, float4& part, float (&pv)[6]) {
    part = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int u = 0; u < 6; ++u) pv[u] = 0.f;
    if (b >= nblocks) return;
    const int rb = b / p.ncb, cb = b - rb * p.ncb;
    const int br = min(kTlPanel, p.n - rb * kTlPanel), bc = min(kTlPanel, p.m - cb * kTlPanel);
    if (line >= (is_row ? br : bc)) return;
    if (is_row) {
      const int64_t gi = (int64_t)rb * kTlPanel + line;
      part = __ldcg(reinterpret_cast<const float4*>(p.rowpart + ((int64_t)cb * p.n + gi) * 4));
      const float4 lo4 = __ldcg(reinterpret_cast<const float4*>(p.PrL + gi * p.ldprl + cb * kTlRows));
      const float4 hi4 = __ldcg(reinterpret_cast<const float4*>(p.PrL + gi * p.ldprl + cb * kTlRows + 4));
      pv[0] = lo4.x; pv[1] = lo4.y; pv[2] = lo4.z; pv[3] = lo4.w; pv[4] = hi4.x; pv[5] = hi4.y;
    } else {
      const int64_t gj = (int64_t)cb * kTlPanel + line;
      part = __ldcg(reinterpret_cast<const float4*>(p.colpart + ((int64_t)rb * p.m + gj) * 4));
#pragma unroll
      for (int u = 0; u < 6; ++u) pv[u] = __ldcg(p.PcL + ((int64_t)rb * kTlRows + u) * p.ldpcl + gj);
    }
  };
  float4 part_n;
  float pv_n[6];
  fetch(blockIdx.x, part_n, pv_n);
  for (int b = blockIdx.x; b < nblocks; b += gridDim.x) {
    const int rb = b / p.ncb, cb = b - rb * p.ncb;
    const int br = min(kTlPanel, p.n - rb * kTlPanel), bc = min(kTlPanel, p.m - cb * kTlPanel);
    double tau[4];
    if (br == kTlPanel && bc == kTlPanel) { for (int q = 0; q < 4; ++q) tau[q] = sh.tau_full[q]; }
    else block_tau(br, bc, tau);  // ragged edge blocks: shorter lines, smaller thresholds
    const bool live = line < (is_row ? br : bc);
    bool flagged = false;
    double a = 0.0, bw = 0.0, t1 = 0.0, t2 = 0.0;
    const float4 part = part_n;
    float pv[6];
#pragma unroll
    for (int u = 0; u < 6; ++u) pv[u] = pv_n[u];
    fetch(b + (int)gridDim.x, part_n, pv_n);
    if (live) {
      double p1, p2;
      if (p.dtype == GECC_BF16) { p1 = (double)pv[0] + (double)pv[1] + (double)pv[2]; p2 = (double)pv[3] + (double)pv[4] + (double)pv[5]; }
      else { p1 = (double)pv[0]; p2 = (double)pv[3]; }
      a = (double)part.x - p1;                        // sum minus parity
      bw = ((double)part.y + (double)part.x) - p2;    // the epilogue's weights are 0-based within the block; the code's are 1-based
      const float len = is_row ? (float)bc : (float)br;
      float fe = sqrtf(part.z * inv_c2 / len);  // line energy over its expectation (fold.cuh's rule); NaN-safe: stays 1
      fe = fe > 1.f ? fe : 1.f;
      t1 = tau[is_row ? 0 : 2] * (double)fe; t2 = tau[is_row ? 1 : 3] * (double)fe;
      flagged = !(fabs(a) <= t1) || (!p.ts.single && !(fabs(bw) <= t2));
      const unsigned long long v1 = (unsigned long long)__double_as_longlong(abs_for_max(a)), v2 = (unsigned long long)__double_as_longlong(abs_for_max(bw));
      mx1 = v1 > mx1 ? v1 : mx1;
      mx2 = v2 > mx2 ? v2 : mx2;
    }
    const int so = is_row ? 0 : 2;
    sh.syn[so][line] = a; sh.syn[so + 1][line] = bw;
    sh.thr[so][line] = t1; sh.thr[so + 1][line] = t2;
    my_flags += flagged ? 1 : 0;
    const int nflag = __syncthreads_count(flagged);
    if (nflag == 0) continue;  // PAPER.md:215 with both sets empty: the block is clean
    {  // the two flag sets as ascending lists, compacted by the CTA
      const unsigned bal = __ballot_sync(0xffffffffu, flagged);
      const int w = tid >> 5, ln = tid & 31;
      if (ln == 0) sh.wcnt[w] = __popc(bal);
      __syncthreads();
      int base = 0;
      for (int u = w & 4; u < w; ++u) base += sh.wcnt[u];
      if (flagged) sh.list[w >> 2][base + __popc(bal & ((1u << ln) - 1u))] = line;
      if (tid < 2) sh.nlist[tid] = sh.wcnt[4 * tid] + sh.wcnt[4 * tid + 1] + sh.wcnt[4 * tid + 2] + sh.wcnt[4 * tid + 3];
      __syncthreads();
    }
    if (tid == 0) tl_decide(sh, br, bc);
    __syncthreads();
    const TlPlan& P = sh.plan;
    if (P.verdict == GECC_CORRECTED) {
      const bool rows_short = P.rows_short != 0;
      const int lo = rows_short ? 2 : 0;
      const int n_long = rows_short ? bc : br;
      const int64_t i0 = (int64_t)rb * kTlPanel, j0 = (int64_t)cb * kTlPanel;
      const double w1 = (double)(P.S[0] + 1), w2 = (double)(P.S[1] + 1);
      // c_true = c - e: whole lines along the line (R6), points where located (R5)
      if ((P.whole[0] || P.whole[1]) && tid < n_long) {
        const int g = tid;
        for (int idx = 0; idx < P.nS; ++idx) {
          if (!P.whole[idx]) continue;
          const int sl = P.S[idx];
          double x;
          if (P.nS == 1) x = sh.syn[lo][g];
          else if ((P.whole[0] != 0) != (P.whole[1] != 0)) {  // the other line holds located points only: the rest of the plain syndrome is this line's
            x = sh.syn[lo][g];
            for (int q = 0; q < P.npts; ++q)
              if (P.pt_l[q] == g && P.pt_s[q] != sl) x -= P.pt_x[q];
          } else { const double y1 = sh.syn[lo][g], x2 = (sh.syn[lo + 1][g] - w1 * y1) / (w2 - w1); x = idx == 0 ? y1 - x2 : x2; }
          const int64_t off = rows_short ? (i0 + sl) * p.ldc + j0 + g : (i0 + g) * p.ldc + j0 + sl;
          p.C[off] = (float)((double)__ldcg(p.C + off) - x);
        }
      }
      if (tid < P.npts) {
        const int sl = P.pt_s[tid], ll = P.pt_l[tid];
        const bool in_whole = (P.whole[0] && P.S[0] == sl) || (P.whole[1] && P.nS > 1 && P.S[1] == sl);
        if (!in_whole) {
          const int64_t off = rows_short ? (i0 + sl) * p.ldc + j0 + ll : (i0 + ll) * p.ldc + j0 + sl;
          p.C[off] = (float)((double)__ldcg(p.C + off) - P.pt_x[tid]);
        }
      }
      if (tid == 0) {
        atomicExch(&p.st->any_corrected, 1u);
        const unsigned int slot = atomicAdd(&p.st->n_found, (unsigned int)P.nf);
        for (int q = 0; q < P.nf; ++q)
          if (slot + q < GECC_TL_MAX_FOUND) {
            gecc_found_t f = P.found[q];
            if (f.row >= 0) f.row += (int)i0;
            if (f.col >= 0) f.col += (int)j0;
            p.st->found[slot + q] = f;
          }
      }
    } else if (tid == 0) atomicExch(&p.st->any_uncorrectable, 1u);
    __syncthreads();
  }
  // totals of this CTA, then the report by the last CTA to finish
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long u1 = __shfl_xor_sync(0xffffffffu, mx1, o), u2 = __shfl_xor_sync(0xffffffffu, mx2, o);
    mx1 = u1 > mx1 ? u1 : mx1;
    mx2 = u2 > mx2 ? u2 : mx2;
    my_flags += __shfl_xor_sync(0xffffffffu, my_flags, o);
  }
  if ((tid & 31) == 0) {
    if (mx1) atomicMax(&shmax[is_row ? 0 : 2], mx1);
    if (mx2) atomicMax(&shmax[is_row ? 1 : 3], mx2);
    if (my_flags) atomicAdd(&shcnt[is_row ? 0 : 1], my_flags);
  }
  __syncthreads();
  __shared__ int sh_last;
  TlState* st = p.st;
  if (tid == 0) {
    for (int q = 0; q < 4; ++q) if (shmax[q]) atomicMax(&st->maxabs[q], shmax[q]);  // results unused: reductions, no round trip
    if (shcnt[0]) atomicAdd(&st->row_flags, (unsigned int)shcnt[0]);
    if (shcnt[1]) atomicAdd(&st->col_flags, (unsigned int)shcnt[1]);
    __threadfence();
    sh_last = atomicAdd(&st->done, 1u) == gridDim.x - 1u ? 1 : 0;
  }
  __syncthreads();
  if (sh_last) {  // the last CTA to finish: every block of C is settled; the report, by the whole CTA
    __threadfence();
    gecc_tl_report_t* r = p.report;
    const unsigned int nf = __ldcg(&st->n_found);
    const int listed = nf < (unsigned int)GECC_TL_MAX_FOUND ? (int)nf : GECC_TL_MAX_FOUND;
    if (tid < GECC_TL_MAX_FOUND) {  // rank sort by (kind, row, col); equal entries (a whole line listed once per block) keep their slot order
      gecc_found_t f = gecc_found_t{-1, -1, -1, 0, 0.0};
      int rank = tid;
      if (tid < listed) {
        const gecc_found_t* g = &st->found[tid];
        f = gecc_found_t{__ldcg(&g->kind), __ldcg(&g->row), __ldcg(&g->col), 0, __ldcg(&g->magnitude)};
        rank = 0;
        for (int o = 0; o < listed; ++o) {
          const gecc_found_t* h = &st->found[o];
          const gecc_found_t e = gecc_found_t{__ldcg(&h->kind), __ldcg(&h->row), __ldcg(&h->col), 0, 0.0};
          if (tl_found_less(e, f) || (!tl_found_less(f, e) && o < tid)) ++rank;
        }
      }
      r->found[rank] = f;
    }
    if (tid == 0) {
      const bool unc = __ldcg(&st->any_uncorrectable) != 0, cor = __ldcg(&st->any_corrected) != 0;
      r->verdict = unc ? GECC_UNCORRECTABLE : (cor ? GECC_CORRECTED : GECC_CLEAN);
      r->n_found = (int)nf;
      r->n_row_flags = (int)__ldcg(&st->row_flags);
      r->n_col_flags = (int)__ldcg(&st->col_flags);
      double tau[4];
      block_tau(min(kTlPanel, p.n), min(kTlPanel, p.m), tau);
      for (int q = 0; q < 4; ++q) {
        r->max_abs_syndrome[q] = __longlong_as_double((long long)__ldcg(&st->maxabs[q]));
        r->tau[q] = tau[q];
      }
    }
    __syncthreads();
    if (tid == 0) {
      for (int q = 0; q < 4; ++q) st->maxabs[q] = 0ull;
      st->done = 0; st->n_found = 0; st->row_flags = 0; st->col_flags = 0; st->any_uncorrectable = 0; st->any_corrected = 0;
      __threadfence();
    }
  }
  if (tid == 0) ws_exit(p.counters, gridDim.x);
}

int tl_decode_dispatch(int dtype, int64_t n, int64_t k, int64_t m, float* C, int64_t ldc, const float* PrL, int64_t ldprl, const float* PcL, int64_t ldpcl,
                       const double* tau, const double* sumsq_a, const double* sumsq_b, int mode, gecc_tl_report_t* report, uint8_t* ws, const WsLayout& L,
                       cudaStream_t stream) {
  static_assert(sizeof(TlState) <= sizeof(BlockStat) * kMaxDecodeBlocks, "TlState lives in the blockstat region of the workspace");
  TlDecodeParams p;
  p.dtype = dtype; p.n = (int)n; p.k = (int)k; p.m = (int)m;
  p.nrb = (int)((n + kTlPanel - 1) / kTlPanel); p.ncb = (int)((m + kTlPanel - 1) / kTlPanel);
  p.rowpart = reinterpret_cast<const float*>(ws + L.rowpart); p.colpart = reinterpret_cast<const float*>(ws + L.colpart);
  p.PrL = PrL; p.ldprl = ldprl; p.PcL = PcL; p.ldpcl = ldpcl;
  p.C = C; p.ldc = ldc;
  p.ts.have_tau = tau ? 1 : 0;
  for (int q = 0; q < 4; ++q) p.ts.tau[q] = tau ? tau[q] : 0.0;
  p.ts.sumsq_a = sumsq_a; p.ts.sumsq_b = sumsq_b; p.ts.noise_c = noise_coeff(dtype, (double)k); p.ts.single = (mode & GECC_SINGLE_CHECKSUM) ? 1 : 0;
  p.st = reinterpret_cast<TlState*>(ws + L.blockstat);
  p.counters = reinterpret_cast<unsigned int*>(ws);
  p.report = report;
  const int sms = num_sms();
  if (sms <= 0) return GECC_ECUDA;
  const int64_t nblocks = (int64_t)p.nrb * p.ncb;
  int per_sm = 0;  // one wave of resident CTAs, each looping over its share of the blocks of C
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, tl_decode_kernel, 256, 0) != cudaSuccess || per_sm < 1) per_sm = 1;
  const int64_t cap = (int64_t)per_sm * sms;
  const int grid = (int)(nblocks < cap ? nblocks : cap);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3(256);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (cudaLaunchKernelEx(&cfg, tl_decode_kernel, p) != cudaSuccess) return GECC_ECUDA;
  return GECC_OK;
}

}  // namespace gecc
