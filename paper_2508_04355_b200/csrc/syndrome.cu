// Detection step: the four syndromes per row / column from the per-tile partial sums and the
// parity symbols the product emitted, thresholds, flag sets E_r / E_t.  Plus the standalone (unfused) pass over a
// stored C that produces the same partials, and the input-fault injection hook.
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "gecc_internal.h"

namespace gecc {

// Automatic thresholds (reading R4; the paper gives one delta without dtype or data scale).
// tau_plain = kappa c(k) 2^-24 sqrt(k m) sigma_a sigma_b (noise_coeff in gecc_internal.h); the weighted syndromes scale
// with the RMS weight.  sigma_c2 = k sigma_a^2 sigma_b^2 is the expected energy of one symbol of C: a line whose measured
// energy exceeds it gets a proportionally larger threshold (rounding noise is relative to what was summed).
__global__ void decode_init_kernel(DecodeState* st, int dtype, int64_t n, int64_t k, int64_t m, bool have_tau, double t0, double t1, double t2,
                                   double t3, const double* sumsq_a, const double* sumsq_b) {
  DecodeState z = {};
  double sa = 0.0, sb = 0.0;
  if (sumsq_a) sa = sqrt(*sumsq_a / ((double)n * (double)k));
  if (sumsq_b) sb = sqrt(*sumsq_b / ((double)k * (double)m));
  z.sigma_a = sa;
  z.sigma_b = sb;
  z.sigma_c2 = (double)k * sa * sa * sb * sb;
  if (have_tau) {
    z.tau[0] = t0; z.tau[1] = t1; z.tau[2] = t2; z.tau[3] = t3;
  } else {
    const double base = kKappa * noise_coeff(dtype, (double)k) * 5.9604644775390625e-08 * sa * sb;
    z.tau[0] = base * sqrt((double)k * (double)m);
    z.tau[2] = base * sqrt((double)k * (double)n);
    z.tau[1] = z.tau[0] * sqrt((double)(m + 1) * (double)(2 * m + 1) / 6.0);
    z.tau[3] = z.tau[2] * sqrt((double)(n + 1) * (double)(2 * n + 1) / 6.0);
  }
  *st = z;
}

__device__ __forceinline__ unsigned long long abs_bits(double x) { return (unsigned long long)__double_as_longlong(fabs(x)); }
__device__ __forceinline__ unsigned long long warp_max(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long w = __shfl_xor_sync(0xffffffffu, v, o);
    v = w > v ? w : v;
  }
  return v;
}

// One thread per row (g < n) or column (g - n < m).  Sum minus parity, global weights restored from
// the block-local ones: weight of 0-based index x is x + 1.
__global__ void __launch_bounds__(256) syndrome_kernel(int dtype, int n, int m, int nb, int slabs, const float* __restrict__ rowpart,
                                                        const float* __restrict__ colpart, const float* __restrict__ P_r,
                                                        const float* __restrict__ P_c, double* __restrict__ syn, uint8_t* __restrict__ flags,
                                                        DecodeState* st) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  const int bn = block_n(dtype);
  double a = 0.0, b = 0.0, en = 0.0;
  unsigned long long mx[4] = {0, 0, 0, 0};
  double* tolx = syn + 2 * ((int64_t)n + m);  // extra tolerance per line, same order as syn
  const double ec2 = st->sigma_c2;
  if (g < n) {
    for (int t = 0; t < nb; ++t) {
      const float4 p = *reinterpret_cast<const float4*>(rowpart + ((int64_t)t * n + g) * 4);
      a += (double)p.x;
      b += (double)(t * bn + 1) * (double)p.x + (double)p.y;
      en += (double)p.z;
    }
    const float* pr = P_r + (int64_t)g * GECC_PR_LD;
    double p1, p2;
    if (dtype == GECC_BF16) { p1 = (double)pr[0] + (double)pr[1] + (double)pr[2]; p2 = (double)pr[3] + (double)pr[4] + (double)pr[5]; }
    else { p1 = (double)pr[0]; p2 = (double)pr[3]; }
    a -= p1; b -= p2;
    double f = ec2 > 0.0 ? sqrt(en / ((double)m * ec2)) : 1.0;
    f = f > 1.0 ? f : 1.0;  // NaN-safe: a non-finite energy leaves f = 1 and the non-finite syndrome flags the line
    const double x1 = st->tau[0] * (f - 1.0), x2 = st->tau[1] * (f - 1.0);
    syn[g] = a;
    syn[n + g] = b;
    tolx[g] = x1;
    tolx[n + g] = x2;
    const bool fl = !(fabs(a) <= st->tau[0] + x1) || !(fabs(b) <= st->tau[1] + x2);
    flags[g] = fl;
    if (fl) atomicAdd(&st->n_row_flags, 1);
    mx[0] = abs_bits(a); mx[1] = abs_bits(b);
  } else if (g - n < m) {
    const int j = g - n;
    for (int s = 0; s < slabs; ++s) {
      const float4 p = *reinterpret_cast<const float4*>(colpart + ((int64_t)s * m + j) * 4);
      a += (double)p.x;
      b += (double)(s * kRowSlab + 1) * (double)p.x + (double)p.y;
      en += (double)p.z;
    }
    double p1, p2;
    if (dtype == GECC_BF16) {
      p1 = (double)P_c[j] + (double)P_c[m + j] + (double)P_c[2 * (int64_t)m + j];
      p2 = (double)P_c[3 * (int64_t)m + j] + (double)P_c[4 * (int64_t)m + j] + (double)P_c[5 * (int64_t)m + j];
    } else { p1 = (double)P_c[j]; p2 = (double)P_c[3 * (int64_t)m + j]; }
    a -= p1; b -= p2;
    double f = ec2 > 0.0 ? sqrt(en / ((double)n * ec2)) : 1.0;
    f = f > 1.0 ? f : 1.0;
    const double x1 = st->tau[2] * (f - 1.0), x2 = st->tau[3] * (f - 1.0);
    syn[2 * (int64_t)n + j] = a;
    syn[2 * (int64_t)n + m + j] = b;
    tolx[2 * (int64_t)n + j] = x1;
    tolx[2 * (int64_t)n + m + j] = x2;
    const bool fl = !(fabs(a) <= st->tau[2] + x1) || !(fabs(b) <= st->tau[3] + x2);
    flags[n + j] = fl;
    if (fl) atomicAdd(&st->n_col_flags, 1);
    mx[2] = abs_bits(a); mx[3] = abs_bits(b);
  }
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const unsigned long long w = warp_max(mx[q]);
    if ((threadIdx.x & 31) == 0 && w) atomicMax(&st->maxabs_bits[q], w);
  }
}

// Unfused detection sums over a stored C: one block per (32-row slab, block column); the same partial layout the
// GEMM epilogue writes.  Reads C once with 16-byte loads.
template <int BN>
__global__ void __launch_bounds__(256) syndrome_unfused_kernel(int n, int m, const float* __restrict__ C, int64_t ldc, float* __restrict__ rowpart,
                                                                float* __restrict__ colpart) {
  constexpr int NV = BN / 128;  // float4 per lane per row
  __shared__ float colacc[8][BN][3];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int nbk = blockIdx.x, slab = blockIdx.y;
  float cs1[NV][4], cs2[NV][4], css[NV][4];
#pragma unroll
  for (int h = 0; h < NV; ++h)
#pragma unroll
    for (int e = 0; e < 4; ++e) { cs1[h][e] = 0.f; cs2[h][e] = 0.f; css[h][e] = 0.f; }
#pragma unroll
  for (int rr = 0; rr < 4; ++rr) {
    const int il = 4 * w + rr;  // row within the slab
    const int64_t row = (int64_t)slab * kRowSlab + il;
    float s1 = 0.f, s2 = 0.f, ss = 0.f;
#pragma unroll
    for (int h = 0; h < NV; ++h) {
      const int jl = 128 * h + 4 * lane;  // column within the block column
      const int64_t col = (int64_t)nbk * BN + jl;
      float4 x = make_float4(0.f, 0.f, 0.f, 0.f);
      if (row < n && col < m) x = __ldg(reinterpret_cast<const float4*>(C + row * ldc + col));
      s1 += (x.x + x.y) + (x.z + x.w);
      ss += (x.x * x.x + x.y * x.y) + (x.z * x.z + x.w * x.w);
      s2 = fmaf((float)jl, x.x, s2); s2 = fmaf((float)(jl + 1), x.y, s2); s2 = fmaf((float)(jl + 2), x.z, s2); s2 = fmaf((float)(jl + 3), x.w, s2);
      const float wt = (float)il;
      cs1[h][0] += x.x; cs1[h][1] += x.y; cs1[h][2] += x.z; cs1[h][3] += x.w;
      cs2[h][0] = fmaf(wt, x.x, cs2[h][0]); cs2[h][1] = fmaf(wt, x.y, cs2[h][1]); cs2[h][2] = fmaf(wt, x.z, cs2[h][2]); cs2[h][3] = fmaf(wt, x.w, cs2[h][3]);
      css[h][0] = fmaf(x.x, x.x, css[h][0]); css[h][1] = fmaf(x.y, x.y, css[h][1]); css[h][2] = fmaf(x.z, x.z, css[h][2]); css[h][3] = fmaf(x.w, x.w, css[h][3]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { s1 += __shfl_xor_sync(0xffffffffu, s1, o); s2 += __shfl_xor_sync(0xffffffffu, s2, o); ss += __shfl_xor_sync(0xffffffffu, ss, o); }
    if (lane == 0 && row < n) *reinterpret_cast<float4*>(rowpart + ((int64_t)nbk * n + row) * 4) = make_float4(s1, s2, ss, 0.f);
  }
#pragma unroll
  for (int h = 0; h < NV; ++h)
#pragma unroll
    for (int e = 0; e < 4; ++e) { colacc[w][128 * h + 4 * lane + e][0] = cs1[h][e]; colacc[w][128 * h + 4 * lane + e][1] = cs2[h][e]; colacc[w][128 * h + 4 * lane + e][2] = css[h][e]; }
  __syncthreads();
  for (int c = threadIdx.x; c < BN; c += 256) {
    const int64_t col = (int64_t)nbk * BN + c;
    if (col >= m) continue;
    float a = 0.f, b = 0.f, e2 = 0.f;
#pragma unroll
    for (int g = 0; g < 8; ++g) { a += colacc[g][c][0]; b += colacc[g][c][1]; e2 += colacc[g][c][2]; }
    *reinterpret_cast<float4*>(colpart + ((int64_t)slab * m + col) * 4) = make_float4(a, b, e2, 0.f);
  }
}

int syndrome_unfused_dispatch(int dtype, int64_t n, int64_t m, const float* C, int64_t ldc, float* rowpart, float* colpart, cudaStream_t stream) {
  const int bn = block_n(dtype);
  dim3 grid((unsigned)((m + bn - 1) / bn), (unsigned)(((n + 127) / 128) * 4));
  if (bn == 256) syndrome_unfused_kernel<256><<<grid, 256, 0, stream>>>((int)n, (int)m, C, ldc, rowpart, colpart);
  else syndrome_unfused_kernel<128><<<grid, 256, 0, stream>>>((int)n, (int)m, C, ldc, rowpart, colpart);
  return cudaGetLastError() == cudaSuccess ? GECC_OK : GECC_ECUDA;
}

// E1 / E2: additive fault on a stored symbol of A or B, as the operand dtype stores it.
__global__ void inject_inputs_kernel(int dtype, void* A, int64_t lda, float* A_lo, void* B, int64_t ldb, float* B_lo, const gecc_fault_t* faults,
                                     int n_faults) {
  const int f = threadIdx.x;
  if (f >= n_faults) return;
  const gecc_fault_t ft = faults[f];
  if (ft.kind != GECC_KIND_A && ft.kind != GECC_KIND_B) return;
  void* X = ft.kind == GECC_KIND_A ? A : B;
  float* X_lo = ft.kind == GECC_KIND_A ? A_lo : B_lo;
  const int64_t idx = (int64_t)ft.row * (ft.kind == GECC_KIND_A ? lda : ldb) + ft.col;
  if (dtype == GECC_BF16) {
    __nv_bfloat16* p = reinterpret_cast<__nv_bfloat16*>(X) + idx;
    *p = __float2bfloat16_rn(__bfloat162float(*p) + ft.value);
  } else {
    float* p = reinterpret_cast<float*>(X) + idx;
    const float v = *p + ft.value;
    *p = v;
    if (X_lo) X_lo[idx] = v - __uint_as_float(__float_as_uint(v) & 0xFFFFE000u);
  }
}

}  // namespace gecc
