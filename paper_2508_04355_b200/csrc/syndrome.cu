// The standalone (unfused) pass over a stored C that produces the same partial sums of the detection step
// as the protected product's epilogue, and the input-fault injection hook.
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "encode_core.cuh"
#include "gecc_internal.h"

namespace gecc {

// One block per kSumRows x kSumCols tile of C (64 KB), read once with 16-byte loads: warp w owns rows 16 w .. 16 w + 15,
// lane l owns columns 4 l .. 4 l + 3; the tile is taken in two halves of 8 rows per warp, the second half's loads in
// flight while the first is reduced.  The pass is HBM-bound only if it stays light on instructions: the per-vector sums
// use packed fp32 pairs (FADD2 / FFMA2), and a row's 32 lane partials are summed through shared memory (one 16-byte store
// per vector, rotated by the row so that both the stores and the reads are conflict-free) instead of 15 shuffles per row.
// Column sums go across the warps through shared memory.
// Partial layout (gecc_internal.h): rowpart[cb][n][4], colpart[rb][m][4] = (sum, local-weighted sum, sum of squares, 0).
__global__ void __launch_bounds__(256, 3) syndrome_unfused_kernel(int n, int m, const float* __restrict__ C, int64_t ldc, float* __restrict__ rowpart,
                                                                   float* __restrict__ colpart) {
  static_assert(kSumRows == 128 && kSumCols == 128, "tile shape of the unfused pass");
  __shared__ float4 rowacc[64][32];  // [row of the half][lane rotated by the row]: (sum, weighted sum, squares, -)
  __shared__ float colacc[8][kSumCols][3];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int cb = blockIdx.x, rb = blockIdx.y;
  const int jl = 4 * lane;
  const int64_t col = (int64_t)cb * kSumCols + jl;
  const f32x2 wj01 = pack2((float)jl, (float)(jl + 1)), wj23 = pack2((float)(jl + 2), (float)(jl + 3));
  f32x2 cs1[2] = {0ull, 0ull}, cs2[2] = {0ull, 0ull}, css[2] = {0ull, 0ull};
  float4 x[8];
  // whole tile inside C (the usual case): one base pointer and a row stride, no per-load checks
  const bool full = (int64_t)(rb + 1) * kSumRows <= n && (int64_t)(cb + 1) * kSumCols <= m;
  const float* base = C + ((int64_t)rb * kSumRows + 16 * w) * ldc + col;
  const uint32_t ldb = (uint32_t)(ldc * 4);  // bytes per row (host checks the range)
  auto load_half = [&](int half) {
    if (full) {
#pragma unroll
      for (int u = 0; u < 8; ++u)
        x[u] = __ldcs(reinterpret_cast<const float4*>(reinterpret_cast<const char*>(base) + (uint64_t)ldb * (uint32_t)(8 * half + u)));
    } else {
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int64_t row = (int64_t)rb * kSumRows + 16 * w + 8 * half + u;
        x[u] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (row < n && col < m) x[u] = __ldcs(reinterpret_cast<const float4*>(C + row * ldc + col));
      }
    }
  };
  load_half(0);
#pragma unroll
  for (int half = 0; half < 2; ++half) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int il = 16 * w + 8 * half + u;  // row within the tile
      const int hl = 8 * w + u;              // row within the half
      const f32x2 p01 = pack2(x[u].x, x[u].y), p23 = pack2(x[u].z, x[u].w);
      const f32x2 q01 = mul2(p01, p01), q23 = mul2(p23, p23);
      const f32x2 wt = pack2((float)il, (float)il);
      cs1[0] = add2(cs1[0], p01); cs1[1] = add2(cs1[1], p23);
      cs2[0] = fma2(wt, p01, cs2[0]); cs2[1] = fma2(wt, p23, cs2[1]);
      css[0] = add2(css[0], q01); css[1] = add2(css[1], q23);
      float a0, a1, b0, b1, c0, c1;
      unpack2(add2(p01, p23), a0, a1);
      unpack2(fma2(wj01, p01, mul2(wj23, p23)), b0, b1);
      unpack2(add2(q01, q23), c0, c1);
      rowacc[hl][(lane + hl) & 31] = make_float4(a0 + a1, b0 + b1, c0 + c1, 0.f);
    }
    if (half == 0) load_half(1);  // in flight during the reduction below
    __syncthreads();
    {
      const int t = threadIdx.x, hl = t >> 2, qd = t & 3;  // four threads per row, eight lane partials each
      f32x2 s12 = 0ull;
      float ss = 0.f;
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        const float4 v = rowacc[hl][(8 * qd + i + hl) & 31];
        s12 = add2(s12, pack2(v.x, v.y));
        ss += v.z;
      }
      float s1, s2;
      unpack2(s12, s1, s2);
#pragma unroll
      for (int o = 1; o <= 2; o <<= 1) {
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
        s2 += __shfl_xor_sync(0xffffffffu, s2, o);
        ss += __shfl_xor_sync(0xffffffffu, ss, o);
      }
      const int64_t row = (int64_t)rb * kSumRows + 16 * (hl >> 3) + 8 * half + (hl & 7);
      if (qd == 0 && row < n) *reinterpret_cast<float4*>(rowpart + ((int64_t)cb * n + row) * 4) = make_float4(s1, s2, ss, 0.f);
    }
    __syncthreads();  // rowacc is reused by the second half
  }
#pragma unroll
  for (int e = 0; e < 2; ++e) {
    float a0, a1, b0, b1, c0, c1;
    unpack2(cs1[e], a0, a1); unpack2(cs2[e], b0, b1); unpack2(css[e], c0, c1);
    colacc[w][jl + 2 * e][0] = a0; colacc[w][jl + 2 * e][1] = b0; colacc[w][jl + 2 * e][2] = c0;
    colacc[w][jl + 2 * e + 1][0] = a1; colacc[w][jl + 2 * e + 1][1] = b1; colacc[w][jl + 2 * e + 1][2] = c1;
  }
  __syncthreads();
  if (threadIdx.x < kSumCols) {
    const int c = threadIdx.x;
    const int64_t gc = (int64_t)cb * kSumCols + c;
    if (gc < m) {
      float a = 0.f, b = 0.f, e2 = 0.f;
#pragma unroll
      for (int g = 0; g < 8; ++g) { a += colacc[g][c][0]; b += colacc[g][c][1]; e2 += colacc[g][c][2]; }
      *reinterpret_cast<float4*>(colpart + ((int64_t)rb * m + gc) * 4) = make_float4(a, b, e2, 0.f);
    }
  }
}

int syndrome_unfused_dispatch(int64_t n, int64_t m, const float* C, int64_t ldc, float* rowpart, float* colpart, cudaStream_t stream) {
  if (ldc * 4 > 0xFFFFFFFFll) return GECC_EUNSUPPORTED;
  dim3 grid((unsigned)((m + kSumCols - 1) / kSumCols), (unsigned)((n + kSumRows - 1) / kSumRows));
  syndrome_unfused_kernel<<<grid, 256, 0, stream>>>((int)n, (int)m, C, ldc, rowpart, colpart);
  return cudaGetLastError() == cudaSuccess ? GECC_OK : GECC_ECUDA;
}

// E1 / E2: additive fault on a stored symbol of A or B, as the operand dtype stores it.
__global__ void inject_inputs_kernel(int dtype, int trans_a, int trans_b, void* A, int64_t lda, float* A_lo, void* B, int64_t ldb, float* B_lo, const gecc_fault_t* faults,
                                     int n_faults) {
  const int f = threadIdx.x;
  if (f >= n_faults) return;
  const gecc_fault_t ft = faults[f];
  if (ft.kind != GECC_KIND_A && ft.kind != GECC_KIND_B) return;
  void* X = ft.kind == GECC_KIND_A ? A : B;
  float* X_lo = ft.kind == GECC_KIND_A ? A_lo : B_lo;
  const bool tr = ft.kind == GECC_KIND_A ? trans_a != 0 : trans_b != 0;  // transposed storage: the symbol (r, c) sits at [c][r]
  const int64_t ldx = ft.kind == GECC_KIND_A ? lda : ldb;
  const int64_t idx = tr ? (int64_t)ft.col * ldx + ft.row : (int64_t)ft.row * ldx + ft.col;
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
