// The standalone (unfused) pass over a stored C that produces the same partial sums of the detection step
// as the protected product's epilogue, and the input-fault injection hook.
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "gecc_internal.h"

namespace gecc {

// One block per kSumRows x kSumCols tile of C (64 KB), read once with 16-byte loads: warp w owns rows 16 w .. 16 w + 15,
// lane l owns columns 4 l .. 4 l + 3.  Row sums by warp shuffles, column sums across the warps through shared memory.
// Partial layout (gecc_internal.h): rowpart[cb][n][4], colpart[rb][m][4] = (sum, local-weighted sum, sum of squares, 0).
__global__ void __launch_bounds__(256) syndrome_unfused_kernel(int n, int m, const float* __restrict__ C, int64_t ldc, float* __restrict__ rowpart,
                                                                float* __restrict__ colpart) {
  static_assert(kSumRows == 128 && kSumCols == 128, "tile shape of the unfused pass");
  __shared__ float colacc[8][kSumCols][3];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int cb = blockIdx.x, rb = blockIdx.y;
  const int jl = 4 * lane;
  const int64_t col = (int64_t)cb * kSumCols + jl;
  float cs1[4] = {0.f, 0.f, 0.f, 0.f}, cs2[4] = {0.f, 0.f, 0.f, 0.f}, css[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
  for (int half = 0; half < 2; ++half) {
    float4 x[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int64_t row = (int64_t)rb * kSumRows + 16 * w + 8 * half + u;
      x[u] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (row < n && col < m) x[u] = __ldcs(reinterpret_cast<const float4*>(C + row * ldc + col));
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int il = 16 * w + 8 * half + u;  // row within the tile
      const int64_t row = (int64_t)rb * kSumRows + il;
      const float4 v = x[u];
      float s1 = (v.x + v.y) + (v.z + v.w);
      float ss = (v.x * v.x + v.y * v.y) + (v.z * v.z + v.w * v.w);
      float s2 = fmaf((float)jl, v.x, fmaf((float)(jl + 1), v.y, fmaf((float)(jl + 2), v.z, (float)(jl + 3) * v.w)));
      const float wt = (float)il;
      cs1[0] += v.x; cs1[1] += v.y; cs1[2] += v.z; cs1[3] += v.w;
      cs2[0] = fmaf(wt, v.x, cs2[0]); cs2[1] = fmaf(wt, v.y, cs2[1]); cs2[2] = fmaf(wt, v.z, cs2[2]); cs2[3] = fmaf(wt, v.w, cs2[3]);
      css[0] = fmaf(v.x, v.x, css[0]); css[1] = fmaf(v.y, v.y, css[1]); css[2] = fmaf(v.z, v.z, css[2]); css[3] = fmaf(v.w, v.w, css[3]);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
        s2 += __shfl_xor_sync(0xffffffffu, s2, o);
        ss += __shfl_xor_sync(0xffffffffu, ss, o);
      }
      if (lane == 0 && row < n) *reinterpret_cast<float4*>(rowpart + ((int64_t)cb * n + row) * 4) = make_float4(s1, s2, ss, 0.f);
    }
  }
#pragma unroll
  for (int e = 0; e < 4; ++e) { colacc[w][jl + e][0] = cs1[e]; colacc[w][jl + e][1] = cs2[e]; colacc[w][jl + e][2] = css[e]; }
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
