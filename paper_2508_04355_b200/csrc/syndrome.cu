// The standalone (unfused) pass over a stored C that produces the same partial sums of the detection step
// as the protected product's epilogue, and the input-fault injection hook.
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "encode_core.cuh"
#include "gecc_internal.h"

namespace gecc {

// Persistent blocks, each taking kSumRows x kSumCols tiles of C (64 KB) round-robin; a tile is read once with 16-byte
// loads: warp w owns rows 16 w .. 16 w + 15, lane l owns columns 4 l .. 4 l + 3, in two halves of 8 rows per warp.  The
// loads of the next half (of this tile or of the block's next one) are issued as soon as the current half has been summed,
// so they are in flight during the barriers and the row reduction: the memory pipe never drains between tiles.  The pass
// is HBM-bound only if it stays light on instructions: the per-vector sums use packed fp32 pairs (FADD2 / FFMA2), and a
// row's 32 lane partials are summed through shared memory (one 16-byte store per vector, rotated so that both the stores
// and the reads are conflict-free) instead of 15 shuffles per row.  Column sums go across the warps through
// shared memory.
// Partial layout (gecc_internal.h): rowpart[cb][n][4], colpart[rb][m][4] = (sum, local-weighted sum, sum of squares, 0).
__global__ void __launch_bounds__(256, 3) syndrome_unfused_kernel(int n, int m, int ncb, int ntiles, const float* __restrict__ C, int64_t ldc,
                                                                   float* __restrict__ rowpart, float* __restrict__ colpart, DecodeState* st) {
  if (blockIdx.x == 0 && threadIdx.x == 0) st->syn_status = 0;  // partial sums only: the decoder folds them itself
  static_assert(kSumRows == 128 && kSumCols == 128, "tile shape of the unfused pass");
  // [row of the half][lane rotated by 4 x row]: (sum, weighted sum, squares, -).  A 16-byte access is served a quarter warp
  // at a time: the rotation makes the eight slots of every quarter distinct modulo 8, for the stores (one row per warp)
  // and for the reads (two rows x four interleaved quarters of a row per quarter warp) alike.
  __shared__ float4 rowacc[64][32];
  __shared__ float4 colacc[3][8][kSumCols / 4];  // [sum, weighted, squares][warp][lane]: the lane's four columns
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int jl = 4 * lane;
  const f32x2 wj01 = pack2((float)jl, (float)(jl + 1)), wj23 = pack2((float)(jl + 2), (float)(jl + 3));
  const uint32_t ldb = (uint32_t)(ldc * 4);  // bytes per row (host checks the range)
  uint4 x[8];
  // the eight vectors of one half of one tile; rows / columns outside C read as zero; nothing is issued past the last tile
  auto issue = [&](int tile, int half) {
    if (tile >= ntiles) return;
    const int rb = tile / ncb, cb = tile - rb * ncb;
    const int64_t row0 = (int64_t)rb * kSumRows + 16 * w + 8 * half, col = (int64_t)cb * kSumCols + jl;
    const char* base = reinterpret_cast<const char*>(C + row0 * ldc + col);
    const bool full = (int64_t)(rb + 1) * kSumRows <= n && (int64_t)(cb + 1) * kSumCols <= m;
    if (full) {
#pragma unroll
      for (int u = 0; u < 8; ++u) ld_stream_if(x[u], base + (uint64_t)ldb * (uint32_t)u, true);
    } else {
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        x[u] = make_uint4(0u, 0u, 0u, 0u);
        ld_stream_if(x[u], base + (uint64_t)ldb * (uint32_t)u, row0 + u < n && col < m);
      }
    }
  };
  issue((int)blockIdx.x, 0);
#pragma unroll 1
  for (int tile = (int)blockIdx.x; tile < ntiles; tile += (int)gridDim.x) {
    const int rb = tile / ncb, cb = tile - rb * ncb;
    f32x2 cs1[2] = {0ull, 0ull}, cs2[2] = {0ull, 0ull}, css[2] = {0ull, 0ull};
#pragma unroll
    for (int half = 0; half < 2; ++half) {
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int il = 16 * w + 8 * half + u;  // row within the tile
        const int hl = 8 * w + u;              // row within the half
        const f32x2 p01 = pack2(__uint_as_float(x[u].x), __uint_as_float(x[u].y)), p23 = pack2(__uint_as_float(x[u].z), __uint_as_float(x[u].w));
        const f32x2 q01 = mul2(p01, p01), q23 = mul2(p23, p23);
        const f32x2 wt = pack2((float)il, (float)il);
        cs1[0] = add2(cs1[0], p01); cs1[1] = add2(cs1[1], p23);
        cs2[0] = fma2(wt, p01, cs2[0]); cs2[1] = fma2(wt, p23, cs2[1]);
        css[0] = add2(css[0], q01); css[1] = add2(css[1], q23);
        float a0, a1, b0, b1, c0, c1;
        unpack2(add2(p01, p23), a0, a1);
        unpack2(fma2(wj01, p01, mul2(wj23, p23)), b0, b1);
        unpack2(add2(q01, q23), c0, c1);
        rowacc[hl][(lane + 4 * hl) & 31] = make_float4(a0 + a1, b0 + b1, c0 + c1, 0.f);
      }
      if (half == 0) issue(tile, 1);  // in flight during the reduction below
      else issue(tile + (int)gridDim.x, 0);
      __syncthreads();
      {
        const int t = threadIdx.x, hl = t >> 2, qd = t & 3;  // four threads per row, eight lane partials each
        f32x2 s12 = 0ull;
        float ss = 0.f;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const float4 v = rowacc[hl][(qd + 4 * i + 4 * hl) & 31];
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
      __syncthreads();  // rowacc is reused by the next half
    }
    {
      float a0, a1, a2, a3;
      unpack2(cs1[0], a0, a1); unpack2(cs1[1], a2, a3);
      colacc[0][w][lane] = make_float4(a0, a1, a2, a3);
      unpack2(cs2[0], a0, a1); unpack2(cs2[1], a2, a3);
      colacc[1][w][lane] = make_float4(a0, a1, a2, a3);
      unpack2(css[0], a0, a1); unpack2(css[1], a2, a3);
      colacc[2][w][lane] = make_float4(a0, a1, a2, a3);
    }
    __syncthreads();  // (the next write of colacc is four barriers away)
    if (threadIdx.x < kSumCols) {
      const int c = threadIdx.x;
      const int64_t gc = (int64_t)cb * kSumCols + c;
      if (gc < m) {
        float a = 0.f, b = 0.f, e2 = 0.f;
#pragma unroll
        for (int g = 0; g < 8; ++g) {
          a += reinterpret_cast<const float*>(&colacc[0][g][0])[c];
          b += reinterpret_cast<const float*>(&colacc[1][g][0])[c];
          e2 += reinterpret_cast<const float*>(&colacc[2][g][0])[c];
        }
        *reinterpret_cast<float4*>(colpart + ((int64_t)rb * m + gc) * 4) = make_float4(a, b, e2, 0.f);
      }
    }
  }
}

int syndrome_unfused_dispatch(int64_t n, int64_t m, const float* C, int64_t ldc, float* rowpart, float* colpart, DecodeState* st, cudaStream_t stream) {
  if (ldc * 4 > 0xFFFFFFFFll) return GECC_EUNSUPPORTED;
  const int64_t ncb = (m + kSumCols - 1) / kSumCols, nrb = (n + kSumRows - 1) / kSumRows, ntiles = ncb * nrb;
  if (ntiles > 0x7FFFFFFFll - 1024) return GECC_EUNSUPPORTED;
  const int64_t cap = 3 * (int64_t)num_sms();
  const unsigned grid = (unsigned)(ntiles < cap ? ntiles : cap);
  syndrome_unfused_kernel<<<grid, 256, 0, stream>>>((int)n, (int)m, (int)ncb, (int)ntiles, C, ldc, rowpart, colpart, st);
  return cudaGetLastError() == cudaSuccess ? GECC_OK : GECC_ECUDA;
}

// E1 / E2: additive fault on a stored symbol of A or B, as the operand dtype stores it.
__global__ void inject_inputs_kernel(int dtype, int trans_a, int trans_b, void* A, int64_t lda, float* A_lo, void* B, int64_t ldb, float* B_lo, const gecc_fault_t* faults,
                                     int n_faults) {
  // launched as a programmatic dependent: the encoder before it has read the operands once this returns (the fault strikes AFTER
  // encoding, reading R1), and the product after it may set itself up meanwhile (it waits for this grid before it reads anything)
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
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
