// Encoder: the plain and the weighted checksum of every column of A (A_P) and of
// every row of B (B_P).  One streaming pass over the operand, 16-byte loads, HBM-bound.
//
// Two reduction directions cover both sides (and, later, transposed operands):
//   colsum: out[c] = sum over storage rows r of w(r) x[r][c]   (GECC_LEFT on a row-major A)
//   rowsum: out[r] = sum over storage cols c of w(c) x[r][c]   (GECC_RIGHT on a row-major B)
// with w = 1 (check 0) and w = index + 1 (check 1).  Sums of 8 elements are formed in fp32 with small local weights
// and folded into fp64 accumulators; the reduction order is fixed, so a second pass over unchanged data reproduces
// the first bit for bit (the input verification of the decoder relies on this).
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "gecc_internal.h"

namespace gecc {

template <typename T>
struct Vec;
template <>
struct Vec<__nv_bfloat16> {
  static constexpr int V = 8;
  __device__ static void load(const __nv_bfloat16* p, float (&x)[8]) {
    const uint4 u = __ldg(reinterpret_cast<const uint4*>(p));
    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      x[2 * i] = __uint_as_float(w[i] << 16);
      x[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    }
  }
};
template <>
struct Vec<float> {
  static constexpr int V = 4;
  __device__ static void load(const float* p, float (&x)[4]) {
    const float4 u = __ldg(reinterpret_cast<const float4*>(p));
    x[0] = u.x; x[1] = u.y; x[2] = u.z; x[3] = u.w;
  }
};

__device__ __forceinline__ float tf32_trunc(float x) { return __uint_as_float(__float_as_uint(x) & 0xFFFFE000u); }

__device__ __forceinline__ void store_lo(float* dst, const float (&x)[4]) {
  *reinterpret_cast<float4*>(dst) = make_float4(x[0] - tf32_trunc(x[0]), x[1] - tf32_trunc(x[1]), x[2] - tf32_trunc(x[2]), x[3] - tf32_trunc(x[3]));
}
__device__ __forceinline__ void store_lo(float*, const float (&)[8]) {}

// The two checks of one line, as the product consumes them: bf16 -> 3 limbs each (rows 3c + l), fp32 -> tf32 hi part in
// `parity` row 3c and the remainder in `parity_lo` row 3c.
__device__ __forceinline__ void write_parity(int dtype, void* parity, float* parity_lo, int64_t len, int64_t idx, double s1, double s2) {
  const double s[2] = {s1, s2};
  if (dtype == GECC_BF16) {
    __nv_bfloat16* P = reinterpret_cast<__nv_bfloat16*>(parity);
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      double rem = s[c];
#pragma unroll
      for (int l = 0; l < 3; ++l) {
        const __nv_bfloat16 h = __double2bfloat16(rem);
        P[(3 * c + l) * len + idx] = h;
        rem -= (double)__bfloat162float(h);
      }
    }
    P[6 * len + idx] = __float2bfloat16(0.f);
    P[7 * len + idx] = __float2bfloat16(0.f);
  } else {
    float* P = reinterpret_cast<float*>(parity);
#pragma unroll
    for (int r = 0; r < GECC_PAR_ROWS; ++r) {
      float hi = 0.f, lo = 0.f;
      if (r == 0 || r == 3) {
        const float v = (float)s[r / 3];
        hi = tf32_trunc(v);
        lo = v - hi;
      }
      P[r * len + idx] = hi;
      parity_lo[r * len + idx] = lo;
    }
  }
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ---------------------------------------------------------------------------------------------
// colsum: block = 32 column-threads x 8 row-groups; covers 32 V columns x kEncRowsPerChunk rows.
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) colsum_kernel(const T* __restrict__ X, int64_t rows, int64_t cols, int64_t ld, float* __restrict__ x_lo,
                                                      double* __restrict__ encpart, double* __restrict__ sumsq_part, const int* enable) {
  if (enable && *enable == 0) return;
  constexpr int V = Vec<T>::V;
  __shared__ double sm[8][32 * V][2];
  __shared__ double sq[8];
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const int64_t c0 = ((int64_t)blockIdx.x * 32 + tx) * V;
  const int64_t rbase = (int64_t)blockIdx.y * kEncRowsPerChunk;
  double S1[V], S2[V];
  float q = 0.f;
#pragma unroll
  for (int v = 0; v < V; ++v) { S1[v] = 0.0; S2[v] = 0.0; }
  if (c0 < cols) {
    for (int g = 0; g < kEncRowsPerChunk / 64; ++g) {  // 8 rows per group, 64 apart in the chunk
      float s[V], sw[V];
#pragma unroll
      for (int v = 0; v < V; ++v) { s[v] = 0.f; sw[v] = 0.f; }
      float x[8][V];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int64_t r = rbase + ty + 64 * g + 8 * u;
        if (r < rows) Vec<T>::load(X + r * ld + c0, x[u]);
        else {
#pragma unroll
          for (int v = 0; v < V; ++v) x[u][v] = 0.f;
        }
      }
      const double wbase = (double)(ty + 64 * g);  // row within the chunk of u = 0
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int64_t r = rbase + ty + 64 * g + 8 * u;
        if (x_lo && r < rows) store_lo(x_lo + r * ld + c0, x[u]);
#pragma unroll
        for (int v = 0; v < V; ++v) {
          q = fmaf(x[u][v], x[u][v], q);
          if (sizeof(T) == 4) {  // fp32 symbols: straight into fp64
            S1[v] += (double)x[u][v];
            S2[v] += (wbase + (double)(8 * u)) * (double)x[u][v];
          } else {               // bf16 symbols: 8-term fp32 sums with 6-bit weights are exact up to exponent spread
            s[v] += x[u][v];
            sw[v] = fmaf((float)(8 * u), x[u][v], sw[v]);
          }
        }
      }
      if (sizeof(T) != 4) {
#pragma unroll
        for (int v = 0; v < V; ++v) {
          S1[v] += (double)s[v];
          S2[v] += wbase * (double)s[v] + (double)sw[v];
        }
      }
    }
  }
#pragma unroll
  for (int v = 0; v < V; ++v) { sm[ty][tx * V + v][0] = S1[v]; sm[ty][tx * V + v][1] = S2[v]; }
  const double qw = warp_sum((double)q);
  if (tx == 0) sq[ty] = qw;
  __syncthreads();
  const int t = threadIdx.x;
  if (t < 32 * V) {
    const int64_t c = (int64_t)blockIdx.x * 32 * V + t;
    if (c < cols) {
      double a = 0.0, b = 0.0;
#pragma unroll
      for (int g = 0; g < 8; ++g) { a += sm[g][t][0]; b += sm[g][t][1]; }
      encpart[((int64_t)blockIdx.y * 2 + 0) * cols + c] = a;
      encpart[((int64_t)blockIdx.y * 2 + 1) * cols + c] = b;  // weights local to the chunk, 0-based
    }
  }
  if (t == 0 && sumsq_part) {
    double a = 0.0;
#pragma unroll
    for (int g = 0; g < 8; ++g) a += sq[g];
    sumsq_part[(int64_t)blockIdx.y * gridDim.x + blockIdx.x] = a;
  }
}

__global__ void colsum_finalize_kernel(int dtype, const double* __restrict__ encpart, int64_t chunks, int64_t len, void* parity, float* parity_lo,
                                       double* __restrict__ par64, const int* enable) {
  if (enable && *enable == 0) return;
  const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= len) return;
  double s1 = 0.0, s2 = 0.0;
  for (int64_t ch = 0; ch < chunks; ++ch) {
    const double a = encpart[(ch * 2 + 0) * len + c], b = encpart[(ch * 2 + 1) * len + c];
    s1 += a;
    s2 += (double)(ch * kEncRowsPerChunk + 1) * a + b;  // weight of 0-based row r is r + 1
  }
  par64[c] = s1;
  par64[len + c] = s2;
  if (parity) write_parity(dtype, parity, parity_lo, len, c, s1, s2);
}

// ---------------------------------------------------------------------------------------------
// rowsum: one warp per storage row, 8 rows per block.
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) rowsum_kernel(int dtype, const T* __restrict__ X, int64_t rows, int64_t cols, int64_t ld,
                                                      float* __restrict__ x_lo, void* parity, float* parity_lo, double* __restrict__ par64,
                                                      double* __restrict__ sumsq_part, const int* enable) {
  if (enable && *enable == 0) return;
  constexpr int V = Vec<T>::V;
  __shared__ double sq[8];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int64_t r = (int64_t)blockIdx.x * 8 + w;
  double S1 = 0.0, S2 = 0.0;
  float q = 0.f;
  if (r < rows) {
    const T* row = X + r * ld;
    const int64_t nvec = cols / V;
    for (int64_t v0 = lane; v0 < nvec; v0 += 32 * 4) {
      float x[4][V];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int64_t vi = v0 + 32 * u;
        if (vi < nvec) Vec<T>::load(row + vi * V, x[u]);
        else {
#pragma unroll
          for (int v = 0; v < V; ++v) x[u][v] = 0.f;
        }
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int64_t vi = v0 + 32 * u;
        if (x_lo && vi < nvec) store_lo(x_lo + r * ld + vi * V, x[u]);
        float s = 0.f, sw = 0.f;
#pragma unroll
        for (int v = 0; v < V; ++v) {
          q = fmaf(x[u][v], x[u][v], q);
          if (sizeof(T) == 4) {
            S1 += (double)x[u][v];
            S2 += (double)(vi * V + v + 1) * (double)x[u][v];  // weight of 0-based column j is j + 1
          } else {
            s += x[u][v];
            sw = fmaf((float)v, x[u][v], sw);
          }
        }
        if (sizeof(T) != 4) {
          S1 += (double)s;
          S2 += (double)(vi * V + 1) * (double)s + (double)sw;
        }
      }
    }
  }
  S1 = warp_sum(S1);
  S2 = warp_sum(S2);
  const double qw = warp_sum((double)q);
  if (lane == 0) {
    sq[w] = qw;
    if (r < rows) {
      par64[r] = S1;
      par64[rows + r] = S2;
      if (parity) write_parity(dtype, parity, parity_lo, rows, r, S1, S2);
    }
  }
  __syncthreads();
  if (threadIdx.x == 0 && sumsq_part) {
    double a = 0.0;
#pragma unroll
    for (int g = 0; g < 8; ++g) a += sq[g];
    sumsq_part[blockIdx.x] = a;
  }
}

__global__ void sum_parts_kernel(const double* __restrict__ parts, int64_t nparts, double* __restrict__ out, const int* enable) {
  if (enable && *enable == 0) return;
  __shared__ double sm[32];
  double a = 0.0;
  for (int64_t i = threadIdx.x; i < nparts; i += blockDim.x) a += parts[i];
  a = warp_sum(a);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = a;
  __syncthreads();
  if (threadIdx.x < 32) {
    a = threadIdx.x < (blockDim.x >> 5) ? sm[threadIdx.x] : 0.0;
    a = warp_sum(a);
    if (threadIdx.x == 0) *out = a;
  }
}

template <typename T>
static int encode_typed(int dtype, bool reduce_over_rows, const T* X, int64_t rows, int64_t cols, int64_t ld, void* parity, float* parity_lo,
                        float* x_lo, double* par64, double* sumsq, double* encpart, double* sumsq_part, const int* enable, cudaStream_t stream) {
  constexpr int V = Vec<T>::V;
  int64_t nparts;
  if (reduce_over_rows) {
    const int64_t chunks = (rows + kEncRowsPerChunk - 1) / kEncRowsPerChunk;
    dim3 grid((unsigned)((cols + 32 * V - 1) / (32 * V)), (unsigned)chunks);
    nparts = (int64_t)grid.x * grid.y;
    colsum_kernel<T><<<grid, 256, 0, stream>>>(X, rows, cols, ld, x_lo, encpart, sumsq ? sumsq_part : nullptr, enable);
    colsum_finalize_kernel<<<(unsigned)((cols + 255) / 256), 256, 0, stream>>>(dtype, encpart, chunks, cols, parity, parity_lo, par64, enable);
  } else {
    const unsigned grid = (unsigned)((rows + 7) / 8);
    nparts = grid;
    rowsum_kernel<T><<<grid, 256, 0, stream>>>(dtype, X, rows, cols, ld, x_lo, parity, parity_lo, par64, sumsq ? sumsq_part : nullptr, enable);
  }
  if (sumsq) sum_parts_kernel<<<1, 1024, 0, stream>>>(sumsq_part, nparts, sumsq, enable);
  return cudaGetLastError() == cudaSuccess ? GECC_OK : GECC_ECUDA;
}

int encode_dispatch(int dtype, bool reduce_over_rows, const void* X, int64_t rows, int64_t cols, int64_t ld, void* parity, float* parity_lo,
                    float* x_lo, double* par64, double* sumsq, double* encpart, double* sumsq_part, const int* enable, cudaStream_t stream) {
  if (dtype == GECC_BF16)
    return encode_typed<__nv_bfloat16>(dtype, reduce_over_rows, reinterpret_cast<const __nv_bfloat16*>(X), rows, cols, ld, parity, nullptr, nullptr,
                                       par64, sumsq, encpart, sumsq_part, enable, stream);
  return encode_typed<float>(dtype, reduce_over_rows, reinterpret_cast<const float*>(X), rows, cols, ld, parity, parity_lo, x_lo, par64, sumsq,
                             encpart, sumsq_part, enable, stream);
}

}  // namespace gecc
