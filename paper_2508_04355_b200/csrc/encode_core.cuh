// Streaming checksum reductions shared by the encoder kernels (encode.cu) and the input verification of the decoder
// (decode.cu): the plain and the weighted sum of every column (colsum) or every row (rowsum) of a row-major operand.
//
//   colsum: out[c] = sum over storage rows r of w(r) x[r][c]   (GECC_LEFT on a row-major A:  A_P)
//   rowsum: out[r] = sum over storage cols c of w(c) x[r][c]   (GECC_RIGHT on a row-major B: B_P)
// with w = 1 (check 0) and w = index + 1 (check 1).
//
// Arithmetic: bf16 symbols are summed 8 at a time in fp32 with small local weights (0..56 / 0..7; exact unless the
// exponents of the 8 symbols spread over more than ~10 bits) and folded into fp64; fp32 symbols go straight to fp64.  The
// order of every sum is fixed by the indices alone, so a second pass over unchanged data reproduces the first bit for
// bit: the input verification compares its sums with the ones stored at encode time for equality.  Explicit _rn
// intrinsics keep the compiler from contracting the sums differently in the two kernels that inline these functions.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include "gecc_internal.h"

namespace gecc {

// 16-byte streaming load.  volatile: the compiler keeps a run of these together, so all of them are in flight before the
// first use (it otherwise sinks loads towards their uses to save registers, which serialises the memory latency).
__device__ __forceinline__ uint4 ld_stream(const void* p) {
  uint4 u;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(u.x), "=r"(u.y), "=r"(u.z), "=r"(u.w) : "l"(p));
  return u;
}

// Ties eight loaded vectors together: every one of them is made to depend (through a value that is zero at run time but
// unknown at compile time) on all eight loads, so the first use cannot be scheduled before the last load was issued.
__device__ __forceinline__ void join_loads(uint4 (&raw)[8], uint32_t runtime_zero) {
  uint32_t dep = raw[0].x;
#pragma unroll
  for (int u = 1; u < 8; ++u) dep ^= raw[u].x;
  dep &= runtime_zero;
#pragma unroll
  for (int u = 0; u < 8; ++u) raw[u].x |= dep;
}

template <typename T>
struct Vec;
template <>
struct Vec<__nv_bfloat16> {
  static constexpr int V = 8;
  __device__ static uint4 raw(const __nv_bfloat16* p) { return ld_stream(p); }
  __device__ static void unpack(const uint4& u, float (&x)[8]) {
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
  __device__ static uint4 raw(const float* p) { return ld_stream(p); }
  __device__ static void unpack(const uint4& u, float (&x)[4]) {
    x[0] = __uint_as_float(u.x); x[1] = __uint_as_float(u.y); x[2] = __uint_as_float(u.z); x[3] = __uint_as_float(u.w);
  }
};

__device__ __forceinline__ float tf32_trunc(float x) { return __uint_as_float(__float_as_uint(x) & 0xFFFFE000u); }

__device__ __forceinline__ void store_lo(float* dst, const float (&x)[4]) {
  *reinterpret_cast<float4*>(dst) = make_float4(x[0] - tf32_trunc(x[0]), x[1] - tf32_trunc(x[1]), x[2] - tf32_trunc(x[2]), x[3] - tf32_trunc(x[3]));
}
__device__ __forceinline__ void store_lo(float*, const float (&)[8]) {}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = __dadd_rn(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

// Arrival on a self-cleaning counter: true in every thread of the block that arrives last of `expected`.
__device__ __forceinline__ bool arrive_last(unsigned int* ctr, unsigned int expected, int& flag_smem) {
  __syncthreads();  // the block's writes happen before the barrier, the fence below makes them visible before the arrival
  if (threadIdx.x == 0) {
    __threadfence();
    const unsigned int t = atomicAdd(ctr, 1u);
    flag_smem = (t == expected - 1);
    if (flag_smem) *ctr = 0;  // leave the counter clean for the next launch
    __threadfence();
  }
  __syncthreads();
  return flag_smem != 0;
}

// Shared memory of one 256-thread block running either reduction.
template <typename T>
struct EncSmem {
  double part[2][8][Vec<T>::V][32];  // [check][warp][column within the lane's vector][lane]: conflict-free both ways
  double sq[8];
  int last;
};

// ---------------------------------------------------------------------------------------------
// colsum, one work item: column strip `strip` (32 V columns) x row chunk `chunk` (chunk_rows rows, a multiple of 64).
// 256 threads: lane -> V columns, warp w -> rows w, w + 8, ... of the chunk.  Writes the chunk's two sums per column
// (weights local to the chunk, 0-based) to encpart[chunk][2][cols]; returns the item's sum of squares in thread 0.
// ---------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ double colsum_item(const T* __restrict__ X, int64_t rows, int64_t cols, int64_t ld, float* __restrict__ x_lo,
                                              double* __restrict__ encpart, int strip, int chunk, int chunk_rows, EncSmem<T>& sm) {
  constexpr int V = Vec<T>::V;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const int64_t c0 = ((int64_t)strip * 32 + tx) * V;
  const int64_t rbase = (int64_t)chunk * chunk_rows;
  double S1[V], S2[V];
  float q = 0.f;
#pragma unroll
  for (int v = 0; v < V; ++v) { S1[v] = 0.0; S2[v] = 0.0; }
  if (c0 < cols) {
#pragma unroll 1
    for (int g = 0; g < chunk_rows / 64; ++g) {  // 8 rows per group, 8 apart
      // all eight loads are issued before any is used (rows past the end re-read the last row and are zeroed)
      uint4 raw[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int64_t r = rbase + ty + 64 * g + 8 * u;
        raw[u] = Vec<T>::raw(X + (r < rows ? r : rows - 1) * ld + c0);
      }
      join_loads(raw, (uint32_t)((uint64_t)rows >> 40));
      float x[8][V];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int64_t r = rbase + ty + 64 * g + 8 * u;
        if (!(r < rows)) raw[u] = make_uint4(0u, 0u, 0u, 0u);
        Vec<T>::unpack(raw[u], x[u]);
      }
      float s[V], sw[V];
#pragma unroll
      for (int v = 0; v < V; ++v) { s[v] = 0.f; sw[v] = 0.f; }
      const double wbase = (double)(ty + 64 * g);  // row within the chunk of u = 0
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int64_t r = rbase + ty + 64 * g + 8 * u;
        if (x_lo && r < rows) store_lo(x_lo + r * ld + c0, x[u]);
#pragma unroll
        for (int v = 0; v < V; ++v) {
          q = fmaf(x[u][v], x[u][v], q);
          if (sizeof(T) == 4) {  // fp32 symbols: straight into fp64
            S1[v] = __dadd_rn(S1[v], (double)x[u][v]);
            S2[v] = __fma_rn(wbase + (double)(8 * u), (double)x[u][v], S2[v]);
          } else {
            s[v] = __fadd_rn(s[v], x[u][v]);
            sw[v] = __fmaf_rn((float)(8 * u), x[u][v], sw[v]);
          }
        }
      }
      if (sizeof(T) != 4) {
#pragma unroll
        for (int v = 0; v < V; ++v) {
          S1[v] = __dadd_rn(S1[v], (double)s[v]);
          S2[v] = __dadd_rn(S2[v], __fma_rn(wbase, (double)s[v], (double)sw[v]));
        }
      }
    }
  }
#pragma unroll
  for (int v = 0; v < V; ++v) { sm.part[0][ty][v][tx] = S1[v]; sm.part[1][ty][v][tx] = S2[v]; }
  const double qw = warp_sum((double)q);
  if (tx == 0) sm.sq[ty] = qw;
  __syncthreads();
  const int t = threadIdx.x;
  if (t < 32 * V) {
    const int tl = t & 31, tv = t >> 5;  // thread t folds the column of lane tl, vector element tv
    const int64_t c = ((int64_t)strip * 32 + tl) * V + tv;
    if (c < cols) {
      double a = 0.0, b = 0.0;
#pragma unroll
      for (int g = 0; g < 8; ++g) { a = __dadd_rn(a, sm.part[0][g][tv][tl]); b = __dadd_rn(b, sm.part[1][g][tv][tl]); }
      encpart[((int64_t)chunk * 2 + 0) * cols + c] = a;
      encpart[((int64_t)chunk * 2 + 1) * cols + c] = b;
    }
  }
  double qs = 0.0;
  if (t == 0) {
#pragma unroll
    for (int g = 0; g < 8; ++g) qs += sm.sq[g];
  }
  __syncthreads();  // sm is reused by the caller's next item
  return qs;
}

// The two checks of column c from the chunk partials, chunks summed in order; weight of 0-based row r is r + 1.
__device__ __forceinline__ void colsum_combine(const double* __restrict__ encpart, int64_t chunks, int chunk_rows, int64_t cols, int64_t c, double& s1,
                                               double& s2) {
  s1 = 0.0;
  s2 = 0.0;
  int64_t ch = 0;
  for (; ch + 8 <= chunks; ch += 8) {
    double a[8], b[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      a[u] = __ldcg(encpart + ((ch + u) * 2 + 0) * cols + c);
      b[u] = __ldcg(encpart + ((ch + u) * 2 + 1) * cols + c);
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      s1 = __dadd_rn(s1, a[u]);
      s2 = __dadd_rn(s2, __fma_rn((double)((ch + u) * chunk_rows + 1), a[u], b[u]));
    }
  }
  for (; ch < chunks; ++ch) {
    const double a = __ldcg(encpart + (ch * 2 + 0) * cols + c), b = __ldcg(encpart + (ch * 2 + 1) * cols + c);
    s1 = __dadd_rn(s1, a);
    s2 = __dadd_rn(s2, __fma_rn((double)(ch * chunk_rows + 1), a, b));
  }
}

// ---------------------------------------------------------------------------------------------
// rowsum: one warp per storage row.  Returns (in every lane) the two checks of the row; q accumulates squares per lane.
// ---------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ void rowsum_warp(const T* __restrict__ row, int64_t cols, float* __restrict__ lo_row, double& S1, double& S2, float& q) {
  constexpr int V = Vec<T>::V;
  const int lane = threadIdx.x & 31;
  const int64_t nvec = cols / V;
  S1 = 0.0;
  S2 = 0.0;
  for (int64_t v0 = lane; v0 < nvec; v0 += 32 * 8) {
    uint4 raw[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int64_t vi = v0 + 32 * u;
      raw[u] = Vec<T>::raw(row + (vi < nvec ? vi : nvec - 1) * V);
    }
    join_loads(raw, (uint32_t)((uint64_t)cols >> 40));
    float x[8][V];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int64_t vi = v0 + 32 * u;
      if (!(vi < nvec)) raw[u] = make_uint4(0u, 0u, 0u, 0u);
      Vec<T>::unpack(raw[u], x[u]);
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int64_t vi = v0 + 32 * u;
      if (lo_row && vi < nvec) store_lo(lo_row + vi * V, x[u]);
      float s = 0.f, sw = 0.f;
#pragma unroll
      for (int v = 0; v < V; ++v) {
        q = fmaf(x[u][v], x[u][v], q);
        if (sizeof(T) == 4) {
          S1 = __dadd_rn(S1, (double)x[u][v]);
          S2 = __fma_rn((double)(vi * V + v + 1), (double)x[u][v], S2);  // weight of 0-based column j is j + 1
        } else {
          s = __fadd_rn(s, x[u][v]);
          sw = __fmaf_rn((float)v, x[u][v], sw);
        }
      }
      if (sizeof(T) != 4) {
        S1 = __dadd_rn(S1, (double)s);
        S2 = __dadd_rn(S2, __fma_rn((double)(vi * V + 1), (double)s, (double)sw));
      }
    }
  }
  S1 = warp_sum(S1);
  S2 = warp_sum(S2);
}

}  // namespace gecc
