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

// Predicated 16-byte streaming load: `raw` keeps its value when `pred` is false.  The reductions below keep a ring of
// eight such loads per thread in flight: a vector is consumed and its register reloaded with the vector eight rows on,
// so the memory pipe never drains while a group is being summed.
__device__ __forceinline__ void ld_stream_if(uint4& raw, const void* p, bool pred) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %5, 0;\n\t@p ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];\n\t}"
      : "+r"(raw.x), "+r"(raw.y), "+r"(raw.z), "+r"(raw.w)
      : "l"(p), "r"((uint32_t)pred));
}

// Packed fp32 pairs (sm_100: FADD2 / FFMA2, round to nearest like the scalar forms): two symbols per instruction.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
  f32x2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
  f32x2 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
// two bf16 symbols of one 32-bit word, widened exactly: (even, odd)
__device__ __forceinline__ f32x2 bf16x2_widen(uint32_t w) { return pack2(__uint_as_float(w << 16), __uint_as_float(w & 0xFFFF0000u)); }

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
// colsum: the groups of one work item for one thread.  The thread's rows are rbase + ty + 8 j; a group is eight of them
// (64 rows of the chunk), summed in fp32 with the local weights 0, 8, .., 56 and folded into fp64 (bf16), or summed
// straight into fp64 (fp32).  RAGGED: the chunk runs past the last row; rows past it count as zero.
// ---------------------------------------------------------------------------------------------
template <typename T, bool RAGGED>
__device__ __forceinline__ void colsum_groups(const T* __restrict__ X, int64_t rows, int64_t ld, float* __restrict__ x_lo, int64_t rbase, int64_t c0,
                                              int chunk_rows, int ty, double (&S1)[Vec<T>::V], double (&S2)[Vec<T>::V], float& q) {
  constexpr int V = Vec<T>::V;
  const int64_t left = rows - rbase;
  const int lim = (int)(left < (int64_t)chunk_rows ? left : (int64_t)chunk_rows) - ty;  // row offsets 8 j < lim exist
  const int groups = chunk_rows / 64;
  const uint32_t step = (uint32_t)(8 * ld * (int64_t)sizeof(T));  // bytes between two rows of this thread (host checks the range)
  const char* pg = reinterpret_cast<const char*>(X + (rbase + ty) * ld + c0);
  float* lo_g = x_lo ? x_lo + (rbase + ty) * ld + c0 : nullptr;
  uint4 raw[8];
#pragma unroll
  for (int u = 0; u < 8; ++u) {
    raw[u] = make_uint4(0u, 0u, 0u, 0u);
    ld_stream_if(raw[u], pg + (uint64_t)step * (uint32_t)u, 8 * u < lim);
  }
  f32x2 q2[V / 2];
#pragma unroll
  for (int i = 0; i < V / 2; ++i) q2[i] = 0ull;
#pragma unroll 1
  for (int g = 0; g < groups; ++g) {
    const double wbase = (double)(ty + 64 * g);  // row within the chunk of u = 0
    const bool more = g + 1 < groups;
    f32x2 s2[V / 2], sw2[V / 2];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const uint4 cur = raw[u];
      if (sizeof(T) == 4) {  // fp32 symbols: straight into fp64
        float x[V];
        Vec<T>::unpack(cur, x);
        if (lo_g && (!RAGGED || 64 * g + 8 * u < lim)) store_lo(lo_g + (int64_t)(8 * u) * ld, x);
#pragma unroll
        for (int v = 0; v < V; ++v) {
          q = fmaf(x[v], x[v], q);
          S1[v] = __dadd_rn(S1[v], (double)x[v]);
          S2[v] = __fma_rn(wbase + (double)(8 * u), (double)x[v], S2[v]);
        }
      } else {
        const uint32_t w[4] = {cur.x, cur.y, cur.z, cur.w};
        const f32x2 wu = pack2((float)(8 * u), (float)(8 * u));
#pragma unroll
        for (int i = 0; i < V / 2; ++i) {
          const f32x2 xx = bf16x2_widen(w[i & 3]);
          q2[i] = fma2(xx, xx, q2[i]);
          s2[i] = u == 0 ? xx : add2(s2[i], xx);
          sw2[i] = u == 0 ? 0ull : fma2(wu, xx, sw2[i]);
        }
      }
      // the vector is summed, its register free: fetch the one eight rows on (next group) into it
      bool pred = more;
      if (RAGGED) {
        raw[u] = make_uint4(0u, 0u, 0u, 0u);
        pred = 64 * (g + 1) + 8 * u < lim;
      }
      ld_stream_if(raw[u], pg + (uint64_t)step * (uint32_t)(8 + u), pred);
    }
    if (sizeof(T) != 4) {
#pragma unroll
      for (int i = 0; i < V / 2; ++i) {
        float a0, a1, b0, b1;
        unpack2(s2[i], a0, a1);
        unpack2(sw2[i], b0, b1);
        S1[2 * i] = __dadd_rn(S1[2 * i], (double)a0);
        S2[2 * i] = __dadd_rn(S2[2 * i], __fma_rn(wbase, (double)a0, (double)b0));
        S1[2 * i + 1] = __dadd_rn(S1[2 * i + 1], (double)a1);
        S2[2 * i + 1] = __dadd_rn(S2[2 * i + 1], __fma_rn(wbase, (double)a1, (double)b1));
      }
    }
    pg += (uint64_t)step * 8u;
    if (lo_g) lo_g += 64 * ld;
  }
  if (sizeof(T) != 4) {
#pragma unroll
    for (int i = 0; i < V / 2; ++i) {
      float a0, a1;
      unpack2(q2[i], a0, a1);
      q = __fadd_rn(q, __fadd_rn(a0, a1));
    }
  }
}

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
    if (rbase + chunk_rows <= rows) colsum_groups<T, false>(X, rows, ld, x_lo, rbase, c0, chunk_rows, ty, S1, S2, q);
    else colsum_groups<T, true>(X, rows, ld, x_lo, rbase, c0, chunk_rows, ty, S1, S2, q);
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
// Lane t sums the vectors t, t + 32, ...; a group is eight of them (256 V consecutive columns per warp).  bf16: within a
// group sum_v v x (v = 0..7, the index inside a vector) is kept in fp32 (exact products, exact sums unless exponents spread
// by more than ~10 bits); each vector's plain sum is taken in fp32 and goes to fp64 at once, where the vector's and the
// group's weights are applied; fp32: straight to fp64.
// RAGGED: the row is not a whole number of groups; vectors past its end count as zero.
// ---------------------------------------------------------------------------------------------
template <typename T, bool RAGGED>
__device__ __forceinline__ void rowsum_groups(const T* __restrict__ row, int nvec, float* __restrict__ lo_row, double& S1, double& S2, float& q) {
  constexpr int V = Vec<T>::V;
  const int lane = threadIdx.x & 31;
  const int groups = (nvec + 255) / 256;
  const char* pg = reinterpret_cast<const char*>(row) + 16 * lane;
  uint4 raw[8];
#pragma unroll
  for (int u = 0; u < 8; ++u) {
    raw[u] = make_uint4(0u, 0u, 0u, 0u);
    ld_stream_if(raw[u], pg + 512 * u, lane + 32 * u < nvec);
  }
  f32x2 q2[V / 2];
#pragma unroll
  for (int i = 0; i < V / 2; ++i) q2[i] = 0ull;
#pragma unroll 1
  for (int g = 0; g < groups; ++g) {
    const int vbase = g * 256 + lane;  // vector of u = 0
    const bool more = g + 1 < groups;
    f32x2 sw2[V / 2];
    double t = 0.0, tw = 0.0;
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const uint4 cur = raw[u];
      if (sizeof(T) == 4) {
        float x[V];
        Vec<T>::unpack(cur, x);
        const int vi = vbase + 32 * u;
        if (lo_row && (!RAGGED || vi < nvec)) store_lo(lo_row + (int64_t)vi * V, x);
#pragma unroll
        for (int v = 0; v < V; ++v) {
          q = fmaf(x[v], x[v], q);
          S1 = __dadd_rn(S1, (double)x[v]);
          S2 = __fma_rn((double)((int64_t)vi * V + v + 1), (double)x[v], S2);  // weight of 0-based column j is j + 1
        }
      } else {
        const uint32_t w[4] = {cur.x, cur.y, cur.z, cur.w};
        f32x2 xx[V / 2];
#pragma unroll
        for (int i = 0; i < V / 2; ++i) {
          xx[i] = bf16x2_widen(w[i & 3]);
          q2[i] = fma2(xx[i], xx[i], q2[i]);
          const f32x2 wv = pack2((float)(2 * i), (float)(2 * i + 1));
          sw2[i] = u == 0 ? fma2(wv, xx[i], 0ull) : fma2(wv, xx[i], sw2[i]);
        }
        float h0, h1;
        unpack2(add2(add2(xx[0], xx[1 % (V / 2)]), add2(xx[2 % (V / 2)], xx[3 % (V / 2)])), h0, h1);
        const double su = (double)__fadd_rn(h0, h1);  // plain sum of the vector; fp64 from here: it is no short-mantissa number any more
        t = __dadd_rn(t, su);
        tw = __fma_rn((double)u, su, tw);
      }
      // the vector is summed, its register free: fetch the next group's vector into it
      bool pred = more;
      if (RAGGED) {
        raw[u] = make_uint4(0u, 0u, 0u, 0u);
        pred = vbase + 256 + 32 * u < nvec;
      }
      ld_stream_if(raw[u], pg + 4096 + 512 * u, pred);
    }
    if (sizeof(T) != 4) {
      float h0, h1;
      unpack2(add2(add2(sw2[0], sw2[1 % (V / 2)]), add2(sw2[2 % (V / 2)], sw2[3 % (V / 2)])), h0, h1);
      const float swg = __fadd_rn(h0, h1);  // sum of (index within its vector) x symbol over the group
      S1 = __dadd_rn(S1, t);
      // weight of element v of vector u: (vbase + 32 u) V + v + 1 = (vbase V + 1) + 256 u + v
      S2 = __dadd_rn(S2, __fma_rn((double)((int64_t)vbase * V + 1), t, __fma_rn(256.0, tw, (double)swg)));
    }
    pg += 4096;
  }
  if (sizeof(T) != 4) {
#pragma unroll
    for (int i = 0; i < V / 2; ++i) {
      float a0, a1;
      unpack2(q2[i], a0, a1);
      q = __fadd_rn(q, __fadd_rn(a0, a1));
    }
  }
}

template <typename T>
__device__ __forceinline__ void rowsum_warp(const T* __restrict__ row, int64_t cols, float* __restrict__ lo_row, double& S1, double& S2, float& q) {
  constexpr int V = Vec<T>::V;
  const int nvec = (int)(cols / V);
  S1 = 0.0;
  S2 = 0.0;
  if (nvec % 256 == 0) rowsum_groups<T, false>(row, nvec, lo_row, S1, S2, q);
  else rowsum_groups<T, true>(row, nvec, lo_row, S1, S2, q);
  S1 = warp_sum(S1);
  S2 = warp_sum(S2);
}

}  // namespace gecc
