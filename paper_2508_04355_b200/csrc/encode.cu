// Encoder: the plain and the weighted checksum of every column of A (A_P) and of
// every row of B (B_P).  One kernel launch per operand, one streaming pass over it with 16-byte loads
// (HBM-bound); the reductions themselves are in encode_core.cuh.  The last block to finish (arrival counters in the
// workspace) folds the per-chunk partials in a fixed order, so the result does not depend on block scheduling.
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <mutex>

#include "encode_core.cuh"
#include "gecc_internal.h"
#include "sm100_ptx.cuh"

namespace gecc {

__device__ __forceinline__ void ptx_griddep_launch_dependents() { ptx::griddep_launch_dependents(); }

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

// Sum of nparts doubles in index order by one 256-thread block (fixed tree), result in thread 0.
__device__ __forceinline__ double block_sum_parts(const double* parts, int64_t nparts, double* sq8) {
  double a = 0.0;
  for (int64_t i = threadIdx.x; i < nparts; i += 256) a += __ldcg(parts + i);
  a = warp_sum(a);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) sq8[threadIdx.x >> 5] = a;
  __syncthreads();
  double t = 0.0;
  if (threadIdx.x == 0)
    for (int g = 0; g < 8; ++g) t += sq8[g];
  return t;
}

// grid = (column strips, row chunks)
template <typename T>
__global__ void __launch_bounds__(256) encode_colsum_kernel(int dtype, const T* __restrict__ X, int64_t rows, int64_t cols, int64_t ld,
                                                             float* __restrict__ x_lo, void* parity, float* parity_lo, double* __restrict__ par64,
                                                             double* sumsq, unsigned int* counters, double* sumsq_part, double* encpart, int chunk_rows) {
  constexpr int V = Vec<T>::V;
  __shared__ EncSmem<T> sm;
  const int strip = blockIdx.x, chunk = blockIdx.y;
  const double qs = colsum_item<T>(X, rows, cols, ld, x_lo, encpart, strip, chunk, chunk_rows, sm);
  if (threadIdx.x == 0) sumsq_part[(int64_t)chunk * gridDim.x + strip] = qs;
  // last chunk of this strip to finish: fold the chunks of the strip's columns
  if (arrive_last(counters + kCtrEncStrip + strip, gridDim.y, sm.last)) {
    const int t = threadIdx.x;
    const int64_t c = (int64_t)strip * 32 * V + t;
    if (t < 32 * V && c < cols) {
      double s1, s2;
      colsum_combine(encpart, gridDim.y, chunk_rows, cols, c, s1, s2);
      par64[c] = s1;
      par64[cols + c] = s2;
      if (parity) write_parity(dtype, parity, parity_lo, cols, c, s1, s2);
    }
  }
  if (sumsq && arrive_last(counters + kCtrEncAll, gridDim.x * gridDim.y, sm.last)) {
    const double tot = block_sum_parts(sumsq_part, (int64_t)gridDim.x * gridDim.y, sm.sq);
    if (threadIdx.x == 0) *sumsq = tot;
  }
}

// one warp per storage row; the rows are dealt round-robin to all warps of the grid (a few blocks per SM), so that every
// SM gets the same share however the row count divides
template <typename T>
__global__ void __launch_bounds__(256, 2) encode_rowsum_kernel(int dtype, const T* __restrict__ X, int64_t rows, int64_t cols, int64_t ld,
                                                                float* __restrict__ x_lo, void* parity, float* parity_lo, double* __restrict__ par64,
                                                                double* sumsq, unsigned int* counters, double* sumsq_part) {
  __shared__ double sq[8];
  __shared__ int last;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  float q = 0.f;
#pragma unroll 1
  for (int64_t r = (int64_t)blockIdx.x * 8 + w; r < rows; r += (int64_t)gridDim.x * 8) {
    double S1, S2;
    rowsum_warp<T>(X + r * ld, cols, x_lo ? x_lo + r * ld : nullptr, S1, S2, q);
    if (lane == 0) {
      par64[r] = S1;
      par64[rows + r] = S2;
      if (parity) write_parity(dtype, parity, parity_lo, rows, r, S1, S2);
    }
  }
  const double qw = warp_sum((double)q);
  if (lane == 0) sq[w] = qw;
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0;
#pragma unroll
    for (int g = 0; g < 8; ++g) a += sq[g];
    sumsq_part[blockIdx.x] = a;
  }
  if (sumsq && arrive_last(counters + kCtrEncAllRow, gridDim.x, last)) {
    const double tot = block_sum_parts(sumsq_part, gridDim.x, sq);
    if (threadIdx.x == 0) *sumsq = tot;
  }
}

template <typename T>
static int encode_typed(int dtype, bool reduce_over_rows, const T* X, int64_t rows, int64_t cols, int64_t ld, void* parity, float* parity_lo,
                        float* x_lo, double* par64, double* sumsq, uint8_t* ws, cudaStream_t stream) {
  constexpr int V = Vec<T>::V;
  const EncLayout L = enc_layout(rows, cols);
  unsigned int* counters = reinterpret_cast<unsigned int*>(ws);
  double* sumsq_part = reinterpret_cast<double*>(ws + L.sumsq_part);
  double* encpart = reinterpret_cast<double*>(ws + L.encpart);
  if (reduce_over_rows) {
    const int64_t strips = (cols + 32 * V - 1) / (32 * V);
    const int chunk_rows = enc_chunk_rows(rows, strips, num_sms());
    const int64_t chunks = (rows + chunk_rows - 1) / chunk_rows;
    if (strips > 512 || chunks > 65535 || 8 * ld * (int64_t)sizeof(T) > 0xFFFFFFFFll) return GECC_EUNSUPPORTED;
    dim3 grid((unsigned)strips, (unsigned)chunks);
    encode_colsum_kernel<T><<<grid, 256, 0, stream>>>(dtype, X, rows, cols, ld, x_lo, parity, parity_lo, par64, sumsq, counters, sumsq_part, encpart, chunk_rows);
  } else {
    const int64_t want = (rows + 7) / 8, cap = 2 * (int64_t)num_sms();
    const unsigned grid = (unsigned)(want < cap ? want : cap);
    if ((size_t)grid * sizeof(double) > (size_t)kEncRowPartBytes) return GECC_EUNSUPPORTED;
    encode_rowsum_kernel<T><<<grid, 256, 0, stream>>>(dtype, X, rows, cols, ld, x_lo, parity, parity_lo, par64, sumsq, counters,
                                                       reinterpret_cast<double*>(ws + kCounterBytes));
  }
  return cudaGetLastError() == cudaSuccess ? GECC_OK : GECC_ECUDA;
}

int encode_dispatch(int dtype, bool reduce_over_rows, const void* X, int64_t rows, int64_t cols, int64_t ld, void* parity, float* parity_lo,
                    float* x_lo, double* par64, double* sumsq, uint8_t* ws, cudaStream_t stream) {
  if (dtype == GECC_BF16)
    return encode_typed<__nv_bfloat16>(dtype, reduce_over_rows, reinterpret_cast<const __nv_bfloat16*>(X), rows, cols, ld, parity, nullptr, nullptr,
                                       par64, sumsq, ws, stream);
  return encode_typed<float>(dtype, reduce_over_rows, reinterpret_cast<const float*>(X), rows, cols, ld, parity, parity_lo, x_lo, par64, sumsq, ws,
                             stream);
}


// ---------------------------------------------------------------------------------------------
// Both operands in ONE launch: the first blocks run the column-direction items, the others the row-direction rows, each
// operand in whichever direction its storage needs (A: over the storage rows unless stored transposed; B: along them
// unless stored transposed).  The two operands use separate arrival counters and scratch, so any combination of
// directions may run side by side; the block scheduler fills the SMs with blocks of either kind as slots come free.
// ---------------------------------------------------------------------------------------------
struct EncOperand {
  const void* X;
  int64_t rows, cols, ld;
  float* x_lo;
  void* parity;
  float* parity_lo;
  double* par64;
  double* sumsq;
  int over_rows;         // 1: column-direction reduction (checks per storage column), 0: one check pair per storage row
  int chunk_rows, strips, chunks;  // column direction
  int blocks;            // blocks of this operand in the launch
  unsigned int* ctr_strip;  // [strips] arrival counters, [1] all-blocks counter right after them
  double* sumsq_part;
  double* encpart;
};

template <typename T>
__global__ void __launch_bounds__(256, 2) encode_both_kernel(int dtype, const EncOperand a, const EncOperand b, unsigned int* counters) {
  __shared__ EncSmem<T> sm;
  // launched as a programmatic dependent itself: its blocks take their places while the kernel before it in the stream drains
  // (the decoder of the previous product, which lets its dependents go at once) and read nothing before that kernel has completed
  ptx::griddep_wait();
  ptx_griddep_launch_dependents();  // the product that follows may take its places as SMs come free; it waits for this grid
  if (blockIdx.x == 0 && threadIdx.x == 0) ws_enter(counters, "gecc_encode_both");
  const bool first = (int)blockIdx.x < a.blocks;
  const EncOperand& o = first ? a : b;
  const int blk = first ? (int)blockIdx.x : (int)blockIdx.x - a.blocks;
  const T* X = reinterpret_cast<const T*>(o.X);
  constexpr int V = Vec<T>::V;
  if (o.over_rows) {
    const int strip = blk % o.strips, chunk = blk / o.strips;
    const double qs = colsum_item<T>(X, o.rows, o.cols, o.ld, o.x_lo, o.encpart, strip, chunk, o.chunk_rows, sm);
    if (threadIdx.x == 0) o.sumsq_part[blk] = qs;
    if (arrive_last(o.ctr_strip + strip, o.chunks, sm.last)) {
      const int t = threadIdx.x;
      const int64_t c = (int64_t)strip * 32 * V + t;
      if (t < 32 * V && c < o.cols) {
        double s1, s2;
        colsum_combine(o.encpart, o.chunks, o.chunk_rows, o.cols, c, s1, s2);
        o.par64[c] = s1;
        o.par64[o.cols + c] = s2;
        if (o.parity) write_parity(dtype, o.parity, o.parity_lo, o.cols, c, s1, s2);
      }
    }
  } else {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    float q = 0.f;
#pragma unroll 1
    for (int64_t r = (int64_t)blk * 8 + w; r < o.rows; r += (int64_t)o.blocks * 8) {
      double S1, S2;
      rowsum_warp<T>(X + r * o.ld, o.cols, o.x_lo ? o.x_lo + r * o.ld : nullptr, S1, S2, q);
      if (lane == 0) {
        o.par64[r] = S1;
        o.par64[o.rows + r] = S2;
        if (o.parity) write_parity(dtype, o.parity, o.parity_lo, o.rows, r, S1, S2);
      }
    }
    const double qw = warp_sum((double)q);
    if (lane == 0) sm.sq[w] = qw;
    __syncthreads();
    if (threadIdx.x == 0) {
      double acc = 0.0;
#pragma unroll
      for (int g = 0; g < 8; ++g) acc += sm.sq[g];
      o.sumsq_part[blk] = acc;
    }
  }
  if (o.sumsq && arrive_last(o.ctr_strip + o.strips, o.blocks, sm.last)) {
    const double tot = block_sum_parts(o.sumsq_part, o.blocks, sm.sq);
    if (threadIdx.x == 0) *o.sumsq = tot;
  }
  __syncthreads();
  if (threadIdx.x == 0) ws_exit(counters, gridDim.x);
}

template <typename T>
static int fill_operand(EncOperand& o, bool over_rows, const void* X, int64_t rows, int64_t cols, int64_t ld, float* x_lo, void* parity, float* parity_lo,
                        double* par64, double* sumsq, unsigned int* ctr, double* sumsq_part, double* encpart) {
  constexpr int V = Vec<T>::V;
  o.X = X; o.rows = rows; o.cols = cols; o.ld = ld; o.x_lo = x_lo; o.parity = parity; o.parity_lo = parity_lo; o.par64 = par64; o.sumsq = sumsq;
  o.over_rows = over_rows ? 1 : 0;
  o.ctr_strip = ctr; o.sumsq_part = sumsq_part; o.encpart = encpart;
  o.chunk_rows = 0; o.chunks = 0;
  if (over_rows) {
    const int64_t strips = (cols + 32 * V - 1) / (32 * V);
    o.chunk_rows = enc_chunk_rows(rows, strips, num_sms());
    const int64_t chunks = (rows + o.chunk_rows - 1) / o.chunk_rows;
    if (strips > 255 || strips * chunks > 65535 || 8 * ld * (int64_t)sizeof(T) > 0xFFFFFFFFll) return GECC_EUNSUPPORTED;
    o.strips = (int)strips; o.chunks = (int)chunks; o.blocks = (int)(strips * chunks);
  } else {
    const int64_t want = (rows + 7) / 8, cap = 2 * (int64_t)num_sms();
    o.strips = 0;
    o.blocks = (int)(want < cap ? want : cap);
    if ((size_t)o.blocks * sizeof(double) > (size_t)kEncRowPartBytes / 2) return GECC_EUNSUPPORTED;
  }
  return GECC_OK;
}

template <typename T>
static int encode_both_typed(int dtype, bool a_over_rows, bool b_over_rows, const void* A, int64_t ra, int64_t ca, int64_t lda, void* A_par, float* A_par_lo,
                             float* A_lo, double* A_par64, double* sumsq_a, const void* B, int64_t rb, int64_t cb, int64_t ldb, void* B_par, float* B_par_lo,
                             float* B_lo, double* B_par64, double* sumsq_b, uint8_t* ws, double* encpart_b, cudaStream_t stream) {
  EncOperand a, b;
  unsigned int* counters = reinterpret_cast<unsigned int*>(ws);
  double* rowparts = reinterpret_cast<double*>(ws + kCounterBytes);  // [kEncRowPartBytes / 8]: first half A, second half B (row direction)
  const EncLayout La = enc_layout(ra, ca);
  int rc;
  if ((rc = fill_operand<T>(a, a_over_rows, A, ra, ca, lda, A_lo, A_par, A_par_lo, A_par64, sumsq_a, counters + kCtrEncStrip,
                            a_over_rows ? reinterpret_cast<double*>(ws + La.sumsq_part) : rowparts, reinterpret_cast<double*>(ws + La.encpart)))) return rc;
  // B: its own counters (second half of the strip range) and scratch (the region the decoder's verification of B^T uses)
  if ((rc = fill_operand<T>(b, b_over_rows, B, rb, cb, ldb, B_lo, B_par, B_par_lo, B_par64, sumsq_b, counters + kCtrEncStrip + 256,
                            rowparts + kEncRowPartBytes / 16, encpart_b))) return rc;
  // one wave of two blocks per SM in all: a row-direction operand takes the slots the other operand leaves
  const int slots = 2 * num_sms();
  if (!a_over_rows && b_over_rows) a.blocks = (int)std::min<int64_t>((ra + 7) / 8, std::max(slots - b.blocks, slots / 4));
  if (!b_over_rows && a_over_rows) b.blocks = (int)std::min<int64_t>((rb + 7) / 8, std::max(slots - a.blocks, slots / 4));
  if (!a_over_rows && !b_over_rows) { a.blocks = (int)std::min<int64_t>(a.blocks, slots / 2); b.blocks = (int)std::min<int64_t>(b.blocks, slots / 2); }
  if (b_over_rows && (size_t)b.blocks * sizeof(double) > (size_t)kEncRowPartBytes / 2) return GECC_EUNSUPPORTED;
  {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(a.blocks + b.blocks));
    cfg.blockDim = dim3(256);
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, encode_both_kernel<T>, dtype, a, b, counters) != cudaSuccess) return GECC_ECUDA;
  }
  return cudaGetLastError() == cudaSuccess ? GECC_OK : GECC_ECUDA;
}

int encode_both_dispatch(int dtype, bool a_over_rows, bool b_over_rows, const void* A, int64_t ra, int64_t ca, int64_t lda, void* A_par, float* A_par_lo, float* A_lo,
                         double* A_par64, double* sumsq_a, const void* B, int64_t rb, int64_t cb, int64_t ldb, void* B_par, float* B_par_lo, float* B_lo,
                         double* B_par64, double* sumsq_b, uint8_t* ws, double* encpart_b, cudaStream_t stream) {
  if (dtype == GECC_BF16)
    return encode_both_typed<__nv_bfloat16>(dtype, a_over_rows, b_over_rows, A, ra, ca, lda, A_par, nullptr, nullptr, A_par64, sumsq_a, B, rb, cb, ldb, B_par, nullptr,
                                            nullptr, B_par64, sumsq_b, ws, encpart_b, stream);
  return encode_both_typed<float>(dtype, a_over_rows, b_over_rows, A, ra, ca, lda, A_par, A_par_lo, A_lo, A_par64, sumsq_a, B, rb, cb, ldb, B_par, B_par_lo, B_lo,
                                  B_par64, sumsq_b, ws, encpart_b, stream);
}

// ---------------------------------------------------------------------------------------------
// gecc_encode_noalloc (include/gecc.h): the same encoder launch with its scratch in a fixed array of the device image
// instead of the caller's workspace.  In host code the array's name is only a stand-in for the symbol: the device address
// comes from cudaGetSymbolAddress, looked up once per device with that device current.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_noalloc_scratch[GECC_NOALLOC_SCRATCH_BYTES];

static int noalloc_scratch(uint8_t** out) {
  constexpr int kMaxDevices = 64;
  static std::mutex mu;
  static uint8_t* addr[kMaxDevices] = {};
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return GECC_ECUDA;
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    void* p = nullptr;
    if (cudaGetSymbolAddress(&p, g_noalloc_scratch) != cudaSuccess || !p) return GECC_ECUDA;
    addr[dev] = reinterpret_cast<uint8_t*>(p);
  }
  *out = addr[dev];
  return GECC_OK;
}

int encode_noalloc_dispatch(int dtype, bool reduce_over_rows, const void* X, int64_t rows, int64_t cols, int64_t ld, void* parity, float* parity_lo,
                            float* x_lo, double* par64, double* sumsq, cudaStream_t stream) {
  if (enc_layout(rows, cols).total > (size_t)GECC_NOALLOC_SCRATCH_BYTES) return GECC_ETOOLARGE;
  uint8_t* ws = nullptr;
  if (const int rc = noalloc_scratch(&ws)) return rc;
  // the array keeps what the last call left: the arrival counters must start at zero even if that call was cut short
  if (cudaMemsetAsync(ws, 0, kCounterBytes, stream) != cudaSuccess) return GECC_ECUDA;
  return encode_dispatch(dtype, reduce_over_rows, X, rows, cols, ld, parity, parity_lo, x_lo, par64, sumsq, ws, stream);
}

}  // namespace gecc
