// Encoded product C_bar = A_bar B_bar as one persistent, warp-specialised tcgen05 kernel.
//
//   warp 0 lane 0 : TMA producer   (global -> 128B-swizzled shared tiles, mbarrier pipeline)
//   warp 1 lane 0 : MMA issuer     (tcgen05.mma, accumulators in TMEM, two accumulator buffers)
//   warp 2        : TMEM allocator
//   warps 4..7    : epilogue       (TMEM -> registers -> shared -> coalesced global stores), with the row and
//                                   column sums of the detection step taken from the
//                                   accumulators on the way out, so C is never read back.
//
// The parity rows A_P and parity columns B_P are not copied next to A and B: they live in side
// buffers ([GECC_PAR_ROWS x k], K-major) and enter the product as one extra block row (128 x BN tiles whose A operand
// is A_P) and one extra block column (128 x 16 tiles whose B operand is B_P).  Their outputs are P_c, P_r, P_g.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>

#include "../../include/gecc.h"
#include "gecc_internal.h"
#include "sm100_ptx.cuh"

namespace gecc {

using namespace ptx;

template <int KIND>
struct Cfg;
template <>
struct Cfg<GECC_BF16> {
  static constexpr int ELT = 2, BK = 64, UK = 16, BN = 256, STAGES = 4, NPROD = 1;
  static constexpr uint32_t FMT = FMT_BF16;
};
template <>
struct Cfg<GECC_F32> {
  static constexpr int ELT = 4, BK = 32, UK = 8, BN = 128, STAGES = 3, NPROD = 3;
  static constexpr uint32_t FMT = FMT_TF32;
};

constexpr int BM = 128;
constexpr int PARN = 16;  // UMMA N of the parity block column (GECC_PAR_ROWS = 8 real columns)
constexpr int NUM_THREADS = 256;
constexpr int EPI_WARP0 = 4;
constexpr int STAGE_EPI_BYTES = 4 * 32 * 32 * 4;  // 4 warps x (32 rows x 32 fp32)

template <int KIND>
struct Smem {
  using C = Cfg<KIND>;
  static constexpr int A_BYTES = BM * 128;             // BM rows x 128 B (one swizzle row = BK elements)
  static constexpr int B_BYTES = C::BN * C::BK * C::ELT;
  static constexpr int NOPS = (KIND == GECC_F32) ? 2 : 1;  // hi and lo copies of each operand for 3xTF32
  static constexpr int STAGE_BYTES = NOPS * (A_BYTES + B_BYTES);
  static constexpr int PIPE_BYTES = C::STAGES * STAGE_BYTES;
  static constexpr int COLACC_BYTES = 4 * C::BN * 3 * 4;  // column sums of the four epilogue warps: [warp][column][sum, weighted, squares]
  static constexpr int TOTAL = 1024 /*alignment slack*/ + PIPE_BYTES + STAGE_EPI_BYTES + COLACC_BYTES + 256 /*barriers*/;
};

struct GemmParams {
  int n, k, m;
  int mb_data, nb_data;  // number of 128-row / BN-column blocks of the data part
  int protect;           // 1: parity tiles + epilogue sums
  float* C;
  int64_t ldc;
  float* P_r;      // [n x GECC_PR_LD]
  float* P_c;      // [GECC_PAR_ROWS x m]
  float* P_g;      // [GECC_PAR_ROWS x GECC_PR_LD]
  float* rowpart;  // [m / 128][n][4] : per row, per block of 128 columns: sum_j c, sum_j jl c, sum_j c^2, 0   (jl = column within the block)
  float* colpart;  // [n / 128][m][4] : per column, per block of 128 rows: sum_i c, sum_i il c, sum_i c^2, 0 (il = row within the block)
  const gecc_fault_t* inject;
  int n_inject;
};

template <int KIND>
__global__ void __launch_bounds__(NUM_THREADS, 1)
gecc_gemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                 const __grid_constant__ CUtensorMap tmAp, const __grid_constant__ CUtensorMap tmBp,
                 const __grid_constant__ CUtensorMap tmAlo, const __grid_constant__ CUtensorMap tmBlo,
                 const __grid_constant__ CUtensorMap tmAplo, const __grid_constant__ CUtensorMap tmBplo,
                 const GemmParams p) {
  using C = Cfg<KIND>;
  using S = Smem<KIND>;
  constexpr int BN = C::BN, BK = C::BK, STAGES = C::STAGES;
  constexpr int NBOX = BN / (128 / C::ELT);        // TMA boxes per B tile (each 128 B of n x BK rows of k)
  constexpr int BOX_BYTES = 128 * BK;              // bytes of one such box
  constexpr uint32_t TMEM_COLS = 2 * BN;           // two accumulator buffers
  constexpr uint32_t IDESC_DATA = make_idesc(C::FMT, 0, 1, BM, BN);
  constexpr uint32_t IDESC_PARN = make_idesc(C::FMT, 0, 0, BM, PARN);

  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t epi_base = smem_base + S::PIPE_BYTES;
  const uint32_t colacc_base = epi_base + STAGE_EPI_BYTES;
  const uint32_t bar_base = colacc_base + S::COLACC_BYTES;
  // barriers: full[STAGES], empty[STAGES], tmem_full[2], tmem_empty[2], then the TMEM base address word
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
  auto tfull_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + a); };
  auto tempty_bar = [&](int a) { return bar_base + 8u * (2 * STAGES + 2 + a); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 4);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int mbt = p.mb_data + p.protect, nbt = p.nb_data + p.protect;
  const int num_tiles = mbt * nbt;
  const int kblocks = (p.k + BK - 1) / BK;

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmA);
    prefetch_tmap(&tmB);
    if (p.protect) { prefetch_tmap(&tmAp); prefetch_tmap(&tmBp); }
  }
  if (warp == 1 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int a = 0; a < 2; ++a) { mbar_init(tfull_bar(a), 1); mbar_init(tempty_bar(a), 4); }
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc(tmem_slot, TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

  if (warp == 0) {
    if (lane == 0) {
      // ================= TMA producer =================
      int stage = 0;
      uint32_t phase = 0;
      for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
        const int nb = t / mbt, mb = t % mbt;
        const bool par_m = p.protect && mb == p.mb_data, par_n = p.protect && nb == p.nb_data;
        const uint32_t a_bytes = par_m ? GECC_PAR_ROWS * 128 : S::A_BYTES;
        const uint32_t b_bytes = par_n ? GECC_PAR_ROWS * 128 : S::B_BYTES;
        for (int kb = 0; kb < kblocks; ++kb) {
          mbar_wait(empty_bar(stage), phase ^ 1);
          const uint32_t sA = smem_base + stage * S::STAGE_BYTES;
          const uint32_t sB = sA + S::NOPS * S::A_BYTES;
          const uint32_t bar = full_bar(stage);
          mbar_expect_tx(bar, S::NOPS * (a_bytes + b_bytes));
          const int k0 = kb * BK;
          if (par_m) tma_load_2d(sA, &tmAp, bar, k0, 0);
          else       tma_load_2d(sA, &tmA, bar, k0, mb * BM);
          if (par_n) tma_load_2d(sB, &tmBp, bar, k0, 0);
          else {
#pragma unroll
            for (int b = 0; b < NBOX; ++b) tma_load_2d(sB + b * BOX_BYTES, &tmB, bar, nb * BN + b * (128 / C::ELT), k0);
          }
          if (KIND == GECC_F32) {
            const uint32_t sAl = sA + S::A_BYTES, sBl = sB + S::B_BYTES;
            if (par_m) tma_load_2d(sAl, &tmAplo, bar, k0, 0);
            else       tma_load_2d(sAl, &tmAlo, bar, k0, mb * BM);
            if (par_n) tma_load_2d(sBl, &tmBplo, bar, k0, 0);
            else {
#pragma unroll
              for (int b = 0; b < NBOX; ++b) tma_load_2d(sBl + b * BOX_BYTES, &tmBlo, bar, nb * BN + b * (128 / C::ELT), k0);
            }
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {
      // ================= MMA issuer =================
      int stage = 0;
      uint32_t phase = 0;
      int acc = 0;
      uint32_t acc_phase = 0;
      for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
        const int nb = t / mbt;
        const bool par_n = p.protect && nb == p.nb_data;
        const uint32_t idesc = par_n ? IDESC_PARN : IDESC_DATA;
        mbar_wait(tempty_bar(acc), acc_phase ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * BN;
        for (int kb = 0; kb < kblocks; ++kb) {
          mbar_wait(full_bar(stage), phase);
          tc_fence_after();
          const uint32_t sA = smem_base + stage * S::STAGE_BYTES;
          const uint32_t sB = sA + S::NOPS * S::A_BYTES;
          // A: K-major, 8-row groups 1024 B apart.  B data: MN-major, 128 B of n per row of k, 8-row k groups 1024 B
          // apart (SBO), 128-byte n groups BOX_BYTES apart (LBO).  B parity: K-major like A.
          const uint64_t a_hi = smem_desc_sw128(sA, 16, 1024);
          const uint64_t b_hi = par_n ? smem_desc_sw128(sB, 16, 1024)
                                : (KIND == GECC_BF16 ? smem_desc_sw128(sB, BOX_BYTES, 1024) : smem_desc_sw128_base32(sB, BOX_BYTES, 512));
          const uint32_t a_step = (C::UK * C::ELT) >> 4;                       // 32 B along K inside the swizzle row
          const uint32_t b_step = par_n ? a_step : ((C::UK * 128) >> 4);       // UK rows of k
#pragma unroll
          for (int ks = 0; ks < BK / C::UK; ++ks) {
            const uint32_t accum = (kb | ks) ? 1u : 0u;
            if (KIND == GECC_BF16) {
              mma_bf16(d_tmem, a_hi + ks * a_step, b_hi + ks * b_step, idesc, accum);
            } else {
              // 3xTF32: a b ~ a_hi b_hi + a_hi b_lo + a_lo b_hi, small terms first
              const uint64_t a_lo = a_hi + (S::A_BYTES >> 4), b_lo = b_hi + (S::B_BYTES >> 4);
              mma_tf32(d_tmem, a_lo + ks * a_step, b_hi + ks * b_step, idesc, accum);
              mma_tf32(d_tmem, a_hi + ks * a_step, b_lo + ks * b_step, idesc, 1u);
              mma_tf32(d_tmem, a_hi + ks * a_step, b_hi + ks * b_step, idesc, 1u);
            }
          }
          mma_commit(empty_bar(stage));
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        mma_commit(tfull_bar(acc));
        if (++acc == 2) { acc = 0; acc_phase ^= 1; }
      }
    }
  } else if (warp >= EPI_WARP0) {
    // ================= epilogue =================
    const int wq = warp - EPI_WARP0;  // TMEM lane quarter this warp may read: lanes 32 wq .. 32 wq + 31
    const uint32_t stg = epi_base + wq * (32 * 32 * 4);
    int acc = 0;
    uint32_t acc_phase = 0;
    for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
      const int nb = t / mbt, mb = t % mbt;
      const bool par_m = p.protect && mb == p.mb_data, par_n = p.protect && nb == p.nb_data;
      const bool reduce = p.protect && !par_m && !par_n;
      // where this tile goes
      float* out;
      int64_t ld;
      int rows_valid, cols_valid;
      if (!par_m && !par_n) { out = p.C + (int64_t)mb * BM * p.ldc + (int64_t)nb * BN; ld = p.ldc; rows_valid = p.n - mb * BM; cols_valid = p.m - nb * BN; }
      else if (par_m && !par_n) { out = p.P_c + (int64_t)nb * BN; ld = p.m; rows_valid = GECC_PAR_ROWS; cols_valid = p.m - nb * BN; }
      else if (!par_m) { out = p.P_r + (int64_t)mb * BM * GECC_PR_LD; ld = GECC_PR_LD; rows_valid = p.n - mb * BM; cols_valid = GECC_PR_LD; }
      else { out = p.P_g; ld = GECC_PR_LD; rows_valid = GECC_PAR_ROWS; cols_valid = GECC_PR_LD; }
      const int nchunks = par_n ? 1 : BN / 32;
      const int my_row = mb * BM + wq * 32 + lane;  // global row of C this thread's TMEM lane holds

      mbar_wait(tfull_bar(acc), acc_phase);
      tc_fence_after();
      float s1 = 0.f, s2 = 0.f, ss = 0.f;
      for (int c = 0; c < nchunks; ++c) {
        uint32_t v[32];
        tmem_ld32(tmem_base + acc * BN + c * 32 + ((uint32_t)(wq * 32) << 16), v);
        tmem_ld_wait();
        if (c == nchunks - 1) {  // accumulator buffer fully read: hand it back to the MMA warp
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(tempty_bar(acc));
        }
        if (p.n_inject > 0 && !par_m && !par_n) {  // E3: fault on a symbol of C during its computation
          for (int f = 0; f < p.n_inject; ++f) {
            const gecc_fault_t ft = p.inject[f];
            const int cc = ft.col - (nb * BN + c * 32);
            if (ft.kind == GECC_KIND_C && ft.row == my_row && cc >= 0 && cc < 32) {
#pragma unroll
              for (int q = 0; q < 32; ++q)
                if (q == cc) v[q] = __float_as_uint(__uint_as_float(v[q]) + ft.value);
            }
          }
        }
        if (reduce) {  // row sums of PAPER.md:194,196 over this block column, local weights
#pragma unroll
          for (int q = 0; q < 32; ++q) {
            const float x = __uint_as_float(v[q]);
            s1 += x;
            s2 = fmaf((float)((c & 3) * 32 + q), x, s2);
            ss = fmaf(x, x, ss);  // line energy: scales the line's threshold (rounding noise is relative)
          }
        }
        // registers -> shared, 16-byte chunks XOR-swizzled by row so both directions are conflict-free
#pragma unroll
        for (int c4 = 0; c4 < 8; ++c4) {
          const uint32_t addr = stg + lane * 128 + ((c4 ^ (lane & 7)) << 4);
          asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v[4 * c4]), "r"(v[4 * c4 + 1]), "r"(v[4 * c4 + 2]), "r"(v[4 * c4 + 3]) : "memory");
        }
        __syncwarp();
        float cs1[4] = {0.f, 0.f, 0.f, 0.f}, cs2[4] = {0.f, 0.f, 0.f, 0.f}, css[4] = {0.f, 0.f, 0.f, 0.f};
        const int c4 = lane & 7;
        const int col = c * 32 + 4 * c4;  // column within the tile
#pragma unroll
        for (int it = 0; it < 8; ++it) {
          const int r = it * 4 + (lane >> 3);
          const uint32_t addr = stg + r * 128 + ((c4 ^ (r & 7)) << 4);
          float4 x;
          asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(x.x), "=f"(x.y), "=f"(x.z), "=f"(x.w) : "r"(addr) : "memory");
          if (wq * 32 + r < rows_valid && col < cols_valid)
            *reinterpret_cast<float4*>(out + (int64_t)(wq * 32 + r) * ld + col) = x;
          if (reduce) {  // column sums of PAPER.md:198,200 over this 32-row slab, local weights
            const float w = (float)r;
            cs1[0] += x.x; cs1[1] += x.y; cs1[2] += x.z; cs1[3] += x.w;
            cs2[0] = fmaf(w, x.x, cs2[0]); cs2[1] = fmaf(w, x.y, cs2[1]); cs2[2] = fmaf(w, x.z, cs2[2]); cs2[3] = fmaf(w, x.w, cs2[3]);
            css[0] = fmaf(x.x, x.x, css[0]); css[1] = fmaf(x.y, x.y, css[1]); css[2] = fmaf(x.z, x.z, css[2]); css[3] = fmaf(x.w, x.w, css[3]);
          }
        }
        if (reduce) {
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            cs1[e] += __shfl_xor_sync(0xffffffffu, cs1[e], 8);
            cs2[e] += __shfl_xor_sync(0xffffffffu, cs2[e], 8);
            cs1[e] += __shfl_xor_sync(0xffffffffu, cs1[e], 16);
            cs2[e] += __shfl_xor_sync(0xffffffffu, cs2[e], 16);
            css[e] += __shfl_xor_sync(0xffffffffu, css[e], 8);
            css[e] += __shfl_xor_sync(0xffffffffu, css[e], 16);
          }
          if (lane < 8) {
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const uint32_t a = colacc_base + ((wq * BN + col + e) * 3) * 4;
              asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(cs1[e]) : "memory");
              asm volatile("st.shared.f32 [%0], %1;" ::"r"(a + 4), "f"(cs2[e]) : "memory");
              asm volatile("st.shared.f32 [%0], %1;" ::"r"(a + 8), "f"(css[e]) : "memory");
            }
          }
          if ((c & 3) == 3) {  // 128 columns done: one row partial (weights local to the block of 128 columns)
            if (my_row < p.n && nb * BN + (c & ~3) * 32 < p.m)
              *reinterpret_cast<float4*>(p.rowpart + ((int64_t)((nb * BN + c * 32) / kSumCols) * p.n + my_row) * 4) = make_float4(s1, s2, ss, 0.f);
            s1 = 0.f; s2 = 0.f; ss = 0.f;
          }
        }
        __syncwarp();
      }
      if (reduce) {
        // column sums of the 128-row tile: add the four warps' 32-row slabs (slab w carries the row offset 32 w)
        asm volatile("bar.sync 1, 128;" ::: "memory");
        for (int cc = threadIdx.x - EPI_WARP0 * 32; cc < BN; cc += 128) {
          float a = 0.f, b = 0.f, e2 = 0.f;
#pragma unroll
          for (int w4 = 0; w4 < 4; ++w4) {
            float x1, x2, x3;
            const uint32_t ad = colacc_base + ((w4 * BN + cc) * 3) * 4;
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(x1) : "r"(ad) : "memory");
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(x2) : "r"(ad + 4) : "memory");
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(x3) : "r"(ad + 8) : "memory");
            a += x1;
            b += fmaf((float)(32 * w4), x1, x2);
            e2 += x3;
          }
          const int gcol = nb * BN + cc;
          if (gcol < p.m) *reinterpret_cast<float4*>(p.colpart + ((int64_t)mb * p.m + gcol) * 4) = make_float4(a, b, e2, 0.f);
        }
        asm volatile("bar.sync 1, 128;" ::: "memory");
      }
      if (++acc == 2) { acc = 0; acc_phase ^= 1; }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem_base, TMEM_COLS);
}

// ------------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (fn) return fn;
  void* sym = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) != cudaSuccess || qres != cudaDriverEntryPointSuccess)
    return nullptr;
  fn = reinterpret_cast<EncodeTiledFn>(sym);
  return fn;
}

// 2-D row-major tensor [outer x inner] with leading dimension ld (elements); box = {box_inner, box_outer}; 128 B swizzle.
static int make_tmap(CUtensorMap* tm, int kind, const void* ptr, int64_t inner, int64_t outer, int64_t ld, int box_inner, int box_outer,
                     CUtensorMapSwizzle swz = CU_TENSOR_MAP_SWIZZLE_128B) {
  EncodeTiledFn fn = get_encode_fn();
  if (!fn) return GECC_ECUDA;
  const int elt = (kind == GECC_BF16) ? 2 : 4;
  cuuint64_t dims[2] = {(cuuint64_t)inner, (cuuint64_t)outer};
  cuuint64_t strides[1] = {(cuuint64_t)ld * elt};
  cuuint32_t box[2] = {(cuuint32_t)box_inner, (cuuint32_t)box_outer};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(tm, kind == GECC_BF16 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(ptr), dims,
                  strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, swz, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    fprintf(stderr, "gecc: cuTensorMapEncodeTiled failed (%d) inner=%lld outer=%lld ld=%lld box=%dx%d\n", (int)r, (long long)inner,
            (long long)outer, (long long)ld, box_inner, box_outer);
    return GECC_ECUDA;
  }
  return GECC_OK;
}

int num_sms() {
  static int sms = 0;
  if (!sms) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) sms = 0;
  }
  return sms;
}

template <int KIND>
static int launch_gemm(bool protect, int64_t n, int64_t k, int64_t m, const void* A, int64_t lda, const void* A_par, const float* A_lo,
                       const float* A_par_lo, const void* B, int64_t ldb, const void* B_par, const float* B_lo, const float* B_par_lo,
                       float* Cout, int64_t ldc, float* P_r, float* P_c, float* P_g, const gecc_fault_t* inject, int n_inject,
                       float* rowpart, float* colpart, cudaStream_t stream) {
  using C = Cfg<KIND>;
  using S = Smem<KIND>;
  CUtensorMap tmA, tmB, tmAp, tmBp, tmAlo, tmBlo, tmAplo, tmBplo;
  int rc;
  const int nsw = 128 / C::ELT;  // elements per 128-byte swizzle row
  if ((rc = make_tmap(&tmA, KIND, A, k, n, lda, C::BK, BM))) return rc;
  // MN-major operand: 16-bit elements take the plain 128B swizzle, 32-bit elements the 32-byte-atom variant
  const CUtensorMapSwizzle swzB = KIND == GECC_BF16 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B;
  if ((rc = make_tmap(&tmB, KIND, B, m, k, ldb, nsw, C::BK, swzB))) return rc;
  tmAp = tmA; tmBp = tmB; tmAlo = tmA; tmBlo = tmB; tmAplo = tmA; tmBplo = tmB;
  if (protect) {
    if ((rc = make_tmap(&tmAp, KIND, A_par, k, GECC_PAR_ROWS, k, C::BK, GECC_PAR_ROWS))) return rc;
    if ((rc = make_tmap(&tmBp, KIND, B_par, k, GECC_PAR_ROWS, k, C::BK, GECC_PAR_ROWS))) return rc;
  }
  if (KIND == GECC_F32) {
    if ((rc = make_tmap(&tmAlo, KIND, A_lo, k, n, lda, C::BK, BM))) return rc;
    if ((rc = make_tmap(&tmBlo, KIND, B_lo, m, k, ldb, nsw, C::BK, swzB))) return rc;
    tmAplo = tmAlo; tmBplo = tmBlo;
    if (protect) {
      if ((rc = make_tmap(&tmAplo, KIND, A_par_lo, k, GECC_PAR_ROWS, k, C::BK, GECC_PAR_ROWS))) return rc;
      if ((rc = make_tmap(&tmBplo, KIND, B_par_lo, k, GECC_PAR_ROWS, k, C::BK, GECC_PAR_ROWS))) return rc;
    }
  }
  GemmParams p;
  p.n = (int)n; p.k = (int)k; p.m = (int)m;
  p.mb_data = (int)((n + BM - 1) / BM);
  p.nb_data = (int)((m + C::BN - 1) / C::BN);
  p.protect = protect ? 1 : 0;
  p.C = Cout; p.ldc = ldc; p.P_r = P_r; p.P_c = P_c; p.P_g = P_g;
  p.rowpart = rowpart; p.colpart = colpart;
  p.inject = inject; p.n_inject = inject ? n_inject : 0;
  const int tiles = (p.mb_data + p.protect) * (p.nb_data + p.protect);
  const int sms = num_sms();
  if (sms <= 0) return GECC_ECUDA;
  static bool attr_set = false;
  if (!attr_set) {
    if (cudaFuncSetAttribute(gecc_gemm_kernel<KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize, S::TOTAL) != cudaSuccess) return GECC_ECUDA;
    attr_set = true;
  }
  const int grid = tiles < sms ? tiles : sms;
  gecc_gemm_kernel<KIND><<<grid, NUM_THREADS, S::TOTAL, stream>>>(tmA, tmB, tmAp, tmBp, tmAlo, tmBlo, tmAplo, tmBplo, p);
  return cudaGetLastError() == cudaSuccess ? GECC_OK : GECC_ECUDA;
}

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

int gemm_dispatch(bool protect, int dtype, int64_t n, int64_t k, int64_t m, const void* A, int64_t lda, const void* A_par, const float* A_lo,
                  const float* A_par_lo, const void* B, int64_t ldb, const void* B_par, const float* B_lo, const float* B_par_lo, float* C,
                  int64_t ldc, float* P_r, float* P_c, float* P_g, const gecc_fault_t* inject, int n_inject, float* rowpart, float* colpart,
                  cudaStream_t stream) {
  if (dtype != GECC_BF16 && dtype != GECC_F32) return GECC_EUNSUPPORTED;
  if (!A || !B || !C || n <= 0 || k <= 0 || m <= 0 || n > (1 << 30) || k > (1 << 30) || m > (1 << 30)) return GECC_EINVAL;
  const int epr = dtype == GECC_BF16 ? 8 : 4;  // elements per 16 bytes
  if (lda < k || ldb < m || ldc < m || lda % epr || ldb % epr || ldc % 4 || m % 4 || k % epr) return GECC_EINVAL;
  if (!aligned16(A) || !aligned16(B) || !aligned16(C)) return GECC_EINVAL;
  if (dtype == GECC_F32 && (!A_lo || !B_lo || !aligned16(A_lo) || !aligned16(B_lo))) return GECC_EINVAL;
  if (protect) {
    if (!A_par || !B_par || !P_r || !P_c || !P_g || !rowpart || !colpart) return GECC_EINVAL;
    if (!aligned16(A_par) || !aligned16(B_par) || !aligned16(P_r) || !aligned16(P_c) || !aligned16(P_g)) return GECC_EINVAL;
    if (dtype == GECC_F32 && (!A_par_lo || !B_par_lo)) return GECC_EINVAL;
    if (n_inject < 0 || (n_inject > 0 && !inject)) return GECC_EINVAL;
  }
  if (dtype == GECC_BF16)
    return launch_gemm<GECC_BF16>(protect, n, k, m, A, lda, A_par, A_lo, A_par_lo, B, ldb, B_par, B_lo, B_par_lo, C, ldc, P_r, P_c, P_g, inject,
                                  n_inject, rowpart, colpart, stream);
  return launch_gemm<GECC_F32>(protect, n, k, m, A, lda, A_par, A_lo, A_par_lo, B, ldb, B_par, B_lo, B_par_lo, C, ldc, P_r, P_c, P_g, inject,
                               n_inject, rowpart, colpart, stream);
}

}  // namespace gecc
