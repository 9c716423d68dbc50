// extern "C" entry points of libgecc (declared and documented in include/gecc.h): argument checks, workspace
// carving, dispatch.  No computation happens here.
#include <cuda_runtime.h>

#include "../../include/gecc.h"
#include "gecc_internal.h"

namespace gecc {
int decode_dispatch(int dtype, int64_t n, int64_t k, int64_t m, float* C, int64_t ldc, float* P_r, float* P_c, const float* P_g, const double* tau,
                    const double* sumsq_a, const double* sumsq_b, int level, int trans_a, int trans_b, void* A, int64_t lda, float* A_lo, const double* A_par64,
                    void* B, int64_t ldb, float* B_lo, const double* B_par64, gecc_report_t* report, uint8_t* ws, const WsLayout& L, cudaStream_t stream);
int tl_encode_dispatch(int dtype, int64_t n, int64_t k, int64_t m, const void* A, int64_t lda, float* A_lo, void* A_PL, float* A_PL_lo, double* sumsq_a,
                       const void* B, int64_t ldb, float* B_lo, void* B_PL, float* B_PL_lo, double* sumsq_b, uint8_t* ws, cudaStream_t stream);
int tl_decode_dispatch(int dtype, int64_t n, int64_t k, int64_t m, float* C, int64_t ldc, const float* PrL, int64_t ldprl, const float* PcL, int64_t ldpcl,
                       const double* tau, const double* sumsq_a, const double* sumsq_b, int mode, gecc_tl_report_t* report, uint8_t* ws, const WsLayout& L,
                       cudaStream_t stream);
__global__ void inject_inputs_kernel(int dtype, int trans_a, int trans_b, void* A, int64_t lda, float* A_lo, void* B, int64_t ldb, float* B_lo, const gecc_fault_t* faults,
                                     int n_faults);
}  // namespace gecc

using namespace gecc;

static bool dtype_ok(int dtype) { return dtype == GECC_BF16 || dtype == GECC_F32; }
constexpr int64_t kMaxDim = 1ll << 30;  // sizes are narrowed to int inside the kernels
static bool al16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

extern "C" {

const char* gecc_version(void) { return "gecc 0.1 (sm_100a)"; }

size_t gecc_workspace_bytes(int dtype, int64_t n, int64_t k, int64_t m) {
  if (!dtype_ok(dtype) || n <= 0 || k <= 0 || m <= 0) return 0;
  return ws_layout(dtype, n, k, m).total;
}

int gecc_encode(int dtype, int side, int trans, const void* X, int64_t rows, int64_t cols, int64_t ld, void* parity, float* parity_lo, float* x_lo,
                double* parity64, double* sumsq, void* workspace, size_t workspace_bytes, void* stream) {
  if (!dtype_ok(dtype)) return GECC_EUNSUPPORTED;
  if (side != GECC_LEFT && side != GECC_RIGHT) return GECC_EINVAL;
  if (!X || !parity || !parity64 || !workspace || rows <= 0 || cols <= 0 || ld < cols) return GECC_EINVAL;
  const int epr = dtype == GECC_BF16 ? 8 : 4;
  if (ld % epr || cols % epr || !al16(X) || !al16(parity)) return GECC_EINVAL;
  if (dtype == GECC_F32 && (!parity_lo || !x_lo || !al16(x_lo))) return GECC_EINVAL;
  // counters and encoder scratch sit at the start of the workspace (enc_layout: a function of this operand's shape only)
  if (workspace_bytes < enc_layout(rows, cols).total) return GECC_EWORKSPACE;
  return encode_dispatch(dtype, (side == GECC_LEFT) != (trans != 0), X, rows, cols, ld, parity, parity_lo, x_lo, parity64, sumsq, reinterpret_cast<uint8_t*>(workspace),
                         reinterpret_cast<cudaStream_t>(stream));
}

int gecc_encode_noalloc(int dtype, int side, int trans, const void* X, int64_t rows, int64_t cols, int64_t ld, void* parity, float* parity_lo, float* x_lo,
                        double* parity64, double* sumsq, void* stream) {
  if (!dtype_ok(dtype)) return GECC_EUNSUPPORTED;
  if (side != GECC_LEFT && side != GECC_RIGHT) return GECC_EINVAL;
  if (!X || !parity || !parity64 || rows <= 0 || cols <= 0 || ld < cols) return GECC_EINVAL;
  const int epr = dtype == GECC_BF16 ? 8 : 4;
  if (ld % epr || cols % epr || !al16(X) || !al16(parity)) return GECC_EINVAL;
  if (dtype == GECC_F32 && (!parity_lo || !x_lo || !al16(x_lo))) return GECC_EINVAL;
  return encode_noalloc_dispatch(dtype, (side == GECC_LEFT) != (trans != 0), X, rows, cols, ld, parity, parity_lo, x_lo, parity64, sumsq,
                                 reinterpret_cast<cudaStream_t>(stream));
}

int gecc_encode_both(int dtype, int64_t n, int64_t k, int64_t m, int trans_a, int trans_b, const void* A, int64_t lda, void* A_par, float* A_par_lo, float* A_lo,
                     double* A_par64, double* sumsq_a, const void* B, int64_t ldb, void* B_par, float* B_par_lo, float* B_lo, double* B_par64, double* sumsq_b,
                     void* workspace, size_t workspace_bytes, void* stream) {
  if (!dtype_ok(dtype)) return GECC_EUNSUPPORTED;
  if (!A || !B || !A_par || !B_par || !A_par64 || !B_par64 || !workspace || n <= 0 || k <= 0 || m <= 0) return GECC_EINVAL;
  if (n > kMaxDim || k > kMaxDim || m > kMaxDim) return GECC_EINVAL;
  const int64_t ra = trans_a ? k : n, ca = trans_a ? n : k, rb = trans_b ? m : k, cb = trans_b ? k : m;  // storage shapes
  const int epr = dtype == GECC_BF16 ? 8 : 4;
  if (lda < ca || ldb < cb || lda % epr || ldb % epr || ca % epr || cb % epr || !al16(A) || !al16(B) || !al16(A_par) || !al16(B_par)) return GECC_EINVAL;
  if (dtype == GECC_F32 && (!A_par_lo || !B_par_lo || !A_lo || !B_lo || !al16(A_lo) || !al16(B_lo))) return GECC_EINVAL;
  const WsLayout L = ws_layout(dtype, n, k, m);
  if (workspace_bytes < L.total) return GECC_EWORKSPACE;
  uint8_t* ws = reinterpret_cast<uint8_t*>(workspace);
  return encode_both_dispatch(dtype, !trans_a, trans_b != 0, A, ra, ca, lda, A_par, A_par_lo, A_lo, A_par64, sumsq_a, B, rb, cb, ldb, B_par, B_par_lo, B_lo, B_par64,
                              sumsq_b, ws, reinterpret_cast<double*>(ws + L.encpart_b), reinterpret_cast<cudaStream_t>(stream));
}

int gecc_matmul_protected(int dtype, int64_t n, int64_t k, int64_t m, int trans_a, int trans_b, const void* A, int64_t lda, const void* A_par, const float* A_lo,
                          const float* A_par_lo, const void* B, int64_t ldb, const void* B_par, const float* B_lo, const float* B_par_lo, float* C,
                          int64_t ldc, float* P_r, float* P_c, float* P_g, const gecc_fault_t* inject, int n_inject, const double* tau,
                          const double* sumsq_a, const double* sumsq_b, gecc_report_t* report, int mode, void* workspace, size_t workspace_bytes,
                          void* stream) {
  if (!dtype_ok(dtype)) return GECC_EUNSUPPORTED;
  if (!workspace || n <= 0 || k <= 0 || m <= 0) return GECC_EINVAL;
  const WsLayout L = ws_layout(dtype, n, k, m);
  if (workspace_bytes < L.total) return GECC_EWORKSPACE;
  uint8_t* ws = reinterpret_cast<uint8_t*>(workspace);
  DetectArgs det;
  det.detect = tau != nullptr || (sumsq_a != nullptr && sumsq_b != nullptr);  // thresholds known: detect inside the product
  det.single = (mode & GECC_SINGLE_CHECKSUM) != 0;
  det.tau = tau; det.sumsq_a = sumsq_a; det.sumsq_b = sumsq_b;
  det.syn = reinterpret_cast<double*>(ws + L.syn);
  det.flags = ws + L.flags;
  det.st = reinterpret_cast<DecodeState*>(ws + L.state);
  det.counters = reinterpret_cast<unsigned int*>(ws);
  det.arrive = reinterpret_cast<unsigned int*>(ws + L.arrive);
  det.lineacc = reinterpret_cast<double*>(ws + L.lineacc);
  det.report = report;
  return gemm_dispatch(true, dtype, n, k, m, trans_a != 0, trans_b != 0, A, lda, A_par, A_lo, A_par_lo, B, ldb, B_par, B_lo, B_par_lo, C, ldc, P_r, P_c, P_g, inject, n_inject,
                       reinterpret_cast<float*>(ws + L.rowpart), reinterpret_cast<float*>(ws + L.colpart), &det, true, reinterpret_cast<cudaStream_t>(stream));
}

int gecc_matmul_plain(int dtype, int64_t n, int64_t k, int64_t m, int trans_a, int trans_b, const void* A, int64_t lda, const float* A_lo, const void* B, int64_t ldb,
                      const float* B_lo, float* C, int64_t ldc, void* stream) {
  if (!dtype_ok(dtype)) return GECC_EUNSUPPORTED;
  return gemm_dispatch(false, dtype, n, k, m, trans_a != 0, trans_b != 0, A, lda, nullptr, A_lo, nullptr, B, ldb, nullptr, B_lo, nullptr, C, ldc, nullptr, nullptr, nullptr,
                       nullptr, 0, nullptr, nullptr, nullptr, false, reinterpret_cast<cudaStream_t>(stream));
}

int gecc_syndrome_unfused(int dtype, int64_t n, int64_t k, int64_t m, const float* C, int64_t ldc, void* workspace, size_t workspace_bytes,
                          void* stream) {
  if (!dtype_ok(dtype)) return GECC_EUNSUPPORTED;
  if (!C || !workspace || n <= 0 || m <= 0 || ldc < m || ldc % 4 || m % 4 || !al16(C)) return GECC_EINVAL;
  if (k <= 0 || n > kMaxDim || k > kMaxDim || m > kMaxDim) return GECC_EINVAL;
  const WsLayout L = ws_layout(dtype, n, k, m);  // the same layout the product and the decoder use
  if (workspace_bytes < L.total) return GECC_EWORKSPACE;
  uint8_t* ws = reinterpret_cast<uint8_t*>(workspace);
  return syndrome_unfused_dispatch(n, m, C, ldc, reinterpret_cast<float*>(ws + L.rowpart), reinterpret_cast<float*>(ws + L.colpart),
                                   reinterpret_cast<DecodeState*>(ws + L.state), reinterpret_cast<cudaStream_t>(stream));
}

int gecc_decode_correct(int dtype, int64_t n, int64_t k, int64_t m, float* C, int64_t ldc, float* P_r, float* P_c, const float* P_g, const double* tau,
                        const double* sumsq_a, const double* sumsq_b, int level, int trans_a, int trans_b, void* A, int64_t lda, float* A_lo,
                        const double* A_par64, void* B, int64_t ldb, float* B_lo, const double* B_par64, gecc_report_t* report, void* workspace,
                        size_t workspace_bytes, void* stream) {
  if (!dtype_ok(dtype)) return GECC_EUNSUPPORTED;
  if (!C || !P_r || !P_c || !report || !workspace || n <= 0 || k <= 0 || m <= 0 || ldc < m) return GECC_EINVAL;
  if (n > kMaxDim || k > kMaxDim || m > kMaxDim) return GECC_EINVAL;
  if (!tau && (!sumsq_a || !sumsq_b)) return GECC_EINVAL;
  if (!al16(P_r)) return GECC_EINVAL;
  if (level < 0 || level > (GECC_LEVEL_X | GECC_SINGLE_CHECKSUM)) return GECC_EINVAL;
  if ((level & GECC_LEVEL_X) && !(level & GECC_SINGLE_CHECKSUM)) {
    if (!A || !B || !A_par64 || !B_par64 || lda < (trans_a ? n : k) || ldb < (trans_b ? k : m)) return GECC_EINVAL;
    if (dtype == GECC_F32 && (!A_lo || !B_lo)) return GECC_EINVAL;
    // the verification pass and the line recomputation read A and B with 16-byte vector loads: the common rules of gecc.h
    const int epr = dtype == GECC_BF16 ? 8 : 4;
    if (!al16(A) || !al16(B) || lda % epr || ldb % epr || k % epr || (trans_a && n % epr) || (!trans_b && m % epr)) return GECC_EINVAL;
    if (dtype == GECC_F32 && (!al16(A_lo) || !al16(B_lo))) return GECC_EINVAL;
  }
  const WsLayout L = ws_layout(dtype, n, k, m);
  if (workspace_bytes < L.total) return GECC_EWORKSPACE;
  return decode_dispatch(dtype, n, k, m, C, ldc, P_r, P_c, P_g, tau, sumsq_a, sumsq_b, level, trans_a != 0, trans_b != 0, A, lda, A_lo, A_par64, B, ldb, B_lo, B_par64, report,
                         reinterpret_cast<uint8_t*>(workspace), L, reinterpret_cast<cudaStream_t>(stream));
}

int gecc_recompute_fallback(int dtype, int64_t n, int64_t k, int64_t m, int trans_a, int trans_b, const void* A, int64_t lda, const float* A_lo, const void* B,
                            int64_t ldb, const float* B_lo, float* C, int64_t ldc, float* P_r, float* P_c, const double* tau, const double* sumsq_a,
                            const double* sumsq_b, gecc_report_t* report, void* workspace, size_t workspace_bytes, void* stream) {
  if (!dtype_ok(dtype)) return GECC_EUNSUPPORTED;
  if (!A || !B || !C || !P_r || !P_c || !report || !workspace || n <= 0 || k <= 0 || m <= 0) return GECC_EINVAL;
  if (!tau && (!sumsq_a || !sumsq_b)) return GECC_EINVAL;
  const WsLayout L = ws_layout(dtype, n, k, m);
  if (workspace_bytes < L.total) return GECC_EWORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  uint8_t* ws = reinterpret_cast<uint8_t*>(workspace);
  gecc_report_t rep;
  if (cudaStreamSynchronize(st) != cudaSuccess) return GECC_ECUDA;
  if (cudaMemcpy(&rep, report, sizeof(rep), cudaMemcpyDeviceToHost) != cudaSuccess) return GECC_ECUDA;
  if (rep.verdict != GECC_UNCORRECTABLE) return 0;
  // the flag bytes the decoder left: which rows / columns of C fail their checks
  const size_t n16 = ((size_t)n + 15) & ~(size_t)15;
  uint8_t* flags = new uint8_t[n16 + (size_t)m];
  if (cudaMemcpy(flags, ws + L.flags, n16 + (size_t)m, cudaMemcpyDeviceToHost) != cudaSuccess) { delete[] flags; return GECC_ECUDA; }
  constexpr int64_t kBlk = 256;
  const int64_t nrb = (n + kBlk - 1) / kBlk, ncb = (m + kBlk - 1) / kBlk;
  bool* rb = new bool[nrb + ncb]();
  bool* cb = rb + nrb;
  int64_t nr = 0, nc = 0;
  for (int64_t i = 0; i < n; ++i) if (flags[i] && !rb[i / kBlk]) { rb[i / kBlk] = true; ++nr; }
  for (int64_t j = 0; j < m; ++j) if (flags[n16 + j] && !cb[j / kBlk]) { cb[j / kBlk] = true; ++nc; }
  delete[] flags;
  const bool rows = nr > 0 && (nc == 0 || nr * m <= nc * n);  // the cheaper side: recomputed symbols
  const size_t es = dtype == GECC_BF16 ? 2 : 4;
  int rc = GECC_OK, done = 0;
  for (int64_t b = 0; b < (rows ? nrb : ncb) && rc == GECC_OK; ++b) {
    if (!(rows ? rb[b] : cb[b])) continue;
    const int64_t o = b * kBlk;
    if (rows) {  // C[o : o + 256, :] = A[o : o + 256, :] B
      const int64_t nn = n - o < kBlk ? n - o : kBlk, ao = trans_a ? o : o * lda;
      rc = gemm_dispatch(false, dtype, nn, k, m, trans_a != 0, trans_b != 0, reinterpret_cast<const uint8_t*>(A) + ao * es, lda, nullptr, A_lo ? A_lo + ao : nullptr, nullptr,
                         B, ldb, nullptr, B_lo, nullptr, C + o * ldc, ldc, nullptr, nullptr, nullptr, nullptr, 0, nullptr, nullptr, nullptr, false, st);
    } else {     // C[:, o : o + 256] = A B[:, o : o + 256]
      const int64_t mm = m - o < kBlk ? m - o : kBlk, bo = trans_b ? o * ldb : o;
      rc = gemm_dispatch(false, dtype, n, k, mm, trans_a != 0, trans_b != 0, A, lda, nullptr, A_lo, nullptr, reinterpret_cast<const uint8_t*>(B) + bo * es, ldb, nullptr,
                         B_lo ? B_lo + bo : nullptr, nullptr, C + o, ldc, nullptr, nullptr, nullptr, nullptr, 0, nullptr, nullptr, nullptr, false, st);
    }
    ++done;
  }
  delete[] rb;
  if (rc != GECC_OK) return rc;
  // the checks again, over the stored C, against the parity of the first product; level 0: C_bar alone
  rc = syndrome_unfused_dispatch(n, m, C, ldc, reinterpret_cast<float*>(ws + L.rowpart), reinterpret_cast<float*>(ws + L.colpart),
                                 reinterpret_cast<DecodeState*>(ws + L.state), st);
  if (rc != GECC_OK) return rc;
  rc = decode_dispatch(dtype, n, k, m, C, ldc, P_r, P_c, nullptr, tau, sumsq_a, sumsq_b, 0, trans_a, trans_b, nullptr, 0, nullptr, nullptr, nullptr, 0, nullptr, nullptr,
                       report, ws, L, st);
  if (rc != GECC_OK) return rc;
  if (cudaStreamSynchronize(st) != cudaSuccess) return GECC_ECUDA;
  gecc_report_t rep2;
  if (cudaMemcpy(&rep2, report, sizeof(rep2), cudaMemcpyDeviceToHost) != cudaSuccess) return GECC_ECUDA;
  bool points_only = rep2.verdict == GECC_CORRECTED;
  for (int a = 0; a < rep2.n_found && a < GECC_MAX_FOUND; ++a) points_only = points_only && rep2.found[a].kind == GECC_KIND_C;
  rep2.n_row_flags = rep.n_row_flags; rep2.n_col_flags = rep.n_col_flags;  // what the first pass saw
  if (rep2.verdict == GECC_CLEAN || points_only) rep2.verdict = GECC_CORRECTED_BY_RECOMPUTE;
  else { rep2 = rep; }  // still not decodable: the first verdict stands
  if (cudaMemcpy(report, &rep2, sizeof(rep2), cudaMemcpyHostToDevice) != cudaSuccess) return GECC_ECUDA;
  return done;
}

int64_t gecc_tl_parity_rows(int64_t len) { return len <= 0 ? 0 : GECC_PAR_ROWS * ((len + GECC_TL_PANEL - 1) / GECC_TL_PANEL); }

int gecc_tl_encode(int dtype, int64_t n, int64_t k, int64_t m, const void* A, int64_t lda, float* A_lo, void* A_PL, float* A_PL_lo, double* sumsq_a, const void* B,
                   int64_t ldb, float* B_lo, void* B_PL, float* B_PL_lo, double* sumsq_b, void* workspace, size_t workspace_bytes, void* stream) {
  if (!dtype_ok(dtype)) return GECC_EUNSUPPORTED;
  if (!A || !B || !A_PL || !B_PL || !sumsq_a || !sumsq_b || !workspace || n <= 0 || k <= 0 || m <= 0 || n > kMaxDim || k > kMaxDim || m > kMaxDim) return GECC_EINVAL;
  const int epr = dtype == GECC_BF16 ? 8 : 4;
  if (lda < k || ldb < m || lda % epr || ldb % epr || k % epr || m % epr || !al16(A) || !al16(B) || !al16(A_PL) || !al16(B_PL)) return GECC_EINVAL;
  if (dtype == GECC_F32 && (!A_lo || !B_lo || !A_PL_lo || !B_PL_lo || !al16(A_lo) || !al16(B_lo))) return GECC_EINVAL;
  if (workspace_bytes < ws_layout(dtype, n, k, m).total) return GECC_EWORKSPACE;
  return tl_encode_dispatch(dtype, n, k, m, A, lda, A_lo, A_PL, A_PL_lo, sumsq_a, B, ldb, B_lo, B_PL, B_PL_lo, sumsq_b, reinterpret_cast<uint8_t*>(workspace),
                            reinterpret_cast<cudaStream_t>(stream));
}

int gecc_tl_matmul(int dtype, int64_t n, int64_t k, int64_t m, const void* A, int64_t lda, const void* A_PL, const float* A_lo, const float* A_PL_lo, const void* B,
                   int64_t ldb, const void* B_PL, const float* B_lo, const float* B_PL_lo, float* C, int64_t ldc, float* P_rL, int64_t ldprl, float* P_cL,
                   int64_t ldpcl, const gecc_fault_t* inject, int n_inject, void* workspace, size_t workspace_bytes, void* stream) {
  if (!dtype_ok(dtype)) return GECC_EUNSUPPORTED;
  if (!workspace || n <= 0 || k <= 0 || m <= 0) return GECC_EINVAL;
  const WsLayout L = ws_layout(dtype, n, k, m);
  if (workspace_bytes < L.total) return GECC_EWORKSPACE;
  uint8_t* ws = reinterpret_cast<uint8_t*>(workspace);
  DetectArgs det = {};
  det.detect = false;  // the per-block sums stay per block: gecc_tl_decode reads them
  det.st = reinterpret_cast<DecodeState*>(ws + L.state);
  det.counters = reinterpret_cast<unsigned int*>(ws);
  det.arrive = reinterpret_cast<unsigned int*>(ws + L.arrive);
  det.lineacc = reinterpret_cast<double*>(ws + L.lineacc);
  det.syn = reinterpret_cast<double*>(ws + L.syn);
  det.flags = ws + L.flags;
  TlArgs tla;
  tla.rows_a = gecc_tl_parity_rows(n); tla.rows_b = gecc_tl_parity_rows(m);
  tla.PcL = P_cL; tla.ldpcl = ldpcl; tla.PrL = P_rL; tla.ldprl = ldprl;
  return gemm_dispatch(true, dtype, n, k, m, false, false, A, lda, A_PL, A_lo, A_PL_lo, B, ldb, B_PL, B_lo, B_PL_lo, C, ldc, nullptr, nullptr, nullptr, inject, n_inject,
                       reinterpret_cast<float*>(ws + L.rowpart), reinterpret_cast<float*>(ws + L.colpart), &det, true, reinterpret_cast<cudaStream_t>(stream), &tla);
}

int gecc_tl_decode(int dtype, int64_t n, int64_t k, int64_t m, float* C, int64_t ldc, const float* P_rL, int64_t ldprl, const float* P_cL, int64_t ldpcl,
                   const double* tau, const double* sumsq_a, const double* sumsq_b, int mode, gecc_tl_report_t* report, void* workspace, size_t workspace_bytes,
                   void* stream) {
  if (!dtype_ok(dtype)) return GECC_EUNSUPPORTED;
  if (!C || !P_rL || !P_cL || !report || !workspace || n <= 0 || k <= 0 || m <= 0 || ldc < m) return GECC_EINVAL;
  if (n > kMaxDim || k > kMaxDim || m > kMaxDim) return GECC_EINVAL;
  if (!tau && (!sumsq_a || !sumsq_b)) return GECC_EINVAL;
  if (mode != 0) return mode == GECC_SINGLE_CHECKSUM ? GECC_EUNSUPPORTED : GECC_EINVAL;  // the block decoder always uses both checks
  if (!al16(P_rL) || !al16(P_cL) || ldprl % 4 || ldpcl % 4 || ldprl < gecc_tl_parity_rows(m) || ldpcl < m) return GECC_EINVAL;
  const WsLayout L = ws_layout(dtype, n, k, m);
  if (workspace_bytes < L.total) return GECC_EWORKSPACE;
  return tl_decode_dispatch(dtype, n, k, m, C, ldc, P_rL, ldprl, P_cL, ldpcl, tau, sumsq_a, sumsq_b, mode, report, reinterpret_cast<uint8_t*>(workspace), L,
                            reinterpret_cast<cudaStream_t>(stream));
}

int gecc_decode_phase_ns(int dtype, int64_t n, int64_t k, int64_t m, const void* workspace, size_t workspace_bytes, double* phase_ns, int max_phases) {
  if (!dtype_ok(dtype)) return GECC_EUNSUPPORTED;
  if (!workspace || !phase_ns || n <= 0 || k <= 0 || m <= 0 || max_phases <= 0) return GECC_EINVAL;
  const WsLayout L = ws_layout(dtype, n, k, m);
  if (workspace_bytes < L.total) return GECC_EWORKSPACE;
  unsigned long long st[kMaxPhaseStamps];
  if (cudaMemcpy(st, reinterpret_cast<const uint8_t*>(workspace) + L.timing, sizeof(st), cudaMemcpyDeviceToHost) != cudaSuccess) return GECC_ECUDA;
  const int cnt = st[0] < (unsigned long long)kMaxPhaseStamps ? (int)st[0] : 0;
  int out = 0;
  for (int i = 2; i <= cnt && out < max_phases; ++i) phase_ns[out++] = (double)(st[i] - st[i - 1]);
  return out;
}

int gecc_inject_inputs(int dtype, int trans_a, int trans_b, void* A, int64_t lda, float* A_lo, void* B, int64_t ldb, float* B_lo, const gecc_fault_t* faults, int n_faults,
                       void* stream) {
  if (!dtype_ok(dtype)) return GECC_EUNSUPPORTED;
  if (n_faults < 0 || n_faults > 32 || (n_faults > 0 && (!faults || !A || !B))) return GECC_EINVAL;
  if (n_faults == 0) return GECC_OK;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(1);
  cfg.blockDim = dim3(32);
  cfg.stream = reinterpret_cast<cudaStream_t>(stream);
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;  // its launch overlaps the encoder's tail; it waits for the encoder inside
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (cudaLaunchKernelEx(&cfg, inject_inputs_kernel, dtype, trans_a, trans_b, A, lda, A_lo, B, ldb, B_lo, faults, n_faults) != cudaSuccess) return GECC_ECUDA;
  return GECC_OK;
}

}  // extern "C"
