"""Thin ctypes binding of libgecc.so (include/gecc.h).  Argument marshalling only: every step of the path runs in the
CUDA kernels behind the C ABI.  PyTorch supplies device memory and streams, nothing else.

There is no CPU fallback: if the library is missing or cannot be loaded, every call raises.
"""
from __future__ import annotations

import ctypes
import os

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libgecc.so")

GECC_BF16, GECC_F32 = 0, 1
GECC_LEFT, GECC_RIGHT = 0, 1
GECC_PAR_ROWS, GECC_PR_LD, GECC_MAX_FOUND = 8, 8, 8
CLEAN, CORRECTED, UNCORRECTABLE, UNCORRECTABLE_INPUT, CORRECTED_BY_RECOMPUTE = 0, 1, 2, 3, 4
KIND_A, KIND_B, KIND_C, KIND_ROW, KIND_COL, KIND_PR, KIND_PC = 0, 1, 2, 3, 4, 5, 6
LEVEL_X, SINGLE_CHECKSUM = 1, 2
STATUS = {0: "GECC_OK", -1: "GECC_EINVAL", -2: "GECC_EUNSUPPORTED", -3: "GECC_ECUDA", -4: "GECC_EWORKSPACE", -5: "GECC_ETOOLARGE"}

EXPORTS = ["gecc_version", "gecc_workspace_bytes", "gecc_encode", "gecc_encode_noalloc", "gecc_encode_both", "gecc_matmul_protected", "gecc_matmul_plain",
           "gecc_syndrome_unfused", "gecc_decode_correct", "gecc_decode_phase_ns", "gecc_inject_inputs", "gecc_recompute_fallback",
           "gecc_tl_parity_rows", "gecc_tl_encode", "gecc_tl_matmul", "gecc_tl_decode"]
TL_PANEL, TL_MAX_FOUND = 128, 64


class GeccFault(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int32), ("row", ctypes.c_int32), ("col", ctypes.c_int32), ("value", ctypes.c_float)]


class GeccFound(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int32), ("row", ctypes.c_int32), ("col", ctypes.c_int32), ("pad_", ctypes.c_int32),
                ("magnitude", ctypes.c_double)]


class GeccReport(ctypes.Structure):
    _fields_ = [("verdict", ctypes.c_int32), ("n_found", ctypes.c_int32), ("n_row_flags", ctypes.c_int32),
                ("n_col_flags", ctypes.c_int32), ("max_abs_syndrome", ctypes.c_double * 4), ("tau", ctypes.c_double * 4),
                ("found", GeccFound * GECC_MAX_FOUND)]

    def located(self):
        return [(f.kind, f.row, f.col) for f in self.found[: self.n_found]]

    def magnitudes(self):
        return [f.magnitude for f in self.found[: self.n_found]]


class GeccTlReport(ctypes.Structure):
    """gecc_tl_report_t: the report of the tile-local grid's decoder (one code per 128 x 128 block of C)."""
    _fields_ = [("verdict", ctypes.c_int32), ("n_found", ctypes.c_int32), ("n_row_flags", ctypes.c_int32),
                ("n_col_flags", ctypes.c_int32), ("max_abs_syndrome", ctypes.c_double * 4), ("tau", ctypes.c_double * 4),
                ("found", GeccFound * TL_MAX_FOUND)]

    def located(self):
        return [(f.kind, f.row, f.col) for f in self.found[: min(self.n_found, TL_MAX_FOUND)]]

    def magnitudes(self):
        return [f.magnitude for f in self.found[: min(self.n_found, TL_MAX_FOUND)]]


_lib = None


def load():
    """Loads libgecc.so (building it first is the job of paper_2508_04355_b200.build / __graft_entry__.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2508_04355_b200.build` (there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i64, sz, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_size_t, ctypes.c_int
    lib.gecc_version.restype = ctypes.c_char_p
    lib.gecc_version.argtypes = []
    lib.gecc_workspace_bytes.restype = sz
    lib.gecc_workspace_bytes.argtypes = [ci, i64, i64, i64]
    lib.gecc_encode.restype = ci
    lib.gecc_encode.argtypes = [ci, ci, ci, vp, i64, i64, i64, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.gecc_encode_noalloc.restype = ci
    lib.gecc_encode_noalloc.argtypes = [ci, ci, ci, vp, i64, i64, i64, vp, vp, vp, vp, vp, vp]
    lib.gecc_encode_both.restype = ci
    lib.gecc_encode_both.argtypes = [ci, i64, i64, i64, ci, ci, vp, i64, vp, vp, vp, vp, vp, vp, i64, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.gecc_matmul_protected.restype = ci
    lib.gecc_matmul_protected.argtypes = [ci, i64, i64, i64, ci, ci, vp, i64, vp, vp, vp, vp, i64, vp, vp, vp, vp, i64, vp, vp, vp, vp, ci,
                                          ctypes.POINTER(ctypes.c_double), vp, vp, vp, ci, vp, sz, vp]
    lib.gecc_matmul_plain.restype = ci
    lib.gecc_matmul_plain.argtypes = [ci, i64, i64, i64, ci, ci, vp, i64, vp, vp, i64, vp, vp, i64, vp]
    lib.gecc_syndrome_unfused.restype = ci
    lib.gecc_syndrome_unfused.argtypes = [ci, i64, i64, i64, vp, i64, vp, sz, vp]
    lib.gecc_decode_correct.restype = ci
    lib.gecc_decode_correct.argtypes = [ci, i64, i64, i64, vp, i64, vp, vp, vp, ctypes.POINTER(ctypes.c_double), vp, vp, ci,
                                        ci, ci, vp, i64, vp, vp, vp, i64, vp, vp, vp, vp, sz, vp]
    lib.gecc_recompute_fallback.restype = ci
    lib.gecc_recompute_fallback.argtypes = [ci, i64, i64, i64, ci, ci, vp, i64, vp, vp, i64, vp, vp, i64, vp, vp, ctypes.POINTER(ctypes.c_double), vp, vp,
                                            vp, vp, sz, vp]
    lib.gecc_decode_phase_ns.restype = ci
    lib.gecc_decode_phase_ns.argtypes = [ci, i64, i64, i64, vp, sz, ctypes.POINTER(ctypes.c_double), ci]
    lib.gecc_inject_inputs.restype = ci
    lib.gecc_inject_inputs.argtypes = [ci, ci, ci, vp, i64, vp, vp, i64, vp, vp, ci, vp]
    lib.gecc_tl_parity_rows.restype = i64
    lib.gecc_tl_parity_rows.argtypes = [i64]
    lib.gecc_tl_encode.restype = ci
    lib.gecc_tl_encode.argtypes = [ci, i64, i64, i64, vp, i64, vp, vp, vp, vp, vp, i64, vp, vp, vp, vp, vp, sz, vp]
    lib.gecc_tl_matmul.restype = ci
    lib.gecc_tl_matmul.argtypes = [ci, i64, i64, i64, vp, i64, vp, vp, vp, vp, i64, vp, vp, vp, vp, i64, vp, i64, vp, i64, vp, ci, vp, sz, vp]
    lib.gecc_tl_decode.restype = ci
    lib.gecc_tl_decode.argtypes = [ci, i64, i64, i64, vp, i64, vp, i64, vp, i64, ctypes.POINTER(ctypes.c_double), vp, vp, ci, vp, vp, sz, vp]
    _lib = lib
    return lib


def _p(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"{what} failed: {STATUS.get(rc, rc)}")


def dtype_code(t: torch.Tensor) -> int:
    if t.dtype == torch.bfloat16:
        return GECC_BF16
    if t.dtype == torch.float32:
        return GECC_F32
    raise TypeError(f"unsupported operand dtype {t.dtype}")


def gecc_version() -> str:
    return load().gecc_version().decode()


def gecc_workspace_bytes(dtype: int, n: int, k: int, m: int) -> int:
    return int(load().gecc_workspace_bytes(dtype, n, k, m))


def faults_to_device(faults, device) -> torch.Tensor | None:
    """[(kind, row, col, value)] -> device buffer of gecc_fault_t (16 bytes each)."""
    if not faults:
        return None
    arr = (GeccFault * len(faults))(*[GeccFault(int(k), int(r), int(c), float(v)) for k, r, c, v in faults])
    host = torch.frombuffer(bytearray(bytes(arr)), dtype=torch.uint8)
    return host.to(device)


def gecc_encode(side, X, parity, parity_lo, x_lo, parity64, sumsq, workspace, stream=None, trans=0):
    """X is the operand as stored; trans = 1: X holds the operand's transpose (A^T: k x n, B^T: m x k)."""
    rows, cols = X.shape
    _same_ld(X, x_lo, "x_lo")
    rc = load().gecc_encode(dtype_code(X), side, int(trans), _p(X), rows, cols, X.stride(0), _p(parity), _p(parity_lo), _p(x_lo), _p(parity64),
                            _p(sumsq), _p(workspace), workspace.numel(), _stream(stream))
    _check(rc, "gecc_encode")


NOALLOC_SCRATCH_BYTES = 9 << 20   # GECC_NOALLOC_SCRATCH_BYTES of include/gecc.h


def gecc_encode_noalloc(side, X, parity, parity_lo, x_lo, parity64, sumsq, stream=None, trans=0):
    """gecc_encode without a workspace: the scratch is a fixed array inside the library (include/gecc.h states the limit
    and the sharing rule); nothing is allocated by the call."""
    rows, cols = X.shape
    _same_ld(X, x_lo, "x_lo")
    rc = load().gecc_encode_noalloc(dtype_code(X), side, int(trans), _p(X), rows, cols, X.stride(0), _p(parity), _p(parity_lo), _p(x_lo), _p(parity64),
                                    _p(sumsq), _stream(stream))
    if rc == -5:
        raise RuntimeError(f"gecc_encode_noalloc failed: GECC_ETOOLARGE (a {rows} x {cols} operand needs more than the library's fixed "
                           f"{NOALLOC_SCRATCH_BYTES} bytes of scratch; use gecc_encode with a workspace)")
    _check(rc, "gecc_encode_noalloc")


def _same_ld(X, X_lo, name):
    """include/gecc.h: the fp32 lo plane of an operand shares the operand's shape AND leading dimension (the kernels index
    both with one ld); a padded operand view needs an equally padded lo plane."""
    if X_lo is not None and (X_lo.stride(0) != X.stride(0) or tuple(X_lo.shape) != tuple(X.shape)):
        raise ValueError(f"{name} must have the operand's shape and leading dimension: {tuple(X_lo.shape)}/{X_lo.stride(0)} vs "
                         f"{tuple(X.shape)}/{X.stride(0)}")


def gecc_encode_both(A, B, buf, stream=None):
    """Both encoders in one launch; A and B as stored (buf.trans_a / buf.trans_b), outputs into buf."""
    n, k, m = _dims(A, B, buf.trans_a, buf.trans_b)
    _same_ld(A, buf.A_lo, "A_lo")
    _same_ld(B, buf.B_lo, "B_lo")
    rc = load().gecc_encode_both(dtype_code(A), n, k, m, buf.trans_a, buf.trans_b, _p(A), A.stride(0), _p(buf.A_par), _p(buf.A_par_lo), _p(buf.A_lo),
                                 _p(buf.A_par64), _p(buf.sumsq_a), _p(B), B.stride(0), _p(buf.B_par), _p(buf.B_par_lo), _p(buf.B_lo), _p(buf.B_par64),
                                 _p(buf.sumsq_b), _p(buf.workspace), buf.workspace.numel(), _stream(stream))
    _check(rc, "gecc_encode_both")


def _dims(A, B, trans_a, trans_b):
    n, k = (A.shape[1], A.shape[0]) if trans_a else A.shape
    m = B.shape[0] if trans_b else B.shape[1]
    return n, k, m


def gecc_matmul_protected(A, A_par, A_lo, A_par_lo, B, B_par, B_lo, B_par_lo, C, P_r, P_c, P_g, inject, n_inject, workspace, stream=None,
                          trans_a=0, trans_b=0, tau=None, sumsq_a=None, sumsq_b=None, report=None, mode=0):
    """tau (4 host values) or sumsq_a / sumsq_b (device, from gecc_encode) switch on the detection inside the product."""
    n, k, m = _dims(A, B, trans_a, trans_b)
    _same_ld(A, A_lo, "A_lo")
    _same_ld(B, B_lo, "B_lo")
    rc = load().gecc_matmul_protected(dtype_code(A), n, k, m, int(trans_a), int(trans_b), _p(A), A.stride(0), _p(A_par), _p(A_lo), _p(A_par_lo), _p(B), B.stride(0),
                                      _p(B_par), _p(B_lo), _p(B_par_lo), _p(C), C.stride(0), _p(P_r), _p(P_c), _p(P_g), _p(inject),
                                      int(n_inject), None if tau is None else (ctypes.c_double * 4)(*[float(x) for x in tau]), _p(sumsq_a), _p(sumsq_b),
                                      _p(report), int(mode), _p(workspace), workspace.numel(), _stream(stream))
    _check(rc, "gecc_matmul_protected")


def gecc_matmul_plain(A, A_lo, B, B_lo, C, stream=None, trans_a=0, trans_b=0):
    n, k, m = _dims(A, B, trans_a, trans_b)
    _same_ld(A, A_lo, "A_lo")
    _same_ld(B, B_lo, "B_lo")
    rc = load().gecc_matmul_plain(dtype_code(A), n, k, m, int(trans_a), int(trans_b), _p(A), A.stride(0), _p(A_lo), _p(B), B.stride(0), _p(B_lo), _p(C), C.stride(0),
                                  _stream(stream))
    _check(rc, "gecc_matmul_plain")


def gecc_syndrome_unfused(dtype, k, C, workspace, stream=None):
    n, m = C.shape
    rc = load().gecc_syndrome_unfused(dtype, n, k, m, _p(C), C.stride(0), _p(workspace), workspace.numel(), _stream(stream))
    _check(rc, "gecc_syndrome_unfused")


def gecc_decode_correct(dtype, n, k, m, C, P_r, P_c, tau, sumsq_a, sumsq_b, level, A, A_lo, A_par64, B, B_lo, B_par64, report, workspace,
                        stream=None, trans_a=0, trans_b=0, P_g=None):
    """level: bit LEVEL_X (input verification), bit SINGLE_CHECKSUM; P_g switches on the global-parity check of Eq. (4)."""
    tau_arr = None if tau is None else (ctypes.c_double * 4)(*[float(x) for x in tau])
    if A is not None:
        _same_ld(A, A_lo, "A_lo")
    if B is not None:
        _same_ld(B, B_lo, "B_lo")
    rc = load().gecc_decode_correct(dtype, n, k, m, _p(C), C.stride(0), _p(P_r), _p(P_c), _p(P_g), tau_arr, _p(sumsq_a), _p(sumsq_b), int(level),
                                    int(trans_a), int(trans_b), _p(A), 0 if A is None else A.stride(0), _p(A_lo), _p(A_par64), _p(B), 0 if B is None else B.stride(0),
                                    _p(B_lo), _p(B_par64), _p(report), _p(workspace), workspace.numel(), _stream(stream))
    _check(rc, "gecc_decode_correct")


def gecc_recompute_fallback(A, A_lo, B, B_lo, C, P_r, P_c, tau, sumsq_a, sumsq_b, report, workspace, stream=None, trans_a=0, trans_b=0):
    """Synchronous.  Returns the number of 256-line blocks of C that were computed again (0: the verdict was not UNCORRECTABLE)."""
    n, k, m = _dims(A, B, trans_a, trans_b)
    tau_arr = None if tau is None else (ctypes.c_double * 4)(*[float(x) for x in tau])
    rc = load().gecc_recompute_fallback(dtype_code(A), n, k, m, int(trans_a), int(trans_b), _p(A), A.stride(0), _p(A_lo), _p(B), B.stride(0), _p(B_lo), _p(C),
                                        C.stride(0), _p(P_r), _p(P_c), tau_arr, _p(sumsq_a), _p(sumsq_b), _p(report), _p(workspace), workspace.numel(),
                                        _stream(stream))
    if rc < 0:
        _check(rc, "gecc_recompute_fallback")
    return rc


def gecc_decode_phase_ns(dtype, n, k, m, workspace):
    """Nanoseconds between the phase boundaries of the last decode on this workspace (synchronises)."""
    out = (ctypes.c_double * 64)()
    rc = load().gecc_decode_phase_ns(dtype, n, k, m, _p(workspace), workspace.numel(), out, 64)
    if rc < 0:
        _check(rc, "gecc_decode_phase_ns")
    return [out[i] for i in range(rc)]


def gecc_inject_inputs(A, A_lo, B, B_lo, faults_dev, n_faults, stream=None, trans_a=0, trans_b=0):
    rc = load().gecc_inject_inputs(dtype_code(A), int(trans_a), int(trans_b), _p(A), A.stride(0), _p(A_lo), _p(B), B.stride(0), _p(B_lo), _p(faults_dev), int(n_faults),
                                   _stream(stream))
    _check(rc, "gecc_inject_inputs")


def read_report(report_dev: torch.Tensor) -> GeccReport:
    """Device report buffer (uint8, sizeof(gecc_report_t)) -> host struct (synchronises)."""
    raw = bytes(report_dev.cpu().numpy().tobytes())
    return GeccReport.from_buffer_copy(raw[: ctypes.sizeof(GeccReport)])


class Buffers:
    """Device buffers of one protected product (allocation only; sizes follow include/gecc.h)."""

    def __init__(self, n: int, k: int, m: int, dtype: torch.dtype, device="cuda", trans_a=0, trans_b=0):
        self.n, self.k, self.m = n, k, m
        self.dtype = dtype
        self.code = GECC_BF16 if dtype == torch.bfloat16 else GECC_F32
        f32 = self.code == GECC_F32
        dev = device
        self.A_par = torch.zeros(GECC_PAR_ROWS, k, dtype=dtype, device=dev)
        self.B_par = torch.zeros(GECC_PAR_ROWS, k, dtype=dtype, device=dev)
        self.A_par_lo = torch.zeros(GECC_PAR_ROWS, k, dtype=torch.float32, device=dev) if f32 else None
        self.B_par_lo = torch.zeros(GECC_PAR_ROWS, k, dtype=torch.float32, device=dev) if f32 else None
        self.trans_a, self.trans_b = int(trans_a), int(trans_b)
        self.A_lo = torch.zeros((k, n) if trans_a else (n, k), dtype=torch.float32, device=dev) if f32 else None
        self.B_lo = torch.zeros((m, k) if trans_b else (k, m), dtype=torch.float32, device=dev) if f32 else None
        self.A_par64 = torch.zeros(2, k, dtype=torch.float64, device=dev)
        self.B_par64 = torch.zeros(2, k, dtype=torch.float64, device=dev)
        self.sumsq_a = torch.zeros(1, dtype=torch.float64, device=dev)
        self.sumsq_b = torch.zeros(1, dtype=torch.float64, device=dev)
        self.C = torch.zeros(n, m, dtype=torch.float32, device=dev)
        self.P_r = torch.zeros(n, GECC_PR_LD, dtype=torch.float32, device=dev)
        self.P_c = torch.zeros(GECC_PAR_ROWS, m, dtype=torch.float32, device=dev)
        self.P_g = torch.zeros(GECC_PAR_ROWS, GECC_PR_LD, dtype=torch.float32, device=dev)
        self.workspace = torch.zeros(gecc_workspace_bytes(self.code, n, k, m), dtype=torch.uint8, device=dev)
        self.report = torch.zeros(ctypes.sizeof(GeccReport), dtype=torch.uint8, device=dev)
        self.side_stream = torch.cuda.Stream(device=dev)
        self.ev_fork, self.ev_join = torch.cuda.Event(), torch.cuda.Event()

    def lo_planes_for(self, A, B):
        """fp32 only: the lo planes must share their operand's leading dimension (include/gecc.h); operands passed as padded
        views get lo planes of the same strides (allocated once per stride)."""
        if self.code != GECC_F32:
            return
        for name, X in (("A_lo", A), ("B_lo", B)):
            lo = getattr(self, name)
            if lo is None or lo.stride(0) != X.stride(0) or tuple(lo.shape) != tuple(X.shape):
                big = torch.zeros(X.shape[0], X.stride(0), dtype=torch.float32, device=X.device)
                setattr(self, name, big[:, : X.shape[1]])


def protected_matmul(A, B, buf: Buffers, faults=(), tau=None, level=1, stream=None, faults_dev=None, report=None, global_parity=True,
                     fallback=False):
    """A and B are the operands AS STORED (buf.trans_a / buf.trans_b say whether they hold the transpose).
    The whole path through the C ABI, in the paper's order: encode A, encode B, input faults E1/E2
    strike the stored operands, encoded product with E3 faults in the epilogue,
    detection and correction.  Returns nothing; results are in buf.C / buf.report (or `report`).
    `faults_dev` (from faults_to_device) avoids the host-to-device copy of the fault list inside the call."""
    main = torch.cuda.current_stream() if stream is None else stream
    buf.lo_planes_for(A, B)
    gecc_encode_both(A, B, buf, main)
    nf = len(faults)
    fdev = faults_dev if faults_dev is not None else faults_to_device(list(faults), A.device)
    if nf:
        gecc_inject_inputs(A, buf.A_lo, B, buf.B_lo, fdev, nf, stream, trans_a=buf.trans_a, trans_b=buf.trans_b)
    rep = buf.report if report is None else report
    gecc_matmul_protected(A, buf.A_par, buf.A_lo, buf.A_par_lo, B, buf.B_par, buf.B_lo, buf.B_par_lo, buf.C, buf.P_r, buf.P_c, buf.P_g,
                          fdev, nf, buf.workspace, stream, trans_a=buf.trans_a, trans_b=buf.trans_b, tau=tau, sumsq_a=buf.sumsq_a, sumsq_b=buf.sumsq_b,
                          report=rep, mode=level & SINGLE_CHECKSUM)
    gecc_decode_correct(buf.code, buf.n, buf.k, buf.m, buf.C, buf.P_r, buf.P_c, tau, buf.sumsq_a, buf.sumsq_b, level,
                        A, buf.A_lo, buf.A_par64, B, buf.B_lo, buf.B_par64, rep, buf.workspace, stream,
                        trans_a=buf.trans_a, trans_b=buf.trans_b, P_g=buf.P_g if global_parity else None)
    if fallback:  # what the code cannot correct "needs to be recalculated" (synchronous: reads the verdict)
        return gecc_recompute_fallback(A, buf.A_lo, B, buf.B_lo, buf.C, buf.P_r, buf.P_c, tau, buf.sumsq_a, buf.sumsq_b, rep, buf.workspace, stream,
                                       trans_a=buf.trans_a, trans_b=buf.trans_b)
    return 0


# ---------------------------------------------------------------------------------------------------------------
# Tile-local grid (include/gecc.h: gecc_tl_*): one code per 128 x 128 block of C
# ---------------------------------------------------------------------------------------------------------------
def gecc_tl_parity_rows(length: int) -> int:
    return int(load().gecc_tl_parity_rows(length))


class TlBuffers:
    """Device buffers of one product protected by the tile-local grid (allocation only; sizes follow include/gecc.h)."""

    def __init__(self, n: int, k: int, m: int, dtype: torch.dtype, device="cuda"):
        self.n, self.k, self.m, self.dtype = n, k, m, dtype
        self.code = GECC_BF16 if dtype == torch.bfloat16 else GECC_F32
        f32 = self.code == GECC_F32
        ra, rb = gecc_tl_parity_rows(n), gecc_tl_parity_rows(m)
        self.A_PL = torch.zeros(ra, k, dtype=dtype, device=device)
        self.B_PL = torch.zeros(rb, k, dtype=dtype, device=device)
        self.A_PL_lo = torch.zeros(ra, k, dtype=torch.float32, device=device) if f32 else None
        self.B_PL_lo = torch.zeros(rb, k, dtype=torch.float32, device=device) if f32 else None
        self.A_lo = torch.zeros(n, k, dtype=torch.float32, device=device) if f32 else None
        self.B_lo = torch.zeros(k, m, dtype=torch.float32, device=device) if f32 else None
        self.sumsq_a = torch.zeros(1, dtype=torch.float64, device=device)
        self.sumsq_b = torch.zeros(1, dtype=torch.float64, device=device)
        self.C = torch.zeros(n, m, dtype=torch.float32, device=device)
        self.P_rL = torch.zeros(n, rb, dtype=torch.float32, device=device)
        self.P_cL = torch.zeros(ra, m, dtype=torch.float32, device=device)
        self.workspace = torch.zeros(gecc_workspace_bytes(self.code, n, k, m), dtype=torch.uint8, device=device)
        self.report = torch.zeros(ctypes.sizeof(GeccTlReport), dtype=torch.uint8, device=device)


def gecc_tl_encode(A, B, buf: TlBuffers, stream=None):
    n, k = A.shape
    m = B.shape[1]
    _same_ld(A, buf.A_lo, "A_lo")
    _same_ld(B, buf.B_lo, "B_lo")
    rc = load().gecc_tl_encode(dtype_code(A), n, k, m, _p(A), A.stride(0), _p(buf.A_lo), _p(buf.A_PL), _p(buf.A_PL_lo), _p(buf.sumsq_a),
                               _p(B), B.stride(0), _p(buf.B_lo), _p(buf.B_PL), _p(buf.B_PL_lo), _p(buf.sumsq_b), _p(buf.workspace), buf.workspace.numel(),
                               _stream(stream))
    _check(rc, "gecc_tl_encode")


def gecc_tl_matmul(A, B, buf: TlBuffers, inject=None, n_inject=0, stream=None):
    n, k = A.shape
    m = B.shape[1]
    rc = load().gecc_tl_matmul(dtype_code(A), n, k, m, _p(A), A.stride(0), _p(buf.A_PL), _p(buf.A_lo), _p(buf.A_PL_lo), _p(B), B.stride(0), _p(buf.B_PL),
                               _p(buf.B_lo), _p(buf.B_PL_lo), _p(buf.C), buf.C.stride(0), _p(buf.P_rL), buf.P_rL.stride(0), _p(buf.P_cL), buf.P_cL.stride(0),
                               _p(inject), int(n_inject), _p(buf.workspace), buf.workspace.numel(), _stream(stream))
    _check(rc, "gecc_tl_matmul")


def gecc_tl_decode(buf: TlBuffers, tau=None, mode=0, stream=None, report=None):
    tau_arr = None if tau is None else (ctypes.c_double * 4)(*[float(x) for x in tau])
    rep = buf.report if report is None else report
    rc = load().gecc_tl_decode(buf.code, buf.n, buf.k, buf.m, _p(buf.C), buf.C.stride(0), _p(buf.P_rL), buf.P_rL.stride(0), _p(buf.P_cL), buf.P_cL.stride(0),
                               tau_arr, _p(buf.sumsq_a), _p(buf.sumsq_b), int(mode), _p(rep), _p(buf.workspace), buf.workspace.numel(), _stream(stream))
    _check(rc, "gecc_tl_decode")


def tl_protected_matmul(A, B, buf: TlBuffers, faults=(), tau=None, stream=None, faults_dev=None):
    """The whole path of the tile-local grid through the C ABI: per-panel encode, input faults, encoded product with E3 faults in
    the epilogue, block-by-block detection and correction.  Results in buf.C / buf.report."""
    gecc_tl_encode(A, B, buf, stream)
    nf = len(faults)
    fdev = faults_dev if faults_dev is not None else faults_to_device(list(faults), A.device)
    if nf:
        gecc_inject_inputs(A, buf.A_lo, B, buf.B_lo, fdev, nf, stream)
    gecc_tl_matmul(A, B, buf, fdev, nf, stream)
    gecc_tl_decode(buf, tau=tau, stream=stream)


def read_tl_report(report_dev: torch.Tensor) -> GeccTlReport:
    raw = bytes(report_dev.cpu().numpy().tobytes())
    return GeccTlReport.from_buffer_copy(raw[: ctypes.sizeof(GeccTlReport)])


# kernel launches of one protected_matmul call (for bench.py's gpu_launches): the encoder (both operands in one launch), inject
# (if any fault), the encoded GEMM, and the decoder (one cooperative kernel, whatever the level)
def launches_per_call(n_faults: int, level: int) -> int:
    return 1 + (1 if n_faults else 0) + 1 + 1
