"""gecc_encode_noalloc (include/gecc.h): the encoder with its scratch in a fixed array of the library's device image, for
callers that cannot allocate.  Checked against the existing path (gecc_encode on a caller's workspace) on two calls in a
row that share the array, with the tolerances tests/test_gpu_parity.py uses for the encoder's outputs.

This file is named so that pytest collects it last: the suite runs with `pytest -x`.
"""
import numpy as np
import pytest
import torch

from paper_2508_04355_b200 import binding as G

pytestmark = pytest.mark.gpu


class Out:
    """Output buffers of one encoder call (len = the operand's inner dimension k)."""

    def __init__(self, X, length):
        f32 = X.dtype == torch.float32
        dev = X.device
        # filled with a sentinel so that an output the call never wrote cannot pass by accident
        self.parity = torch.full((G.GECC_PAR_ROWS, length), 7.0, dtype=X.dtype, device=dev)
        self.parity_lo = torch.full((G.GECC_PAR_ROWS, length), 7.0, dtype=torch.float32, device=dev) if f32 else None
        self.x_lo = torch.full(tuple(X.shape), 7.0, dtype=torch.float32, device=dev) if f32 else None
        self.par64 = torch.full((2, length), 7.0, dtype=torch.float64, device=dev)
        self.sumsq = torch.full((1,), 7.0, dtype=torch.float64, device=dev)


def _encode_pair(X, side, trans):
    """(existing path, no-allocation path) on the same operand."""
    rows, cols = X.shape
    over_rows = (side == G.GECC_LEFT) != bool(trans)
    length = cols if over_rows else rows
    ref, new = Out(X, length), Out(X, length)
    code = G.dtype_code(X)
    ws = torch.zeros(G.gecc_workspace_bytes(code, max(rows, cols), max(rows, cols), max(rows, cols)), dtype=torch.uint8, device=X.device)
    G.gecc_encode(side, X, ref.parity, ref.parity_lo, ref.x_lo, ref.par64, ref.sumsq, ws, trans=trans)
    G.gecc_encode_noalloc(side, X, new.parity, new.parity_lo, new.x_lo, new.par64, new.sumsq, trans=trans)
    torch.cuda.synchronize()
    return ref, new


def _compare(ref, new, X):
    scale = float(ref.par64.abs().max())
    assert scale > 0.0
    # the checks as accumulated (fp64 side copy): tests/test_gpu_parity.py allows 1e-6 of the largest check
    assert float((new.par64 - ref.par64).abs().max()) <= 1e-6 * scale
    # the parity operand handed to the tensor cores (limbs / hi + lo): 2^-22 of the largest check
    def symbol(o):
        p = o.parity.double()
        if o.parity_lo is not None:
            p = p + o.parity_lo.double()
        return torch.stack([p[0:3].sum(0), p[3:6].sum(0)])
    assert float((symbol(new) - symbol(ref)).abs().max()) <= 2.0 ** -22 * scale
    assert float(new.sumsq) == pytest.approx(float(ref.sumsq), rel=1e-5)
    assert float(ref.sumsq) == pytest.approx(float((X.double() ** 2).sum()), rel=1e-5)
    if ref.x_lo is not None:
        assert torch.equal(new.x_lo, ref.x_lo)                         # x - tf32_trunc(x): no sum involved
    # the same launch on the same data in the same fixed order: equality is expected, the tolerances above are the bar
    assert torch.equal(new.par64, ref.par64) and torch.equal(new.parity, ref.parity)


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_no_alloc_encoder_matches_the_workspace_path_on_two_calls_in_a_row(dtype):
    tdt = torch.bfloat16 if dtype == "bf16" else torch.float32
    gen = torch.Generator(device="cuda")
    gen.manual_seed(20250804)
    # several strips / chunks and a ragged tail in both directions; the second call is a different shape, direction and
    # data, so whatever the first call left in the shared array would show
    calls = [((1000, 1544), G.GECC_LEFT, 0), ((712, 2056), G.GECC_RIGHT, 0), ((1000, 1544), G.GECC_RIGHT, 1), ((264, 136), G.GECC_LEFT, 1)]
    for shape, side, trans in calls:
        X = (torch.randn(*shape, device="cuda", generator=gen) * 1.7 + 0.05).to(tdt)
        ref, new = _encode_pair(X, side, trans)
        _compare(ref, new, X)
    # the same operand twice in a row, back to back on one stream, without a synchronisation in between
    X = torch.randn(2048, 1032, device="cuda", generator=gen).to(tdt)
    a, b, ref = Out(X, 1032), Out(X, 1032), Out(X, 1032)
    G.gecc_encode_noalloc(G.GECC_LEFT, X, a.parity, a.parity_lo, a.x_lo, a.par64, a.sumsq)
    G.gecc_encode_noalloc(G.GECC_LEFT, X, b.parity, b.parity_lo, b.x_lo, b.par64, b.sumsq)
    ws = torch.zeros(G.gecc_workspace_bytes(G.dtype_code(X), 2048, 2048, 2048), dtype=torch.uint8, device="cuda")
    G.gecc_encode(G.GECC_LEFT, X, ref.parity, ref.parity_lo, ref.x_lo, ref.par64, ref.sumsq, ws)
    torch.cuda.synchronize()
    _compare(ref, a, X)
    _compare(ref, b, X)


def test_no_alloc_encoder_allocates_nothing_and_refuses_what_does_not_fit():
    X = torch.randn(4096, 8192, device="cuda").to(torch.bfloat16)        # the largest shape the header names as fitting
    o = Out(X, 8192)
    G.gecc_encode_noalloc(G.GECC_LEFT, X, o.parity, o.parity_lo, o.x_lo, o.par64, o.sumsq)   # set-up call (symbol address)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        G.gecc_encode_noalloc(G.GECC_LEFT, X, o.parity, o.parity_lo, o.x_lo, o.par64, o.sumsq)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                                               # no device memory was taken by the calls
    want = X.double().sum(0)
    assert float((o.par64[0] - want).abs().max()) <= 1e-6 * float(want.abs().max())
    big = torch.zeros(8192, 8192, dtype=torch.bfloat16, device="cuda")
    ob = Out(big, 8192)
    with pytest.raises(RuntimeError, match="GECC_ETOOLARGE"):
        G.gecc_encode_noalloc(G.GECC_LEFT, big, ob.parity, ob.parity_lo, ob.x_lo, ob.par64, ob.sumsq)
    torch.cuda.synchronize()
    assert float(ob.sumsq) == 7.0                                       # refused before anything was launched
