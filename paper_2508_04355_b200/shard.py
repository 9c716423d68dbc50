"""Row sharding of a protected product over ranks: host logic only.

A is split by row blocks; rank g holds A_g (n_g x k) and all of B and runs its own complete code M(n_g + 2, k, m + 2) with
local weights 1..n_g (PAPER.md:71-113 applied to the shard).  Encode, product and decode never look at another shard, so
there is no data-path collective; the correcting power becomes <= 2 errors per shard.  What is left for the host: the
row plan, mapping global fault positions into shards, mapping located positions back, and folding the verdicts.
No arithmetic of the method lives here.
"""
from __future__ import annotations

CLEAN, CORRECTED, UNCORRECTABLE, UNCORRECTABLE_INPUT = 0, 1, 2, 3
KIND_A, KIND_B, KIND_C, KIND_ROW, KIND_COL = 0, 1, 2, 3, 4


def plan_rows(n: int, world_size: int, align: int = 256):
    """[(row0, row1)] per rank: contiguous, covering [0, n), sizes multiples of `align` except the last non-empty one,
    as even as the alignment allows.  Ranks beyond the number of aligned blocks get an empty range."""
    if n <= 0 or world_size <= 0 or align <= 0:
        raise ValueError("plan_rows: n, world_size, align must be positive")
    blocks = (n + align - 1) // align
    base, extra = divmod(blocks, world_size)
    plan, row = [], 0
    for g in range(world_size):
        nb = base + (1 if g < extra else 0)
        stop = min(n, row + nb * align)
        plan.append((row, stop))
        row = stop
    return plan


def faults_for_shard(faults, row0: int, row1: int):
    """Global fault list -> the faults this shard sees, in shard coordinates.  A faults (i, l) and C faults (i, j) belong
    to the shard that holds row i; B faults (l, j) hit the copy of B of EVERY shard (B is replicated)."""
    out = []
    for kind, r, c, v in faults:
        if kind == KIND_B:
            out.append((kind, r, c, v))
        elif row0 <= r < row1:
            out.append((kind, r - row0, c, v))
    return out


def found_to_global(found, row0: int):
    """Located positions of one shard -> global coordinates (rows of A / C shift by the shard's first row)."""
    out = []
    for kind, r, c in found:
        if kind in (KIND_A, KIND_C, KIND_ROW):
            out.append((kind, r + row0, c))
        else:
            out.append((kind, r, c))
    return out


def fold_verdicts(verdicts):
    """Verdict of the whole product from the shards': the most severe one (CLEAN < CORRECTED < UNCORRECTABLE <
    UNCORRECTABLE_INPUT)."""
    v = list(verdicts)
    return max(v) if v else CLEAN


def fold_found(per_shard_found):
    """Union of the shards' located positions (global coordinates), sorted by (kind, row, col); a B symbol reported by
    several shards (B is replicated) is listed once."""
    seen = set()
    for f in per_shard_found:
        seen.update(tuple(x) for x in f)
    return sorted(seen)
