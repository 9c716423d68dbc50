"""world_size-2 test of the multi-rank path on CPU (gloo): the row-shard plan with every rank running the
complete code on its shard.  There is no GPU here, so each rank's shard product is computed by the CPU oracle; what is
under test is the host logic of paper_2508_04355_b200/shard.py and the rendezvous / gather plumbing bench.py relies on."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import gecc_oracle as O
from paper_2508_04355_b200 import inputs as I
from paper_2508_04355_b200 import shard as S


def test_plan_rows_covers_and_aligns():
    for n, w, al in [(4096, 2, 256), (1000, 3, 256), (64, 4, 256), (8192, 8, 256), (300, 2, 128)]:
        plan = S.plan_rows(n, w, al)
        assert len(plan) == w and plan[0][0] == 0 and plan[-1][1] == n
        for (a0, a1), (b0, b1) in zip(plan, plan[1:]):
            assert a1 == b0 and a0 <= a1
        for r0, r1 in plan:
            assert r0 % al == 0 or r0 == n
        sizes = [r1 - r0 for r0, r1 in plan if r1 > r0]
        assert max(sizes) - min(sizes) < 2 * al      # block counts differ by at most one; the last block may be partial


def test_fault_mapping_round_trip():
    faults = [(S.KIND_A, 300, 5, 1.0), (S.KIND_B, 7, 9, 2.0), (S.KIND_C, 10, 11, 3.0)]
    plan = S.plan_rows(512, 2, 256)
    f0, f1 = (S.faults_for_shard(faults, *plan[g]) for g in range(2))
    assert f0 == [(S.KIND_B, 7, 9, 2.0), (S.KIND_C, 10, 11, 3.0)]
    assert f1 == [(S.KIND_A, 44, 5, 1.0), (S.KIND_B, 7, 9, 2.0)]
    back = S.fold_found([S.found_to_global([(k, r, c) for k, r, c, _ in f0], plan[0][0]),
                         S.found_to_global([(k, r, c) for k, r, c, _ in f1], plan[1][0])])
    assert back == sorted((k, r, c) for k, r, c, _ in faults)
    assert S.fold_verdicts([S.CLEAN, S.CORRECTED]) == S.CORRECTED
    assert S.fold_verdicts([S.CORRECTED, S.UNCORRECTABLE_INPUT, S.UNCORRECTABLE]) == S.UNCORRECTABLE_INPUT


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n, k, m, faults, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        A, B = I.make_operands(n, k, m, seed=11, dtype="f32")
        r0, r1 = S.plan_rows(n, world, align=16)[rank]
        mine = S.faults_for_shard(faults, r0, r1)
        rep = O.protected_matmul(A[r0:r1], B, faults=mine, level=1)       # the shard's own complete code
        t = torch.tensor([rep.verdict], dtype=torch.int64)
        verdicts = [torch.zeros_like(t) for _ in range(world)]
        dist.all_gather(verdicts, t)
        found = [None] * world
        dist.all_gather_object(found, S.found_to_global(rep.located(), r0))
        # max-over-ranks reduction, as bench.py does with its device times
        tmax = torch.tensor([float(rank + 1)])
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        assert tmax.item() == float(world)
        Cs = [None] * world
        dist.all_gather_object(Cs, rep.C)
        if rank == 0:
            np.save(os.path.join(out_dir, "C.npy"), np.vstack(Cs))
            np.save(os.path.join(out_dir, "verdict.npy"), np.array([S.fold_verdicts(int(v.item()) for v in verdicts)]))
            np.save(os.path.join(out_dir, "found.npy"), np.array(S.fold_found(found), dtype=np.int64).reshape(-1, 3))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("faults", [
    [],
    [(0, 5, 7, 12.0), (2, 40, 3, -6.0)],          # A fault in shard 0, C fault in shard 1
    [(1, 9, 4, 8.0), (2, 1, 1, 5.0)],             # B fault (seen by both shards) + C fault in shard 0
])
def test_two_rank_row_sharded_product_matches_the_unsharded_oracle(tmp_path, faults):
    n, k, m, world = 64, 24, 40, 2
    mp.spawn(_worker, args=(world, _free_port(), n, k, m, faults, str(tmp_path)), nprocs=world, join=True)
    A, B = I.make_operands(n, k, m, seed=11, dtype="f32")
    clean = A.astype(np.float64) @ B.astype(np.float64)
    C = np.load(tmp_path / "C.npy")
    assert np.abs(C - clean).max() <= 1e-9 * np.abs(clean).max()
    assert int(np.load(tmp_path / "verdict.npy")[0]) == (S.CORRECTED if faults else S.CLEAN)
    found = [tuple(int(x) for x in row) for row in np.load(tmp_path / "found.npy")]
    assert found == sorted((kd, r, c) for kd, r, c, _ in faults)
