"""Row-sharded multi-GPU host logic on CPU: world_size 2, gloo backend.

The local evaluator injected into `ShardedEbic` is the CPU oracle on the rank's own row slice, so
these tests check exactly what the N > 1 path adds: the row partition, the one all-reduce of the
counts and the concatenation of mask shards.
"""
from __future__ import annotations

import os
import socket

import numpy as np
import pytest

from paper_1807_09932_b200 import workloads as W
from paper_1807_09932_b200.sharded import ShardedEbic, row_partition


@pytest.mark.parametrize("rows,world", [(1, 1), (1, 4), (63, 2), (64, 2), (65, 2), (200, 3), (436_444, 8),
                                        (65_537, 5)])
def test_row_partition(rows, world):
    b = row_partition(rows, world)
    assert len(b) == world and b[0][0] == 0 and b[-1][1] == rows
    for (b0, e0), (b1, e1) in zip(b, b[1:]):
        assert e0 == b1 and b0 <= e0
    for b0, e0 in b[:-1]:
        assert e0 % 64 == 0 or e0 == rows                      # mask words never straddle ranks
    words = [(e - s + 63) // 64 for s, e in b]
    assert max(words) - min(words) <= 1                        # balanced to within one 64-row word


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str, rows: int = 3001):
    import torch
    import torch.distributed as dist
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = W.make_workload(1, rows=rows, n_ind=120)             # ragged: 3001 = 46*64 + 57
        chosen = np.array([0, 4, 7, 119], dtype=np.int32)
        b, e = row_partition(w.rows, world)[rank]
        local = np.ascontiguousarray(w.matrix[b:e])

        def local_eval(off, ids):
            return oracle.eval_fitness(local, w.missing_mode, off, ids)[1]

        def local_extract(off, ids, ch):
            return oracle.extract_rows(local, w.missing_mode, off, ids, ch)[1]

        sh = ShardedEbic(w.rows, rank, world, local_eval, local_extract)
        counts, shard = sh.step(w.offsets, w.col_ids, chosen)
        assert shard.shape == (len(chosen), sh.local_words)
        masks = sh.gather_masks(shard)
        np.save(os.path.join(out_dir, f"counts{rank}.npy"), counts.numpy())
        np.save(os.path.join(out_dir, f"masks{rank}.npy"), masks.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,rows", [(2, 3001), (3, 100)])    # (3, 100): two 64-row words, rank 2 holds no rows
def test_gloo_matches_unsharded_oracle(tmp_path, oracle_mod, world, rows):
    import torch.multiprocessing as mp
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path), rows), nprocs=world, join=True)
    w = W.make_workload(1, rows=rows, n_ind=120)
    chosen = np.array([0, 4, 7, 119], dtype=np.int32)
    _, want = oracle_mod.eval_fitness(w.matrix, w.missing_mode, w.offsets, w.col_ids)
    _, want_masks, _ = oracle_mod.extract_rows(w.matrix, w.missing_mode, w.offsets, w.col_ids, chosen)
    for rank in range(world):
        counts = np.load(tmp_path / f"counts{rank}.npy")
        masks = np.load(tmp_path / f"masks{rank}.npy")
        assert (counts.view(np.uint64) == want).all()
        assert masks.shape == want_masks.shape
        assert (masks.view(np.uint64) == want_masks).all()
