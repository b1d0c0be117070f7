"""CPU-only: the N > 1 bookkeeping (frame sharding, max-over-ranks time, catalogue offsets) with world_size 2 over gloo."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2502_10783_b200 import shard


def test_shard_range_partitions_units():
    for n in (0, 1, 7, 64, 65):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                a, b = shard.shard_range(n, r, world)
                assert 0 <= a <= b <= n and b - a in (n // world, n // world + 1)
                seen += list(range(a, b))
            assert seen == list(range(n))
    with pytest.raises(ValueError):
        shard.shard_range(4, 2, 2)
    assert shard.rank_seed(5, 0) == 5 and len({shard.rank_seed(5, r) for r in range(8)}) == 8


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n_frames = 5
        a, b = shard.shard_range(n_frames, rank, world)
        # each rank "detects" (frame + 1) sources per frame of its shard and takes (rank + 1) ms per step
        n_local = sum(f + 1 for f in range(a, b))
        t_max = shard.max_over_ranks(1.0 + rank, dist)
        px_all = shard.sum_over_ranks(100.0 * (b - a), dist)
        off, total = shard.catalogue_offsets(n_local, dist)
        dist.barrier()
        np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([a, b, n_local, t_max, px_all, off, total], dtype=np.float64))
    finally:
        dist.destroy_process_group()


def test_two_ranks_over_gloo(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r0, r1 = np.load(tmp_path / "r0.npy"), np.load(tmp_path / "r1.npy")
    assert (r0[0], r0[1], r1[0], r1[1]) == (0, 3, 3, 5)                 # 5 frames -> 3 + 2, contiguous
    assert r0[3] == r1[3] == 2.0                                       # max over ranks of (1, 2) ms
    assert r0[4] == r1[4] == 500.0                                     # all ranks' pixels
    assert (r0[5], r1[5]) == (0, 6) and r0[6] == r1[6] == 15           # catalogue offsets 1+2+3 | 4+5
    assert shard.whole_job_value(r0[4], r0[3] * 1e-3) == 500.0 / 2e-3


def test_single_process_paths():
    assert shard.max_over_ranks(3.5) == 3.5 and shard.sum_over_ranks(2.0) == 2.0
    assert shard.catalogue_offsets(7) == (0, 7)
