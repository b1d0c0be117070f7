"""Host-side sharding helpers for N > 1 (one process per GPU).  The path shards by FRAME: frames are
independent units, every rank runs the same calls on its own frames and there is no data-path collective.  The only
exchanges are bookkeeping: the max-over-ranks step time (bench.py) and the per-rank catalogue counts when a caller
wants one concatenated catalogue.  Works with any torch.distributed backend (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations

import torch


def shard_range(n_units: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous, balanced split of units 0..n_units-1: returns [start, stop) of `rank`."""
    if world <= 0 or not (0 <= rank < world) or n_units < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n_units, world)
    start = rank * base + min(rank, rem)
    return start, start + base + (1 if rank < rem else 0)


def rank_seed(seed: int, rank: int) -> int:
    """Seed of the synthetic frames of `rank` in the weak-scaling bench (rank 0 keeps the config's own seed)."""
    return seed + 7919 * rank


def _reduce(value: float, op, dist, device) -> float:
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=op)
    return float(t.item())


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """Step time of the job = the slowest rank's."""
    return _reduce(value, None if dist is None else dist.ReduceOp.MAX, dist, device)


def sum_over_ranks(value: float, dist=None, device="cpu") -> float:
    return _reduce(value, None if dist is None else dist.ReduceOp.SUM, dist, device)


def whole_job_value(units_all_ranks: float, seconds_max_over_ranks: float) -> float:
    """Aggregate throughput: units all ranks processed / the max-over-ranks time."""
    return units_all_ranks / seconds_max_over_ranks


def catalogue_offsets(n_local: int, dist=None, device="cpu") -> tuple[int, int]:
    """(offset of this rank's records, total records) in the rank-ordered concatenation of the per-rank catalogues
    (frames are sharded contiguously, so rank order = frame order)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return 0, int(n_local)
    world, rank = dist.get_world_size(), dist.get_rank()
    counts = [torch.zeros(1, dtype=torch.int64, device=device) for _ in range(world)]
    dist.all_gather(counts, torch.tensor([n_local], dtype=torch.int64, device=device))
    counts = [int(c.item()) for c in counts]
    return sum(counts[:rank]), sum(counts)
