"""Multi-GPU plumbing of the LSA path: sequences are independent units, so ranks shard them and never
exchange data on the path.  Only timing is reduced across ranks.

Used by bench.py (NCCL, one rank per GPU) and tested on CPU with a world-size-2 gloo group
(tests/test_multirank_cpu.py).  No CUDA needed to import."""
from __future__ import annotations

from typing import List, Tuple

import torch
import torch.distributed as dist


def shard_sequences(n_seq: int, world: int, rank: int) -> Tuple[int, int]:
    """Contiguous, balanced [lo, hi) range of the batch's sequences served by `rank`
    (the first n_seq % world ranks get one more)."""
    if world < 1 or not (0 <= rank < world) or n_seq < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(n_seq, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def max_over_ranks(ms: float, device=None) -> float:
    """Device time of the slowest rank (the job's time); identity without a process group."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(units: int, device=None) -> int:
    """Units (steps x sequences) processed by the whole job."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return int(units)
    t = torch.tensor([int(units)], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return int(t.item())


def job_throughput(units_this_rank: int, ms_this_rank: float, device=None) -> Tuple[float, float]:
    """(whole-job units per second, job milliseconds): all ranks' units / slowest rank's time."""
    ms = max_over_ranks(ms_this_rank, device)
    units = sum_over_ranks(units_this_rank, device)
    return units / (ms * 1e-3), ms


def all_shards(n_seq: int, world: int) -> List[Tuple[int, int]]:
    return [shard_sequences(n_seq, world, r) for r in range(world)]
