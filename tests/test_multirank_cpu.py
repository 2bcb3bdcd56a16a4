"""The N > 1 path on CPU: a world-size-2 gloo group exercises the sequence sharding and the
max-over-ranks / sum-over-ranks reductions bench.py uses (sequences are
independent units, no data-path collective)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_09079_b200.dist import all_shards, job_throughput, max_over_ranks, shard_sequences


def test_shards_partition_the_batch():
    for n in (0, 1, 7, 8, 32, 33):
        for world in (1, 2, 3, 8):
            sh = all_shards(n, world)
            assert sh[0][0] == 0 and sh[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(sh, sh[1:]))
            sizes = [hi - lo for lo, hi in sh]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        shard_sequences(4, 2, 2)


def test_single_process_is_identity():
    assert max_over_ranks(3.5) == 3.5
    assert job_throughput(100, 50.0) == (2000.0, 50.0)


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        lo, hi = shard_sequences(33, world, rank)
        units = (hi - lo) * 10                       # 10 steps of this rank's sequences
        ms = 20.0 if rank == 0 else 50.0             # rank 1 is the slow one
        value, job_ms = job_throughput(units, ms)
        # no rank ever needs another rank's sequences: the only traffic is the two scalars above
        out[rank] = (lo, hi, value, job_ms)
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert out[0][:2] == (0, 17) and out[1][:2] == (17, 33)
    for r in (0, 1):
        assert out[r][3] == 50.0                                  # slowest rank's time
        assert out[r][2] == pytest.approx(330 / 0.050)            # all ranks' units / that time
