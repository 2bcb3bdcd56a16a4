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


def test_bench_launcher_world_size_2_dry_run():
    """`bench.py --gpus 2` without a torchrun environment re-executes itself under torch.distributed.run; --dry-run keeps the
    launcher, the sequence sharding of cfg 5 (strong scaling) and the two reductions, and needs no GPU (gloo)."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--config", "5", "--steps", "10", "--dry-run"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads([x for x in r.stdout.splitlines() if x.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["scaling"] == "strong" and line["dry_run"] is True
    assert [s[:2] for s in line["shards"]] == [[0, 4], [4, 8]]                 # 8 sequences over 2 ranks
    assert line["shards"][0][2] == line["shards"][1][2] == 2 * 128 * 4          # each rank's pool: 2k pages per sequence
    assert line["ms_per_step"] == pytest.approx(2.0) and line["value"] == pytest.approx(10 / 0.020)   # steps do not add up over shards
    # a single-sequence config runs one replica set per rank (weak scaling): the units add up
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--config", "3", "--steps", "10", "--dry-run"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads([x for x in r.stdout.splitlines() if x.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["scaling"] == "weak" and line["value"] == pytest.approx(20 / 0.020)


def test_shard_config_keeps_the_sequences_of_the_whole_batch():
    from paper_2606_09079_b200.workloads import LsaWorkload, make_small_config, shard_config
    import numpy as np
    cfg = make_small_config("f32", B=4, L=[4096, 2432, 1024, 2048], stagger=True, hot_pages=64)
    whole = LsaWorkload(cfg)
    lo, hi = 1, 3
    part = LsaWorkload(shard_config(cfg, lo, hi))
    assert part.cfg.B == 2 and part.cfg.hot_pages >= 2 * sum(cfg.k_eff(b) for b in range(lo, hi))
    for j, b in enumerate(range(lo, hi)):
        assert np.array_equal(part.hca_k[j], whole.hca_k[b]) and np.array_equal(part.cold_csa[j], whole.cold_csa[b])
        assert np.array_equal(part.chunk_emb(j, 0), whole.chunk_emb(b, 0))
        assert part.cfg.step0(j) == cfg.step0(b)                                # same trigger phase as in the whole batch
