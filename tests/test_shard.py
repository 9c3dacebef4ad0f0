"""Multi-GPU host logic on CPU: sharding by whole packed words and the one
reduction of the sharded job, with a world-size-2 `gloo` process group on 127.0.0.1.

Each rank follows ITS shard of a small disorder pool with the CPU oracle (keyed by the global sample
index, as the library is through sg_set_first_sample), the per-slot moment sums are all-reduced with
shard.reduce_moment_sums, and the result must equal the single-process sum over the whole pool.
"""
import os
import socket

import numpy as np
import pytest

from paper_1403_4560_b200 import shard, workloads as W


def test_shard_range_partitions_whole_words():
    for n_samples in (1, 31, 32, 33, 64, 2048, 2049, 8192, 100):
        for world in (1, 2, 3, 4, 8):
            ranges = [shard.shard_range(n_samples, world, r) for r in range(world)]
            nxt = 0
            for first, count in ranges:
                assert first % 32 == 0                       # whole words only
                assert first == nxt or count == 0
                nxt = first + count if count else nxt
            assert sum(c for _, c in ranges) == n_samples
            words = [(c + 31) // 32 for _, c in ranges]
            assert max(words) - min(words) <= 1              # as even as possible
    with pytest.raises(ValueError):
        shard.shard_range(64, 2, 2)
    with pytest.raises(ValueError):
        shard.shard_range(0, 1, 0)


L, H_FIELD, R, NT, SEED, N_SAMPLES, SWEEPS = 4, 0.3, 4, 4, 11, 70, 12


def _local_sums(first, count):
    from oracle import ea_oracle as O
    temps = W.ladder(0.6, 1.9, NT)
    tot = np.zeros((NT, O.NMOM))
    for s in range(first, first + count):
        o = O.Oracle(L, H_FIELD, R, temps, kind=O.PMJ, seed=SEED, sample=s)
        o.run(SWEEPS, 1, 4)
        m, n = o.moments()
        assert n == SWEEPS // 4
        tot += m
        o.close()
    return tot


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        first, count = shard.shard_range(N_SAMPLES, world, rank)
        local = torch.from_numpy(_local_sums(first, count))
        keep = local.clone()
        out = shard.reduce_moment_sums(local)
        assert torch.equal(local, keep)                      # input not modified
        q.put((rank, first, count, out.numpy()))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_reduction_equals_single_process():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = [q.get(timeout=240) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    got.sort(key=lambda g: g[0])
    assert got[0][1] == 0 and got[1][1] == got[0][2] and got[0][2] + got[1][2] == N_SAMPLES
    want = _local_sums(0, N_SAMPLES)
    for _, _, _, out in got:
        assert np.all(np.abs(out - want) <= 1e-12 * np.maximum(np.abs(want), 1.0))
    assert np.array_equal(got[0][3], got[1][3])              # same on every rank


def test_reduce_without_process_group_is_identity():
    import torch
    x = torch.arange(6, dtype=torch.float64).reshape(2, 3)
    assert torch.equal(shard.reduce_moment_sums(x), x)
