"""Multi-rank host logic of the batch sharding (independent members, no data-path collective),
run as two gloo processes on the CPU: the member partition, the per-rank seeded inputs of bench.py and the
max-over-ranks timing reduction."""
import os
import socket

import numpy as np
import pytest

import kx_inputs as kin
from paper_2607_00755_b200 import shard


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        B = 5
        c = bench._inputs(rank, B, 3)
        ids = shard.weak_member_ids(B, rank, world)
        # the rank's batch is exactly the global members it owns
        want = np.stack([kin._random_bimodal(c["p"], 3000 + int(g)) for g in ids])
        assert np.array_equal(c["f"], want)
        # every rank sees every rank's ids: disjoint, covering 0 .. W*B-1
        gathered = [torch.zeros(B, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(gathered, torch.from_numpy(ids))
        allids = torch.cat(gathered).numpy()
        assert sorted(allids.tolist()) == list(range(world * B))
        # timing reduction: max over ranks, element by element
        t = shard.max_over_ranks([1.0 + rank, 5.0 - rank, 0.25], dist)
        assert t == [float(world), 5.0, 0.25]
        # strong split of a fixed batch
        r = shard.member_range(11, rank, world)
        lens = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(lens, torch.tensor([len(r)], dtype=torch.int64))
        assert sum(int(x) for x in lens) == 11
        np.save(os.path.join(out_dir, f"f_rank{rank}.npy"), c["f"])
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_weak_sharding_two_ranks_gloo(tmp_path):
    import torch.multiprocessing as mp
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    f0 = np.load(tmp_path / "f_rank0.npy")
    f1 = np.load(tmp_path / "f_rank1.npy")
    assert f0.shape == f1.shape == (5, 256)
    assert not np.array_equal(f0, f1)
    # rank 0 of a multi-rank job evaluates the same members as the single-GPU job
    assert np.array_equal(f0, kin.config(3, B=5)["f"])


@pytest.mark.parametrize("n,world", [(0, 1), (7, 1), (11, 2), (64, 8), (5, 8)])
def test_member_range_partitions(n, world):
    got = [i for r in range(world) for i in shard.member_range(n, r, world)]
    assert got == list(range(n))
    sizes = [len(shard.member_range(n, r, world)) for r in range(world)]
    assert max(sizes) - min(sizes) <= 1


def test_aggregate_rate():
    assert shard.aggregate_rate(64, 8, 10, 2.0) == 64 * 8 * 10 / 2.0
    with pytest.raises(ValueError):
        shard.member_range(4, 2, 2)
