"""N>1 plumbing on CPU: world_size-2 gloo.  Replicas only -- no data-path collective; the batch is
sharded by cloud, every rank computes its own clouds (here with the CPU oracle standing in for the
GPU call), and only the timing is MAX-reduced."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_06255_b200 import inputs, sharding


def test_shard_range_partitions():
    for B in (0, 1, 4, 16, 17):
        for world in (1, 2, 3, 8):
            got = []
            for r in range(world):
                lo, hi = sharding.shard_range(B, r, world)
                got += list(range(lo, hi))
            assert got == list(range(B))
    with pytest.raises(ValueError):
        sharding.shard_range(4, 2, 2)
    assert sharding.rank_seed(1234, 0, 16) == 1234 and sharding.rank_seed(1234, 3, 16) == 1234 + 48


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, tmp):
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = inputs.scaled("C2", 1200, 150, B=5)
    P = inputs.make_batch(w)
    lo, hi = sharding.shard_range(w.B, rank, world)
    idx, mind = oracle.fps(P[lo:hi], w.M, 0, threads=1)
    np.save(os.path.join(tmp, f"idx{rank}.npy"), idx)
    np.save(os.path.join(tmp, f"mind{rank}.npy"), mind)
    t = sharding.max_over_ranks(1.0 + rank, dist)          # rank 1 is "slower"
    dist.barrier()
    if rank == 0:
        np.save(os.path.join(tmp, "tmax.npy"), np.array([t]))
    dist.destroy_process_group()


def test_world_size_2_shards_and_max_time(tmp_path):
    import oracle
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w = inputs.scaled("C2", 1200, 150, B=5)
    ref_idx, ref_mind = oracle.fps(inputs.make_batch(w), w.M, 0)
    idx = np.concatenate([np.load(tmp_path / f"idx{r}.npy") for r in range(world)])
    mind = np.concatenate([np.load(tmp_path / f"mind{r}.npy") for r in range(world)])
    assert np.array_equal(idx, ref_idx)
    assert np.array_equal(mind.view(np.uint32), ref_mind.view(np.uint32))
    assert float(np.load(tmp_path / "tmax.npy")[0]) == 2.0
