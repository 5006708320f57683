"""World-size-2 gloo test (CPU) of the N > 1 host logic: contiguous sharding of independent projections with no
data-path collective, a barrier, and the max-over-ranks time reduction bench.py reports."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from epr_inputs import shard_range


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, total, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    lo, hi = shard_range(total, rank, world)
    # every rank "processes" its own shard (stand-in for epr_retrieve on its GPU) and reports a time
    d = np.arange(total, dtype=np.float32)[lo:hi] * 2.0
    ranges = [None] * world
    dist.all_gather_object(ranges, (lo, hi))
    dist.barrier()
    t = bench.max_over_ranks(10.0 + rank, torch.device("cpu"))
    np.save(os.path.join(out_dir, f"r{rank}.npy"), d)
    if rank == 0:
        assert ranges[0][0] == 0 and ranges[-1][1] == total
        assert all(ranges[i][1] == ranges[i + 1][0] for i in range(world - 1))
        assert t == 10.0 + world - 1
    dist.destroy_process_group()


def test_shard_ranges_cover_and_balance():
    for total in (1, 2, 7, 64):
        for world in (1, 2, 3, 8):
            r = [shard_range(total, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == total
            assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1


def test_two_rank_gloo_sharding(tmp_path):
    world, total = 2, 7
    mp.spawn(_worker, args=(world, _free_port(), total, str(tmp_path)), nprocs=world, join=True)
    got = np.concatenate([np.load(tmp_path / f"r{k}.npy") for k in range(world)])
    assert np.array_equal(got, np.arange(total, dtype=np.float32) * 2.0)
