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


def test_library_shard_range_is_the_same_split():
    """epr_shard_range (include/epr.h; what epr_retrieve_host_multi gives plan k of n) against `shard_range`, which the
    one-process-per-GPU launch uses: the same ranges for every (total, parts), and argument errors.  Host arithmetic: the
    library is loaded, no device is touched."""
    import shutil
    import pytest
    import paper_2601_22793_b200 as E
    if not os.path.exists(E.lib_path()):
        if shutil.which("nvcc") is None:
            pytest.skip("nvcc not available and libepr.so not built")
        from paper_2601_22793_b200 import build
        build.build()
    for total in (0, 1, 2, 5, 7, 64, 8000):
        for parts in (1, 2, 3, 8):
            for k in range(parts):
                assert E.epr_shard_range(total, k, parts) == shard_range(total, k, parts)
    for bad in ((5, 2, 2), (5, -1, 2), (5, 0, 0), (-1, 0, 1)):
        with pytest.raises(E.EprError):
            E.epr_shard_range(*bad)


def test_ranks_generate_their_share_of_one_seeded_batch():
    """bench.py --gpus N: ONE seeded batch of N x B projections, rank k generates and retrieves the range shard_range gives
    it (make_workload(first=lo)); put together the shares are the batch a single process would have generated."""
    from epr_inputs import make_workload
    whole = make_workload("C1", n=32, batch=7, distinct=2)
    parts = []
    for k in range(3):
        lo, hi = shard_range(7, k, 3)
        part = make_workload("C1", n=32, batch=hi - lo, distinct=2, first=lo)
        assert part.L_m == whole.L_m
        parts.append(part.d)
    assert np.array_equal(np.concatenate(parts), whole.d)


def test_two_rank_gloo_sharding(tmp_path):
    world, total = 2, 7
    mp.spawn(_worker, args=(world, _free_port(), total, str(tmp_path)), nprocs=world, join=True)
    got = np.concatenate([np.load(tmp_path / f"r{k}.npy") for k in range(world)])
    assert np.array_equal(got, np.arange(total, dtype=np.float32) * 2.0)


def _run_bench(env_extra, *args):
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, **env_extra)
    return subprocess.run([sys.executable, os.path.join(root, "bench.py"), *args], cwd=root, env=env,
                          capture_output=True, text=True, timeout=600)


def test_bench_reference_arm_contract():
    """`bench.py --impl reference` (the oracle on the host cores) prints ONE JSON line with the base contract's keys on
    rank 0; under a multi-rank launch the other ranks exit 0 without work or output."""
    import json
    res = _run_bench({"RANK": "0", "WORLD_SIZE": "1"}, "--impl", "reference", "--config", "C1", "--steps", "1", "--warmup", "0")
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [ln for ln in res.stdout.splitlines() if ln.strip()]
    assert len(lines) == 1
    j = json.loads(lines[0])
    assert j["impl"] == "reference" and j["unit"] == "projections/s" and j["higher_is_better"] is True
    assert j["value"] > 0 and j["steps"] == 1 and j["dtype"] == "f64" and j["data"] == "synthetic"
    assert j["cpu_baseline"]["kind"] == "oracle" and j["cpu_baseline"]["value"] == j["value"]
    assert j["e2e"] == {"value": j["value"], "unit": j["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert j["config"]["workload"].startswith("C1")
    other = _run_bench({"RANK": "1", "WORLD_SIZE": "2", "LOCAL_RANK": "1"}, "--impl", "reference", "--config", "C1",
                       "--gpus", "2", "--steps", "1", "--warmup", "0")
    assert other.returncode == 0 and other.stdout.strip() == ""
    # a budget too small for whole projections: each step runs the first iterations only and says so
    res = _run_bench({"RANK": "0", "WORLD_SIZE": "1"}, "--impl", "reference", "--config", "C1", "--steps", "3", "--warmup", "1",
                     "--ref-budget", "0.01")
    assert res.returncode == 0, res.stderr[-2000:]
    j = json.loads(res.stdout.strip())
    assert j["config"]["iterations_run_per_step"] == 1 and "extrapolated" in j["cpu_baseline"]["sample"]
    # ONE time base: value and ms_per_step both describe the full workload; what was timed sits in config
    assert j["config"]["extrapolated"] is True and j["ms_per_step"] > j["config"]["ms_per_step_measured"] > 0
    assert abs(1e3 / j["value"] - j["ms_per_step"]) < 1e-9 * j["ms_per_step"]
