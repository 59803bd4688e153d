"""world_size-2 `gloo` test (CPU) of the N>1 host logic of bench.py: every rank draws its own seeded
trajectories (weak scaling, no data-path collective) and the whole-job figure is SUM(units) / MAX(time)."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = bench.make_workload("cfg2", rank)                 # rank-specific seed
    ms, units = bench.aggregate_over_ranks(10.0 * (rank + 1), 1000.0 * (rank + 1), world)
    out.put((rank, float(w.waypoints.sum()), ms, units))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_by_seed_and_aggregate_max_time_sum_units():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] != res[1][1]                          # different trajectories per rank
    for r in res:
        assert r[2] == 20.0 and r[3] == 3000.0             # MAX time, SUM units on every rank


def test_single_rank_aggregate_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_over_ranks(3.5, 7.0, 1) == (3.5, 7.0)
