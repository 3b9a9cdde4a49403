"""The N > 1 path of bench.py on CPU: world_size 2 over gloo ("replicas only").

The path has no data-path collective; the only multi-rank logic is the aggregation of the JSON line
(time = MAX over ranks, pairs = SUM over ranks) and the per-rank replica seeds."""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, str(ROOT))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    times = torch.tensor([1.0 + rank, 5.0 - rank], dtype=torch.float64)
    pairs = torch.tensor([10.0 * (rank + 1), 7.0], dtype=torch.float64)
    t, p = bench.aggregate_over_ranks(times, pairs)
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, t, p))


def test_aggregate_is_max_time_and_summed_work_over_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for _, t, p in res:
        assert t == [2.0, 5.0]          # max over ranks of (1, 2) and (5, 4)
        assert p == [30.0, 14.0]        # sum over ranks


def test_aggregate_without_process_group_is_identity():
    sys.path.insert(0, str(ROOT))
    import bench
    t, p = bench.aggregate_over_ranks(torch.tensor([1.5, 2.5], dtype=torch.float64),
                                      torch.tensor([3.0, 4.0], dtype=torch.float64))
    assert t == [1.5, 2.5] and p == [3.0, 4.0]


def test_replicas_differ_by_seed_only():
    """--gpus N runs N independent replicas of the same workload: same species tables, different draws."""
    sys.path.insert(0, str(ROOT))
    from paper_2212_00663_b200 import workloads as W
    a = W.make(4, n_per_species=64, seed=4)
    b = W.make(4, n_per_species=64, seed=4 + 1000)
    assert np.array_equal(a.mass, b.mass) and np.array_equal(a.charge, b.charge) and a.n_markers == b.n_markers
    assert not np.array_equal(a.v, b.v)
