"""The N > 1 path of bench.py on CPU: world_size 2 over gloo ("replicas only").

The path has no data-path collective; the only multi-rank logic is the aggregation of the JSON line
(time = MAX over ranks, pairs = SUM over ranks) and the per-rank replica seeds."""
import os
import socket
import sys
from pathlib import Path

import numpy as np
import pytest
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


def _shard_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, str(ROOT))
    from paper_2212_00663_b200 import workloads as W
    dist.init_process_group("gloo", rank=rank, world_size=world)
    rng = np.random.default_rng(7)                                  # the same ragged batch on every rank
    n = rng.integers(0, 1025, size=301)
    off = np.concatenate([[0], np.cumsum(n)]).astype(np.int64)
    c0, c1 = W.shard_cells(off, rank, world)
    mine = torch.tensor([c0, c1, int((n[c0:c1].astype(np.int64) ** 2).sum())], dtype=torch.int64)
    allr = [torch.zeros(3, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(allr, mine)
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, [t.tolist() for t in allr], int((n.astype(np.int64) ** 2).sum()), int(n.size), int(n.max())))


def test_cells_shard_over_ranks_is_a_balanced_partition_over_gloo():
    """NEXT-3 multi-GPU path (cells_bench under torchrun): workloads.shard_cells gives every rank a contiguous range of
    cells, every cell exactly once, pairwise work balanced to within one cell -- no data-path collective is needed."""
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_shard_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == res[1][1]                                   # every rank sees the same table
    _, table, total, ncells, nmax = res[0]
    assert table[0][0] == 0 and table[-1][1] == ncells
    assert all(table[r][1] == table[r + 1][0] for r in range(world - 1))
    assert sum(t[2] for t in table) == total
    assert max(t[2] for t in table) <= total / world + nmax * nmax


def test_shard_cells_edge_cases():
    sys.path.insert(0, str(ROOT))
    from paper_2212_00663_b200 import workloads as W
    assert W.shard_cells(np.array([0]), 0, 4) == (0, 0)                                  # no cells
    off = np.array([0, 0, 0, 0], dtype=np.int64)                                          # only empty cells
    assert [W.shard_cells(off, r, 2) for r in range(2)] == [(0, 1), (1, 3)]
    off = np.array([0, 1000], dtype=np.int64)                                             # fewer cells than ranks
    got = [W.shard_cells(off, r, 3) for r in range(3)]
    assert sorted(b - a for a, b in got) == [0, 0, 1] and got[0][0] == 0 and got[-1][1] == 1
    assert all(got[r][1] == got[r + 1][0] for r in range(2))
    for world in (1, 2, 3, 5, 8):
        rng = np.random.default_rng(world)
        n = rng.integers(1, 600, size=97)
        off = np.concatenate([[0], np.cumsum(n)])
        cuts = [W.shard_cells(off, r, world) for r in range(world)]
        assert cuts[0][0] == 0 and cuts[-1][1] == 97 and all(cuts[r][1] == cuts[r + 1][0] for r in range(world - 1))
    with pytest.raises(ValueError):
        W.shard_cells(off, 2, 2)


def test_reference_arm_iteration_table_covers_every_workload(tmp_path, monkeypatch):
    """bench_iters.json (tracked; rewritten by the GPU arm when a run measures another count) is what --impl reference
    scales its oracle sample with: every bench workload has an entry, and record_iters only touches the file on a change."""
    sys.path.insert(0, str(ROOT))
    import bench
    for w in bench.WORKLOADS:
        assert 1 <= bench.ref_iters(w) <= 50, w
    copy = tmp_path / "bench_iters.json"
    copy.write_text(bench.REF_ITERS_FILE.read_text())
    monkeypatch.setattr(bench, "REF_ITERS_FILE", copy)
    before = copy.stat().st_mtime_ns
    bench.record_iters("c0", bench.ref_iters("c0"))
    assert copy.stat().st_mtime_ns == before
    bench.record_iters("c0", 11)
    assert bench.ref_iters("c0") == 11 and bench.ref_iters("c1") == 13
