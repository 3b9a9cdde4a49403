"""Throughput of the batched collision-cell path (landau_cells_run) against the single-cell path.

    python -m paper_2212_00663_b200.cells_bench [--cells 1184] [--per-species 64 128 256 512] [--steps 5]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        -m paper_2212_00663_b200.cells_bench ...      # the batch sharded over N GPUs (workloads.shard_cells), no collective

Synthetic PIC-like batch: `cells` independent cells, each an e-i plasma shaped like BASELINE config 0 (2 species,
Maxwellian, T_e = 1, T_i = 0.5, random weights) with its own seed.  Reports cell-steps/s and ordered pass-2 pairs/s
of the one-launch batch (CUDA events), the same cells stepped one after the other through landau_set_markers +
landau_run (what a caller without the batch entry point would do), and the conservation drifts of the batch.
Prints one JSON line per cell size.
"""
from __future__ import annotations

import argparse
import json
import os

import numpy as np


def main():
    import torch
    from . import binding as B, workloads as W
    ap = argparse.ArgumentParser()
    ap.add_argument("--cells", type=int, default=1184)              # 8 cells per SM
    ap.add_argument("--per-species", type=int, nargs="+", default=[64, 128, 256, 512])
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--dt", type=float, default=0.002, help="config 0 uses 0.01 at 256 markers per species; cells "
                    "of 32..128 markers per species have closer unlike pairs and need a shorter step to contract")
    ap.add_argument("--sequential-cells", type=int, default=32, help="cells timed through the single-cell path")
    args = ap.parse_args()
    # one process per GPU under torchrun: every rank advances its own contiguous range of cells (cells are independent:
    # no data-path collective; a fixed batch split over the ranks); time = MAX over ranks, work = SUM over ranks
    rank, world, local = (int(os.environ.get(k, d)) for k, d in (("RANK", 0), ("WORLD_SIZE", 1), ("LOCAL_RANK", 0)))
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    base = W.make(0, n_per_species=8)
    dev = torch.device("cuda", local)
    torch.cuda.set_device(dev)
    g = B.Landau(base.mass, base.charge, base.eps, device=local)
    for nps in args.per_species:
        n = 2 * nps
        off_all = np.arange(args.cells + 1, dtype=np.int64) * n
        c0, c1 = W.shard_cells(off_all, rank, world)
        ncell = c1 - c0
        vs, ws, ss = [], [], []
        for k in range(c0, c1):
            wl = W.make(0, n_per_species=nps, seed=10_000 + k, shuffled=True)
            vs.append(wl.v); ws.append(wl.w); ss.append(wl.species_id)
        off = off_all[c0:c1 + 1] - off_all[c0]
        v = torch.tensor(np.concatenate(vs), device=dev); w = torch.tensor(np.concatenate(ws), device=dev)
        sid = torch.tensor(np.concatenate(ss), device=dev)
        out = torch.empty_like(v)
        dt = args.dt
        g.cells_run(off, v, w, sid, 1, dt, 1e-12, 50, out=out)      # warm-up
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        e0.record()
        rc, out, info = g.cells_run(off, v, w, sid, args.steps, dt, 1e-12, 50, out=out)
        e1.record()
        torch.cuda.synchronize()
        t_batch = e0.elapsed_time(e1) * 1e-3
        iters = int(info["iterations"].sum())
        wm = (w * torch.tensor(base.mass, device=dev)[sid.long()])[:, None]
        K0 = 0.5 * (wm * v * v).sum().item(); K1 = 0.5 * (wm * out * out).sum().item()
        dP = (wm * (out - v)).reshape(ncell, n, 3).sum(1).abs().max().item() / (wm * v.abs()).sum().item() * ncell
        # the same cells through the single-cell path
        ns = min(args.sequential_cells, ncell)
        torch.cuda.synchronize()
        e0.record()
        for k in range(ns):
            a, b = int(off[k]), int(off[k + 1])
            g.set_markers(v[a:b], w[a:b], sid[a:b])
            g.run(args.steps, dt, 1e-12, 50)
            g.get_markers()
        e1.record()
        torch.cuda.synchronize()
        t_seq = e0.elapsed_time(e1) * 1e-3 / ns * ncell
        notconv = int(info["steps_not_converged"].sum()); allconv = bool((info["status"] == 0).all())
        if world > 1:
            # whole-job figures: MAX of the times, SUM of the work, worst drift
            tmax = torch.tensor([t_batch, t_seq, abs(K1 - K0) / K0, dP], dtype=torch.float64, device=dev)
            tsum = torch.tensor([float(iters), float(notconv), float(not allconv)], dtype=torch.float64, device=dev)
            dist.all_reduce(tmax, op=dist.ReduceOp.MAX); dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
            t_batch, t_seq, dK, dP = (float(x) for x in tmax)
            iters, notconv, allconv = int(tsum[0]), int(tsum[1]), tsum[2].item() == 0.0
        else:
            dK = abs(K1 - K0) / K0
        if rank == 0:
            print(json.dumps({"cells": args.cells, "n_gpus": world, "markers_per_cell": n, "steps": args.steps,
                              "batch_cell_steps_per_s": args.cells * args.steps / t_batch,
                              "batch_pairs_per_s": iters * n * (n - 1) / t_batch, "batch_ms": 1e3 * t_batch,
                              "iterations_per_step_mean": iters / (args.cells * args.steps),
                              "all_converged": allconv, "dt": dt,
                              "cell_steps_not_converged": notconv,
                              "sequential_cell_steps_per_s": args.cells * args.steps / t_seq,
                              "speedup_vs_sequential": t_seq / t_batch,
                              "energy_drift_rel": dK, "momentum_drift_rel_worst_cell": dP}), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
