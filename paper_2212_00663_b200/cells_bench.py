"""Throughput of the batched collision-cell path (landau_cells_run) against the single-cell path.

    python -m paper_2212_00663_b200.cells_bench [--cells 1184] [--per-species 64 128 256 512] [--steps 5]

Synthetic PIC-like batch: `cells` independent cells, each an e-i plasma shaped like BASELINE config 0 (2 species,
Maxwellian, T_e = 1, T_i = 0.5, random weights) with its own seed.  Reports cell-steps/s and ordered pass-2 pairs/s
of the one-launch batch (CUDA events), the same cells stepped one after the other through landau_set_markers +
landau_run (what a caller without the batch entry point would do), and the conservation drifts of the batch.
Prints one JSON line per cell size.
"""
from __future__ import annotations

import argparse
import json

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
    base = W.make(0, n_per_species=8)
    g = B.Landau(base.mass, base.charge, base.eps)
    dev = torch.device("cuda", 0)
    for nps in args.per_species:
        vs, ws, ss = [], [], []
        for k in range(args.cells):
            wl = W.make(0, n_per_species=nps, seed=10_000 + k, shuffled=True)
            vs.append(wl.v); ws.append(wl.w); ss.append(wl.species_id)
        n = 2 * nps
        off = np.arange(args.cells + 1, dtype=np.int64) * n
        v = torch.tensor(np.concatenate(vs), device=dev); w = torch.tensor(np.concatenate(ws), device=dev)
        sid = torch.tensor(np.concatenate(ss), device=dev)
        out = torch.empty_like(v)
        dt = args.dt
        g.cells_run(off, v, w, sid, 1, dt, 1e-12, 50, out=out)      # warm-up
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        rc, out, info = g.cells_run(off, v, w, sid, args.steps, dt, 1e-12, 50, out=out)
        e1.record()
        torch.cuda.synchronize()
        t_batch = e0.elapsed_time(e1) * 1e-3
        iters = int(info["iterations"].sum())
        wm = (w * torch.tensor(base.mass, device=dev)[sid.long()])[:, None]
        K0 = 0.5 * (wm * v * v).sum().item(); K1 = 0.5 * (wm * out * out).sum().item()
        dP = (wm * (out - v)).reshape(args.cells, n, 3).sum(1).abs().max().item() / (wm * v.abs()).sum().item() * args.cells
        # the same cells through the single-cell path
        ns = min(args.sequential_cells, args.cells)
        torch.cuda.synchronize()
        e0.record()
        for k in range(ns):
            a, b = int(off[k]), int(off[k + 1])
            g.set_markers(v[a:b], w[a:b], sid[a:b])
            g.run(args.steps, dt, 1e-12, 50)
            g.get_markers()
        e1.record()
        torch.cuda.synchronize()
        t_seq = e0.elapsed_time(e1) * 1e-3 / ns * args.cells
        print(json.dumps({"cells": args.cells, "markers_per_cell": n, "steps": args.steps,
                          "batch_cell_steps_per_s": args.cells * args.steps / t_batch,
                          "batch_pairs_per_s": iters * n * (n - 1) / t_batch, "batch_ms": 1e3 * t_batch,
                          "iterations_per_step_mean": iters / (args.cells * args.steps),
                          "all_converged": bool((info["status"] == 0).all()), "dt": dt,
                          "cell_steps_not_converged": int(info["steps_not_converged"].sum()),
                          "sequential_cell_steps_per_s": args.cells * args.steps / t_seq,
                          "speedup_vs_sequential": t_seq / t_batch,
                          "energy_drift_rel": abs(K1 - K0) / K0, "momentum_drift_rel_worst_cell": dP}), flush=True)


if __name__ == "__main__":
    main()
