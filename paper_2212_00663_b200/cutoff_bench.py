"""Pass 1 with and without the Gaussian cutoff (second half).

    python -m paper_2212_00663_b200.cutoff_bench [--out gpurun_out/cutoff_bench.md]

Workloads: the paper's own meshes (workloads.paper_test, test 3.3: electrons + deuterons on an N x N mesh, 2-V) with
its mollifier rule eps_s = 1.2 (L_s/N)^1.98, N = 32 ... 256; BASELINE config 4 (3-V Maxwellians,
lognormal weights) at eps_s = 0.05 T/m (the config's value) and at smaller mollifiers.  For each: the pass-1 kernels'
time (CUDA events around bounds + tile boxes + tables + node-sum kernel, landau_profile_*) and the fraction of
(target block, source tile) pairs skipped, for  all pairs / cutoff in caller order / cutoff after Morton bucketing,
plus the largest difference of G between the variants (the oracle comparison is tests/test_gpu_parity.py).
Nothing here touches oracle/.
"""
from __future__ import annotations

import argparse
from pathlib import Path

import numpy as np

from . import binding as B
from . import workloads as W


def measure(wl, cutoff, morton, reps=3, entropy_kernel=0):
    g = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0, entropy_kernel=entropy_kernel)
    g.set_cutoff(cutoff, morton)
    G = g.entropy_grad(wl.v, wl.w, wl.species_id)          # warm-up, sizes every buffer
    g.profile_enable(True)
    for _ in range(reps):
        G = g.entropy_grad(wl.v, wl.w, wl.species_id)
    pr = g.profile_read()
    g.profile_enable(False)
    considered, skipped = g.cutoff_stats()
    return dict(ms=pr["entropy_ms"] / max(pr["entropy_launches"], 1), considered=considered, skipped=skipped,
                kernels=g.last_kernels(), G=G.cpu().numpy())


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default="gpurun_out/cutoff_bench.md")
    ap.add_argument("--max-grid", type=int, default=256)
    args = ap.parse_args()
    cases = []
    for n in (32, 64, 128, 256):
        if n <= args.max_grid:
            cases.append((f"paper test 3.3 mesh {n}x{n} (2 x {n * n} markers, 2-V), eps = 1.2 (L/N)^1.98", W.paper_test(3, n_grid=n)))
    for nps, rule in ((1 << 14, 0.05), (1 << 14, 0.005), (1 << 14, 0.0005), (1 << 16, 0.05), (1 << 16, 0.002)):
        cases.append((f"config 4, 3 x {nps} markers (3-V, shuffled), eps = {rule} T/m",
                      W.make(4, n_per_species=nps, shuffled=True, eps_rule=rule)))
    lines = ["| workload | kernel | all pairs ms | cutoff (caller order) ms | skipped | cutoff + Morton ms | skipped | speed-up | max rel. diff of G |",
             "|---|---|---|---|---|---|---|---|---|"]
    for name, wl in cases:
        a = measure(wl, False, False)
        b = measure(wl, True, False)
        c = measure(wl, True, True)
        nrm = np.linalg.norm(a["G"])
        diff = max(np.linalg.norm(b["G"] - a["G"]), np.linalg.norm(c["G"] - a["G"])) / nrm
        fb = b["skipped"] / max(b["considered"], 1)
        fc = c["skipped"] / max(c["considered"], 1)
        line = (f"| {name} | {c['kernels'].split('entropy=')[-1].split()[0]} | {a['ms']:.3f} | {b['ms']:.3f} | {100 * fb:.1f} % | "
                f"{c['ms']:.3f} | {100 * fc:.1f} % | {a['ms'] / c['ms']:.2f}x | {diff:.1e} |")
        print(line, flush=True)
        lines.append(line)
    out = Path(args.out)
    out.parent.mkdir(parents=True, exist_ok=True)
    out.write_text("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()
