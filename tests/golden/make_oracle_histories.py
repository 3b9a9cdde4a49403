#!/usr/bin/env python
"""Write the ORACLE's moment histories of BASELINE configs 0-3 to tests/golden/oracle_history_*.csv.

    python tests/golden/make_oracle_histories.py --config 1 --steps 200 [--n-per-species N]
           [--entropy-every 10] [--threads T] [--out tests/golden] [--resume]

This script calls ONLY oracle/ (the plain CPU restatement of PAPER.md) and the seeded input generator
paper_2212_00663_b200/workloads.py (random draws, none of the method's arithmetic).  Nothing here touches the
CUDA path, so the stored values are expected values in the sense of the parity contract: `tests/
test_gpu_history_parity.py` runs the CUDA path on the same seeded cloud and compares its per-step moments with
these files (north_star: "multi-step runs are compared by their moment and temperature histories";
SURVEY.md section 8(d) "Oracle timing beside it": full-length oracle histories for c0 and c1, the first steps at
full size for c2 and c3, full-length runs at N_s = 2048).

Every step is landau_ref_step = Eqs. (24)-(25) by the Jacobi fixed point of Algorithm 1
 with tol / max_iter of the workload; each row records the oracle's own iteration count,
final residual and converged flag, so that a step the oracle ALSO fails to converge can
be told apart from a defect of the CUDA path.  Moments per row: n_s (Eq. 33), P_s (Eq. 26), K_s (Eq. 28), the
second moments m_s sum w v_i v_j and central fourth moments (per-axis temperatures Eqs. 30-31, kurtosis), and,
every `--entropy-every` steps (it costs one more pass 1 of the oracle), S_eps,s (Eq. 20); other rows hold nan there.

Rows are appended and flushed as they are computed; with --resume the run continues from the state saved next to
the CSV (`<name>.state.npz`, git-ignored) after the last complete row.
"""
from __future__ import annotations

import argparse
import sys
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parents[2]
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

from oracle import landau_ref  # noqa: E402
from paper_2212_00663_b200 import workloads as W  # noqa: E402


def columns(S: int):
    c = ["step", "t", "iterations", "residual", "converged", "oracle_seconds"]
    c += [f"n_{s}" for s in range(S)]
    c += [f"P{a}_{s}" for s in range(S) for a in "xyz"]
    c += [f"K_{s}" for s in range(S)]
    c += [f"S_eps_{s}" for s in range(S)]
    c += [f"stress_{ij}_{s}" for s in range(S) for ij in ("xx", "yy", "zz", "xy", "xz", "yz")]
    c += [f"m4{a}_{s}" for s in range(S) for a in "xyz"]
    return c


def moment_row(o, S, with_entropy):
    m = o.moments(with_entropy=with_entropy)
    stress, m4 = o.moments_ext()
    Seps = m["S_eps"] if with_entropy else np.full(S, np.nan)
    return np.concatenate([m["n"], m["P"].ravel(), m["K"], Seps, stress.ravel(), m4.ravel()])


def file_stem(config: int, n_per_species: int, steps: int) -> str:
    return f"oracle_history_c{config}_n{n_per_species}_s{steps}"


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--config", type=int, required=True, choices=[0, 1, 2, 3])
    ap.add_argument("--n-per-species", type=int, default=None)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--entropy-every", type=int, default=10, help="S_eps every k steps (0 = first and last row only)")
    ap.add_argument("--threads", type=int, default=0, help="OpenMP threads of the oracle (0 = all)")
    ap.add_argument("--out", default=str(Path(__file__).resolve().parent))
    ap.add_argument("--resume", action="store_true")
    args = ap.parse_args()

    landau_ref.build()
    if args.threads > 0:
        landau_ref.set_num_threads(args.threads)
    wl = W.make(args.config, n_per_species=args.n_per_species)
    nps = int(wl.counts()[0])
    steps = int(args.steps if args.steps is not None else wl.n_steps)
    S = wl.n_species
    out = Path(args.out)
    out.mkdir(parents=True, exist_ok=True)
    stem = file_stem(args.config, nps, steps)
    csv, state = out / f"{stem}.csv", out / f"{stem}.state.npz"
    o = landau_ref.LandauRef(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    cols = columns(S)

    def want_entropy(k):
        return k == 0 or k == steps or (args.entropy_every > 0 and k % args.entropy_every == 0)

    start = 0
    if args.resume and csv.exists() and state.exists():
        st = np.load(state)
        start = int(st["step"])
        o.set_markers(st["v"], wl.w, wl.species_id)
        lines = csv.read_text().splitlines()
        keep = [ln for ln in lines if ln.startswith("#") or ln.startswith("step,") or int(float(ln.split(",")[0])) <= start]
        csv.write_text("\n".join(keep) + "\n")
        fh = csv.open("a")
        print(f"resuming {stem} after step {start}", flush=True)
    else:
        o.set_markers(wl.v, wl.w, wl.species_id)
        fh = csv.open("w")
        fh.write(f"# oracle moment history: BASELINE config {args.config} ({wl.name}), {S} species x {nps} markers, seed {wl.seed}, "
                 f"unshuffled, n_q = {wl.n_q}, nu0 = {wl.nu0}, dt = {wl.dt!r}, tol = {wl.tol!r}, max_iter = {wl.max_iter}\n")
        fh.write(f"# written by: python tests/golden/make_oracle_histories.py --config {args.config} --n-per-species {nps} "
                 f"--steps {steps} --entropy-every {args.entropy_every}   (calls only oracle/; {landau_ref.num_threads()} threads)\n")
        fh.write("# eps = " + " ".join(repr(float(e)) for e in wl.eps) + "\n")
        fh.write(",".join(cols) + "\n")
        row = np.concatenate([[0, 0.0, 0, 0.0, 1, 0.0], moment_row(o, S, True)])
        fh.write(",".join(repr(float(x)) for x in row) + "\n")
        fh.flush()
    t_all = time.time()
    for k in range(start + 1, steps + 1):
        t0 = time.time()
        rc, it, res, conv = o.step(wl.dt, wl.tol, wl.max_iter)
        sec = time.time() - t0
        row = np.concatenate([[k, k * wl.dt, it, res, int(conv), sec], moment_row(o, S, want_entropy(k))])
        fh.write(",".join(repr(float(x)) for x in row) + "\n")
        fh.flush()
        np.savez(state, step=k, v=o.get_markers())
        print(f"{stem}: step {k}/{steps}: {it} iterations, residual {res:.2e}, converged {conv}, {sec:.1f} s "
              f"(total {time.time() - t_all:.0f} s)", flush=True)
    fh.close()
    if state.exists():
        state.unlink()
    print(f"wrote {csv}")


if __name__ == "__main__":
    main()
