"""Moment / temperature / entropy histories of BASELINE configs 1-3 on the CUDA path, with the analytic
curves the paper compares against (north_star: "multi-step runs are compared by their moment and temperature
histories").

    python -m paper_2212_00663_b200.histories --config 1 [--n-per-species N] [--steps K] [--out DIR]

Runs `landau_step` K times on cuda:0 (device-driven fixed point), reads `landau_moments` (+ `_ext`) after every
step, and writes  DIR/history_c<config>.csv  (one row per step) and  DIR/history_c<config>.json  (summary:
conservation drifts, iteration counts, fitted vs analytic rates).  Nothing here touches oracle/.

Analytic comparisons (paper_2212_00663_b200.analytic):
  config 1  e-i temperature relaxation: fitted d ln(T_e - T_i)/dt  vs  Eqs. (44)-(45), PAPER.md:271-275;
  config 2  isotropisation: T_par - T_perp of the electrons at t_end  vs  the ODE of Eqs. (40)-(41),
            PAPER.md:251-261 (like-particle formula; e-i scattering adds to it, so the run relaxes faster);
  config 3  thermalisation of a shell: S_eps history (Eq. 20) and per-axis kurtosis 9/5 -> 3.
"""
from __future__ import annotations

import argparse
import json
import time
from pathlib import Path

import numpy as np

from . import analytic as A
from . import binding as B
from . import workloads as W


def _kurtosis(mass, n, P, stress, m4):
    """kappa_i = n_s sum w (v_i-u_i)^4 / (sum w (v_i-u_i)^2)^2; Maxwellian 3, thin shell 9/5."""
    m2 = (stress[:, :3] - P ** 2 / (mass * n)[:, None]) / mass[:, None]
    return n[:, None] * m4 / m2 ** 2


def run_history(config: int, n_per_species=None, steps=None, every_ext: int = 1, verbose: bool = False,
                solver: int = 0, depth: int = 3, substep: int = 0, n_q=None, max_iter=None, stiff: float = 0.0, eps_rule=None):
    wl = W.make(config, n_per_species=n_per_species, **({} if eps_rule is None else {"eps_rule": float(eps_rule)}))
    if n_q is not None:
        wl.n_q = int(n_q)
    if max_iter is not None:
        wl.max_iter = int(max_iter)
    n_steps = int(steps if steps is not None else wl.n_steps)
    g = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    if solver:
        g.set_solver(solver, depth)
    if substep:
        g.set_substep(substep)
    if stiff:
        g.set_stiff_pairs(stiff)
    g.set_markers(wl.v, wl.w, wl.species_id)
    S = wl.n_species
    stiff_pairs = []
    cols = dict(t=[], iterations=[], residual=[], converged=[], K=[], S_eps=[], T=[], T_axis=[], kurt=[], P=[])

    def sample(t, info):
        m = g.moments(with_entropy=True)
        stress, m4 = g.moments_ext()
        tm = A.temperatures_from_moments(wl.mass, m["n"], m["P"], m["K"], stress)
        cols["t"].append(t)
        cols["iterations"].append(info[0]); cols["residual"].append(info[1]); cols["converged"].append(info[2])
        cols["K"].append(m["K"].copy()); cols["S_eps"].append(m["S_eps"].copy()); cols["P"].append(m["P"].copy())
        cols["T"].append(tm["T"].copy()); cols["T_axis"].append(tm["T_axis"].copy())
        cols["kurt"].append(_kurtosis(wl.mass, m["n"], m["P"], stress, m4))
        return m

    t0 = time.time()
    m0 = sample(0.0, (0, 0.0, True))
    not_conv = 0
    for k in range(n_steps):
        rc, it, res, conv = g.step(wl.dt, wl.tol, wl.max_iter)
        not_conv += 0 if conv else 1
        if stiff:
            stiff_pairs.append(g.stiff_pairs_last()[0])
        sample((k + 1) * wl.dt, (it, res, conv))
        if verbose and (k + 1) % 50 == 0:
            print(f"  step {k + 1}/{n_steps}: {it} iterations, T = {cols['T'][-1]}", flush=True)
    wall = time.time() - t0
    H = {k: np.array(v) for k, v in cols.items()}
    K = H["K"].sum(axis=1)
    Ptot = H["P"].sum(axis=1)
    wm_abs = float((wl.w * wl.mass[wl.species_id] * np.abs(wl.v).sum(axis=1)).sum())
    summary = dict(config=config, workload=wl.name, n_markers=wl.n_markers, n_species=S, steps=n_steps, dt=wl.dt,
                   n_q=wl.n_q, eps=wl.eps.tolist(), kernels=g.last_kernels(),
                   solver={0: "jacobi", 1: f"anderson depth {depth}", 2: f"newton-krylov restart {depth}"}[solver],
                   substep_levels=substep, wall_s=wall,
                   steps_per_s=n_steps / wall, iterations_mean=float(H["iterations"][1:].mean()),
                   pass2_evaluations_total=int(H["iterations"][1:].sum()), max_iter=wl.max_iter, stiff_theta=stiff,
                   stiff_pairs_per_step_max=int(max(stiff_pairs)) if stiff_pairs else 0,
                   steps_with_stiff_pairs=int(sum(1 for x in stiff_pairs if x > 0)),
                   iterations_max=int(H["iterations"].max()), steps_not_converged=not_conv,
                   energy_drift_rel_max=float(np.abs(K - K[0]).max() / K[0]),
                   energy_drift_rel_per_step_max=float(np.abs(np.diff(K)).max() / K[0]),
                   momentum_drift_rel_max=float(np.abs(Ptot - Ptot[0]).max() / wm_abs),
                   S_eps_total_first_last=[float(H["S_eps"][0].sum()), float(H["S_eps"][-1].sum())],
                   S_eps_monotone=bool(np.all(np.diff(H["S_eps"].sum(axis=1)) >= -1e-12 * abs(H["S_eps"][0].sum()))),
                   T_first=H["T"][0].tolist(), T_last=H["T"][-1].tolist())
    coupling = A.coupling_from_nu(wl.nu0 * wl.charge[0] ** 4)
    t = H["t"]
    if config == 1 and S >= 2:
        gap = H["T"][:, 0] - H["T"][:, 1]
        n = m0["n"]
        rate_ana = A.temperature_gap_rate(wl.mass[0], wl.mass[1], n[0], n[1], H["T"][0, 0], H["T"][0, 1],
                                          A.coupling_from_nu(wl.nu0 * wl.charge[0] ** 2 * wl.charge[1] ** 2))
        rate_fit = A.fit_exponential_rate(t, gap)
        summary["temperature_gap"] = dict(first=float(gap[0]), last=float(gap[-1]), fitted_rate=rate_fit,
                                          analytic_rate_eq45=rate_ana, fitted_over_analytic=rate_fit / rate_ana)
    if config == 2:
        Tpar, Tperp = H["T_axis"][:, 0, 2], 0.5 * (H["T_axis"][:, 0, 0] + H["T_axis"][:, 0, 1])
        ta, Tpa, Tpe = A.integrate_isotropisation(wl.mass[0], m0["n"][0], Tpar[0], Tperp[0], coupling, t[-1])
        summary["anisotropy"] = dict(first=float(Tpar[0] - Tperp[0]), last=float(Tpar[-1] - Tperp[-1]),
                                     analytic_last_eq41=float(Tpa[-1] - Tpe[-1]),
                                     fitted_rate=A.fit_exponential_rate(t, Tpar - Tperp),
                                     analytic_initial_rate=-1.5 * A.isotropisation_rate(
                                         wl.mass[0], m0["n"][0], Tpar[0], Tperp[0], coupling))
    if config == 3:
        summary["kurtosis_e_first_last"] = [H["kurt"][0, 0].tolist(), H["kurt"][-1, 0].tolist()]
        summary["S_eps_e_first_last"] = [float(H["S_eps"][0, 0]), float(H["S_eps"][-1, 0])]
    return wl, H, summary


def write(outdir: Path, config, H, summary):
    outdir.mkdir(parents=True, exist_ok=True)
    S = H["T"].shape[1]
    hdr = (["t", "iterations", "residual", "converged", "K_total", "S_eps_total"] + [f"T_{s}" for s in range(S)]
           + [f"T{ax}_{s}" for s in range(S) for ax in "xyz"] + [f"kurt{ax}_{s}" for s in range(S) for ax in "xyz"]
           + [f"S_eps_{s}" for s in range(S)])
    rows = np.column_stack([H["t"], H["iterations"], H["residual"], H["converged"], H["K"].sum(axis=1),
                            H["S_eps"].sum(axis=1), H["T"], H["T_axis"].reshape(len(H["t"]), -1),
                            H["kurt"].reshape(len(H["t"]), -1), H["S_eps"]])
    np.savetxt(outdir / f"history_c{config}.csv", rows, delimiter=",", header=",".join(hdr), comments="")
    (outdir / f"history_c{config}.json").write_text(json.dumps(summary, indent=1))


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--config", type=int, required=True, choices=[0, 1, 2, 3])
    ap.add_argument("--n-per-species", type=int, default=None)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--out", default="gpurun_out")
    ap.add_argument("--solver", choices=["jacobi", "anderson", "newton"], default="jacobi")
    ap.add_argument("--anderson-depth", type=int, default=3)
    ap.add_argument("--newton-restart", type=int, default=20)
    ap.add_argument("--n-q", type=int, default=None, help="Gauss-Hermite knots per axis (default: the workload's, 4)")
    ap.add_argument("--max-iter", type=int, default=None)
    ap.add_argument("--eps-rule", type=float, default=None, help="eps_s = EPS_RULE * T_s/m_s (default 0.05, reading U2)")
    ap.add_argument("--stiff", type=float, default=0.0,
                    help="landau_set_stiff_pairs threshold (0 = off): stiff two-marker interactions solved implicitly")
    ap.add_argument("--substep", type=int, default=0, help="levels of step halving for unconverged steps")
    ap.add_argument("--tag", default="", help="suffix of the output file names")
    args = ap.parse_args()
    solver = {"jacobi": 0, "anderson": 1, "newton": 2}[args.solver]
    wl, H, summary = run_history(args.config, args.n_per_species, args.steps, verbose=True, solver=solver,
                                 depth=args.newton_restart if solver == 2 else args.anderson_depth,
                                 substep=args.substep, n_q=args.n_q, max_iter=args.max_iter, stiff=args.stiff, eps_rule=args.eps_rule)
    write(Path(args.out), f"{args.config}{args.tag}", H, summary)
    print(json.dumps(summary))


if __name__ == "__main__":
    main()
