#!/usr/bin/env python
"""bench.py -- one JSON line for the hot path of arXiv:2212.00663 on B200 (contract: DESIGN.md "Measurement").

A "step" is one pass of the WHOLE hot path over one synthetic marker
cloud: pack/bucket (landau_set_markers), pass 1 (entropy gradient), the implicit step of Eq. (24) with
pass 2 once per fixed-point iteration, update/residual, diagnostics (landau_moments incl. S_eps, which
costs a second pass 1) and the read-back of the new velocities (landau_get_markers).

    python bench.py --gpus 1 --steps 5 --warmup 3                  # the CUDA path
    python bench.py --impl reference --steps 2 --warmup 1          # the CPU oracle, bounded sample

metric  = pair interactions per second (FP64): ordered (target, source) evaluations of Eq. (23) done by
          the fixed-point iterations of the timed steps, divided by the time of the whole steps.
e2e     = the same, through the *_host entry points: host->device copies of (v, w, species_id) and the
          device->host read of the new velocities inside the timed region, every step.
N > 1   : the path does not shard (north_star: one GPU, no collectives): --gpus N runs N independent
          replicas ("replicas only"), value = pairs of all replicas / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_2212_00663_b200 import workloads as W  # noqa: E402

METRIC = "pair_interactions_per_s"
UNIT = "pairs/s"
FLOPS_PER_PAIR = 33.0          # canonical algorithmic count of one ordered pair
# nominal FP64 vector peak: 148 SMs x 64 FP64 FMA lanes x 2 flop x 1.965 GHz
FP64_PEAK_NOMINAL = 148 * 64 * 2 * 1.965e9

WORKLOADS = {
    # name: (config index, markers per species)
    "c4_2e16": (4, 1 << 16),
    "c4_2e15": (4, 1 << 15),
    "c4_2e14": (4, 1 << 14),
    "c4_2e17": (4, 1 << 17),
    "c1": (1, 4096),
    "c0": (0, 256),
    "c2": (2, 8192),
    "c3": (3, 32768),
}
DEFAULT_WORKLOAD = "c4_2e16"     # >= 1e5 markers: the size north_star's roofline target is quoted on
# fixed-point iterations one step of each workload takes: the "ms/step (iters)" column of BASELINE.md section 3,
# measured on the GPU path; used only to scale the oracle's bounded sample in --impl reference (which must not
# touch the GPU) to the pass-1 / pass-2 mix of the step the GPU arm runs
# The table lives in bench_iters.json (tracked): the GPU arm rewrites a workload's entry whenever a default Jacobi run
# measures a different count, so the two arms cannot drift apart unnoticed.
REF_ITERS_FILE = ROOT / "bench_iters.json"


def ref_iters(workload):
    return int(json.loads(REF_ITERS_FILE.read_text())["iterations_per_step"][workload])


def record_iters(workload, iters):
    """GPU arm, rank 0: keep bench_iters.json equal to what the CUDA path measures (no-op when it already is)."""
    try:
        d = json.loads(REF_ITERS_FILE.read_text())
        if d["iterations_per_step"].get(workload) != int(iters):
            d["iterations_per_step"][workload] = int(iters)
            REF_ITERS_FILE.write_text(json.dumps(d, indent=1) + "\n")
    except (OSError, ValueError, KeyError):
        pass


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="budget of the oracle sample")
    ap.add_argument("--pair-kernel", type=int, default=0)
    ap.add_argument("--entropy-kernel", type=int, default=0)
    ap.add_argument("--solver", choices=["jacobi", "anderson", "newton"], default="jacobi",
                    help="solver of Eq. (24): the paper's Jacobi iteration (default), Anderson or Newton-Krylov (NEXT-4)")
    ap.add_argument("--anderson-depth", type=int, default=3)
    ap.add_argument("--newton-restart", type=int, default=20)
    ap.add_argument("--no-dg", action="store_true", help="skip the discrete-gradient step block (NEXT-1)")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for k, nm in enumerate(names):
                if len(r) > 3 + k and r[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample(wl, iters, seconds, name):
    """The oracle, as it stands, on a bounded sample: a random subset of target rows of pass 1 and
    pass 2 against all sources.  Returns (pairs/s extrapolated to the whole path, dict)."""
    from oracle import landau_ref
    landau_ref.build()
    o = landau_ref.LandauRef(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    N = wl.n_markers
    rng = np.random.default_rng(12345)
    G = rng.standard_normal((N, 3))
    # calibrate on a few rows, then size the sample for ~`seconds`
    rows = rng.choice(N, size=min(N, 16), replace=False).astype(np.int64)
    t0 = time.perf_counter(); o.pair_field_rows(wl.v, wl.w, wl.species_id, G, rows); tp = (time.perf_counter() - t0) / len(rows)
    t0 = time.perf_counter(); o.entropy_grad_rows(wl.v, wl.w, wl.species_id, rows[:8]); te = (time.perf_counter() - t0) / 8
    per_row = te + iters * tp
    m = int(max(8, min(N, seconds / max(per_row, 1e-9))))
    rows = rng.choice(N, size=m, replace=False).astype(np.int64)
    t0 = time.perf_counter()
    o.entropy_grad_rows(wl.v, wl.w, wl.species_id, rows)
    t_e = time.perf_counter() - t0
    t0 = time.perf_counter()
    for _ in range(iters):
        o.pair_field_rows(wl.v, wl.w, wl.species_id, G, rows)
    t_p = time.perf_counter() - t0
    pairs = float(iters) * m * (N - 1)
    value = pairs / (t_e + t_p)
    info = {"value": value, "unit": UNIT, "cores": landau_ref.num_threads(), "kind": "oracle",
            "sample": f"{name}: {m} of {N} target rows against all sources; pass 1 once ({t_e:.2f} s) + pass 2 x {iters} "
                      f"iterations ({t_p:.2f} s); pairs = iterations*rows*(N-1); pass-2-only rate "
                      f"{pairs / t_p:.3e} pairs/s"}
    return value, info, (t_e + t_p)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg, nps = WORKLOADS[args.workload]
    wl = W.make(cfg, n_per_species=nps)
    iters = ref_iters(args.workload)
    per_step = max(2.0, min(args.cpu_seconds, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample(wl, iters, per_step, args.workload)
    vals, infos, times = [], [], []
    for _ in range(args.steps):
        v, info, t = oracle_sample(wl, iters, per_step, args.workload)
        vals.append(v); infos.append(info); times.append(t)
    value = float(np.mean(vals))
    info = dict(infos[-1]); info["value"] = value
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(times)), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "reference",
            "config": config_dict(args, wl, iters), "cpu_baseline": info,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def config_dict(args, wl, iters=None):
    d = {"workload": f"{args.workload}: {wl.name}, {wl.n_species} species x {int(wl.counts()[0])} markers "
                     f"(N = {wl.n_markers}), FP64, n_q = {wl.n_q}, dt = {wl.dt}, tol = {wl.tol}, max_iter = {wl.max_iter}",
         "n_markers": wl.n_markers, "n_species": wl.n_species,
         "step": "set_markers + landau_step (pass 1, fixed-point iterations of pass 2) + moments(S_eps) + get_markers",
         "l2": "inputs re-packed every step; pass-2 working set is L2-resident by design (56 B/marker); "
               "compute-bound path, cache state does not change the timing",
         "parallelism": "replicas only" if args.gpus > 1 else "single GPU",
         "solver": {"jacobi": "jacobi (paper)", "anderson": f"anderson depth {args.anderson_depth}",
                    "newton": f"newton-krylov restart {args.newton_restart}"}[getattr(args, "solver", "jacobi")]}
    if iters is not None:
        d["iterations_per_step"] = iters
    return d


def aggregate_over_ranks(times, pairs):
    """Contract of the multi-rank line ("replicas only"): time = MAX over ranks, work = SUM
    over ranks.  `times` / `pairs` are tensors on the backend's device (cuda for nccl, cpu for gloo); a
    no-op without an initialised process group.  Covered on CPU by tests/test_bench_multirank.py (gloo)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(times, op=dist.ReduceOp.MAX)
        dist.all_reduce(pairs, op=dist.ReduceOp.SUM)
    return times.tolist(), pairs.tolist()


def ncu_traffic(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed summary of
    an `ncu --set full` capture (profiles/ncu_traffic.csv: workload,kernel,dram_read_bytes,dram_write_bytes,source).
    None when no capture is on file for this workload / kernel."""
    try:
        for ln in (ROOT / "profiles" / "ncu_traffic.csv").read_text().splitlines():
            f = [x.strip() for x in ln.split(",")]
            if len(f) >= 5 and f[0] == workload and f[1] == kernel:
                return {"bytes": float(f[2]) + float(f[3]), "source": f[4]}
    except (OSError, ValueError):
        pass
    return None


def run_ours(args):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2212_00663_b200 import binding as B

    cfg, nps = WORKLOADS[args.workload]
    wl = W.make(cfg, n_per_species=nps, seed=cfg + 1000 * rank)       # replicas differ by seed
    N = wl.n_markers
    g = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0, pair_kernel=args.pair_kernel,
                 entropy_kernel=args.entropy_kernel)
    if args.solver == "anderson":
        g.set_solver(1, args.anderson_depth)
    if args.solver == "newton":
        g.set_solver(2, args.newton_restart)
    dev = torch.device("cuda", local)
    v_d = torch.tensor(wl.v, device=dev); w_d = torch.tensor(wl.w, device=dev)
    s_d = torch.tensor(wl.species_id, device=dev)
    v_h = torch.from_numpy(wl.v).pin_memory(); w_h = torch.from_numpy(wl.w).pin_memory()
    s_h = torch.from_numpy(wl.species_id).pin_memory()
    out_h = torch.empty((N, 3), dtype=torch.float64).pin_memory()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step_device():
        g.set_markers(v_d, w_d, s_d)
        rc, it, res, conv = g.step(wl.dt, wl.tol, wl.max_iter)
        m = g.moments(with_entropy=True)
        vnew = g.get_markers()
        return it, conv, m, vnew

    lib, h = g._lib, g._h

    def step_host():
        rc = lib.landau_set_markers_host(h, N, v_h.data_ptr(), w_h.data_ptr(), s_h.data_ptr())
        assert rc == 0, rc
        g.N = N
        rc, it, res, conv = g.step(wl.dt, wl.tol, wl.max_iter)
        m = g.moments(with_entropy=True)
        rc = lib.landau_get_markers_host(h, out_h.data_ptr())
        assert rc == 0, rc
        return it, conv, m

    g.set_markers(v_d, w_d, s_d)
    m0 = g.moments(with_entropy=False)          # invariants of the initial cloud
    for _ in range(max(args.warmup, 1)):
        step_device()
    # ---- device-resident timed region
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    # per-kernel CUDA events ride in the timed region, except for clouds small enough for the CUDA-graph step
    # (landau_set_step_graph, <= 65536 slots): graph replays cannot carry per-kernel events, so those workloads
    # get their kernel times from extra profiled steps after the timed region
    prof_in_timed = N > 60000
    if prof_in_timed:
        g.profile_enable(True)
    l0 = g.launch_count()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    iters_total, all_conv = 0, True
    e0.record()
    for _ in range(args.steps):
        it, conv, m1, vnew = step_device()
        iters_total += it; all_conv &= bool(conv)
    e1.record()
    barrier()
    t_dev = e0.elapsed_time(e1) * 1e-3
    t_prof = t_dev
    if prof_in_timed:
        prof = g.profile_read()
        g.profile_enable(False)
    launches = g.launch_count() - l0
    clocks = sampler.stop()
    if not prof_in_timed:
        g.profile_enable(True)
        e0.record()
        for _ in range(2):
            step_device()
        e1.record()
        torch.cuda.synchronize()
        t_prof = e0.elapsed_time(e1) * 1e-3
        prof = g.profile_read()
        g.profile_enable(False)
    # ---- end-to-end timed region (host buffers)
    step_host()
    barrier()
    e0.record()
    it_h = 0
    for _ in range(args.steps):
        it, conv, _m = step_host()
        it_h += it
    e1.record()
    barrier()
    t_e2e = e0.elapsed_time(e1) * 1e-3

    times = torch.tensor([t_dev, t_e2e], dtype=torch.float64, device=dev)
    pairs = torch.tensor([float(iters_total) * N * (N - 1), float(it_h) * N * (N - 1)], dtype=torch.float64, device=dev)
    (t_dev_max, t_e2e_max), (pairs_dev, pairs_e2e) = aggregate_over_ranks(times, pairs)

    if rank == 0:
        value = pairs_dev / t_dev_max
        if args.solver == "jacobi" and all_conv and iters_total % args.steps == 0:
            record_iters(args.workload, iters_total // args.steps)
        # roofline of the dominant kernel (pass 2), timed live with CUDA events on the context's stream
        pair_s = prof["pair_ms"] * 1e-3 / max(prof["pair_launches"], 1)
        achieved = FLOPS_PER_PAIR * N * (N - 1) / pair_s / 1e12
        peak_meas = g.fp64_peak(5) / 1e12
        peak_dmma = g.fp64_peak_dmma(5) / 1e12
        traffic = ncu_traffic(args.workload, "sym" if "pair=sym" in g.last_kernels() else "onesided")
        same_pairs = float((wl.counts().astype(float) ** 2).sum())
        ent_s = prof["entropy_ms"] * 1e-3 / max(prof["entropy_launches"], 1)
        ent_flop = 2.0 * wl.n_q ** 3 + 25.0               # n_q^3 FMAs + 1 exponential per same-species pair
        # what the kernel EXECUTES, beside the algorithmic rate: FP64 instructions per ordered pair in the inner loop
        # (15 in the symmetric action-reaction form, where one evaluation serves both markers of a pair;
        # 26 in the one-sided form), each at most one FMA = 2 flop, against the issue rate of the FP64 pipe
        instr_pp = 15.0 if "pair=sym" in g.last_kernels() else 26.0
        pairs_ps = N * (N - 1) / pair_s
        lanes_ps = FP64_PEAK_NOMINAL / 2.0                     # FP64 instructions (lanes) per second, nominal
        executed = {"fp64_instr_per_ordered_pair": instr_pp, "flop_per_ordered_pair_at_most": 2.0 * instr_pp,
                    "tflops_at_most": 2.0 * instr_pp * pairs_ps / 1e12,
                    "fp64_pipe_issue_frac_of_nominal": instr_pp * pairs_ps / lanes_ps,
                    "fp64_pipe_issue_frac_of_measured_dfma": instr_pp * pairs_ps / (peak_meas * 1e12 / 2.0),
                    "note": "inner-loop instructions only; ncu's sm__inst_executed_pipe_fp64 (profiles/) is the "
                            "measured pipe utilisation and includes the loop's other FP64 work"}
        roofline = {"bound": "alu", "kernel": g.last_kernels(), "achieved": achieved, "peak": FP64_PEAK_NOMINAL / 1e12,
                    "achieved_is": "ALGORITHMIC rate = SURVEY.md section 8(d)'s 33 flop per ordered pair of the one-sided "
                                   "form x pairs / kernel time (a one-sided-equivalent rate, not pipe utilisation: a "
                                   "kernel that uses the pair symmetry can exceed 1.0 of peak on it); see `executed`",
                    "executed": executed,
                    "unit": "TFLOP/s", "frac": achieved / (FP64_PEAK_NOMINAL / 1e12),
                    "traffic": traffic["bytes"] if traffic else None,
                    "traffic_source": traffic["source"] if traffic else None,
                    "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum)",
                    "algorithmic_bytes": 56.0 * N + 24.0 * N,
                    "peak_source": "nominal FP64 FMA rate 148 SM x 64 lanes x 2 x 1.965 GHz (DESIGN.md); "
                                   "MEASURED_PEAKS.json has no FP64 figure",
                    "peak_measured_dfma": peak_meas, "frac_of_measured_dfma": achieved / peak_meas,
                    "flops_per_pair": FLOPS_PER_PAIR, "pairs_per_launch": float(N) * (N - 1),
                    "avg_launch_ms": pair_s * 1e3, "launches_timed": prof["pair_launches"],
                    "pair_kernel_pairs_per_s": N * (N - 1) / pair_s,
                    "pair_share_of_step": prof["pair_ms"] * 1e-3 / t_prof,
                    "kernel_times_from": "the timed region" if prof_in_timed else
                                         "2 extra profiled steps (the timed region replays CUDA-graph steps)",
                    "entropy_kernel_ms": prof["entropy_ms"] / max(prof["entropy_launches"], 1),
                    "entropy_same_species_pairs_per_s": float((wl.counts().astype(float) ** 2).sum()) /
                                                        (prof["entropy_ms"] * 1e-3 / max(prof["entropy_launches"], 1)),
                    "entropy_share_of_step": prof["entropy_ms"] * 1e-3 / t_prof,
                    "pass1": {"bound": "alu (FP64 pipe: DMMA + the exponentials)", "flops_per_same_species_pair": ent_flop,
                              "achieved": ent_flop * same_pairs / ent_s / 1e12, "unit": "TFLOP/s",
                              "peak_measured_dmma": peak_dmma, "frac_of_measured_dmma": ent_flop * same_pairs / ent_s / 1e12 / peak_dmma,
                              "frac_of_nominal": ent_flop * same_pairs / ent_s / FP64_PEAK_NOMINAL,
                              "dmma_only_frac_of_measured_dmma": 2.0 * wl.n_q ** 3 * same_pairs / ent_s / 1e12 / peak_dmma,
                              "note": "`achieved` counts 25 flop for the exponential, which runs on the FP64 VECTOR "
                                      "lanes of the same pipe, against a DMMA-only peak: an algorithmic rate; "
                                      "dmma_only_frac_of_measured_dmma counts the contraction alone"}}
        h2d = int(v_h.numel() * 8 + w_h.numel() * 8 + s_h.numel() * 4)
        d2h = int(out_h.numel() * 8 + 4 * 8 * wl.n_species)
        K0 = float(m0["K"].sum()); K1 = float(m1["K"].sum())
        wm_abs = float((wl.w * wl.mass[wl.species_id] * np.abs(wl.v).sum(axis=1)).sum())
        dP = float(np.abs(m1["P"].sum(axis=0) - m0["P"].sum(axis=0)).max()) / wm_abs
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 1), "ms_per_step": 1e3 * t_dev_max / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": config_dict(args, wl, iters_total / args.steps),
                "steps_per_s": args.steps * world / t_dev_max, "all_converged": bool(all_conv),
                "energy_drift_rel": abs(K1 - K0) / K0, "momentum_drift_rel": dP,
                "e2e": {"value": pairs_e2e / t_e2e_max, "unit": UNIT, "h2d_bytes_per_step": h2d,
                        "d2h_bytes_per_step": d2h, "ms_per_step": 1e3 * t_e2e_max / args.steps},
                "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline}
        # HBM-streaming rows (a0 pack, a6 moments): whole API calls (several small launches + one synchronisation),
        # so these are latency figures at this size, quoted against the measured copy bandwidth
        try:
            hbm_gbs = json.loads((ROOT / "MEASURED_PEAKS.json").read_text())["hbm_gbs"]
            hbm_src = "MEASURED_PEAKS.json"
        except Exception:
            hbm_gbs, hbm_src = 6650.0, "fallback of B200_PROFILING.md"
        reps = 10
        e0.record()
        for _ in range(reps):
            g.set_markers(v_d, w_d, s_d)
        e1.record(); torch.cuda.synchronize()
        t_pack = e0.elapsed_time(e1) * 1e-3 / reps
        e0.record()
        for _ in range(reps):
            g.moments(with_entropy=False)
        e1.record(); torch.cuda.synchronize()
        t_mom = e0.elapsed_time(e1) * 1e-3 / reps
        line["streaming"] = {"hbm_gbs_peak": hbm_gbs, "peak_source": hbm_src,
                             "pack": {"ms": 1e3 * t_pack, "algorithmic_bytes": 72.0 * N, "GBps": 72.0 * N / t_pack / 1e9,
                                      "frac": 72.0 * N / t_pack / 1e9 / hbm_gbs},
                             "moments": {"ms": 1e3 * t_mom, "algorithmic_bytes": 32.0 * N, "GBps": 32.0 * N / t_mom / 1e9,
                                         "frac": 32.0 * N / t_mom / 1e9 / hbm_gbs},
                             "note": "whole API calls incl. launches and one host synchronisation; per-kernel times: profiles/"}
        if N >= 16384 and args.solver == "jacobi":
            # mixed-precision implicit step (landau_set_mixed_precision): FP32 pass 2 while the residual is above 1e-7,
            # FP64 for the iterations that finish the step; same fixed point, same stopping rule.  Reported beside
            # the headline, which stays pure FP64.
            v_ref = step_device()[3].clone()
            g.set_mixed_precision(1e-7)
            step_device()
            torch.cuda.synchronize()
            e0.record()
            it_mx, conv_mx = 0, True
            for _ in range(2):
                it, conv, m_mx, v_mx = step_device()
                it_mx += it; conv_mx &= bool(conv)
            e1.record(); torch.cuda.synchronize()
            t_mx = e0.elapsed_time(e1) * 1e-3 / 2
            g.set_mixed_precision(0.0)
            line["mixed_precision_step"] = {
                "f32_until_residual": 1e-7, "ms_per_step": 1e3 * t_mx, "steps_per_s": 1.0 / t_mx,
                "iterations_per_step": it_mx / 2, "all_converged": conv_mx, "kernels": "pair=sym_mixed",
                "state_rel_diff_vs_fp64_step": float(torch.linalg.norm(v_mx - v_ref) / torch.linalg.norm(v_ref)),
                "energy_drift_rel": abs(float(m_mx["K"].sum()) - K0) / K0,
                "speedup_vs_fp64_step": (t_dev_max / args.steps) / t_mx}
        if not args.no_dg:
            # one discrete-gradient step (Eqs. 46-49), device driven; every iteration costs two
            # pass-1 and one pass-2 evaluations.  Its fixed point (G re-evaluated every iteration) is solved with
            # Anderson mixing of depth 5: the plain Jacobi sweep stops contracting at >= 1e5 markers
            g.set_solver(1, 5)
            g.set_markers(v_d, w_d, s_d)
            dg_tol = 1e-10 if args.workload.startswith("c4") else wl.tol          # reading DG2 (round-off floor of lambda)
            rc_dg, it_dg, res_dg, conv_dg = g.step_dg(wl.dt, dg_tol, 100)         # sizes every buffer
            g.set_markers(v_d, w_d, s_d)
            torch.cuda.synchronize()
            e0.record()
            rc_dg, it_dg, res_dg, conv_dg = g.step_dg(wl.dt, dg_tol, 100)
            e1.record(); torch.cuda.synchronize()
            line["dg_step"] = {"ms_per_step": e0.elapsed_time(e1), "iterations": it_dg, "residual": res_dg,
                               "converged": bool(conv_dg), "tol": dg_tol, "pass1_evaluations": 1 + 2 * (it_dg - 1),
                               "pass2_evaluations": it_dg, "solver": "anderson depth 5"}
            g.set_solver(0)
            if args.solver == "anderson":
                g.set_solver(1, args.anderson_depth)
            if args.solver == "newton":
                g.set_solver(2, args.newton_restart)
        if args.solver == "jacobi":
            # SURVEY.md NEXT-4, reported beside the headline (which stays the paper's Jacobi iteration): the same
            # step with the Anderson-accelerated fixed point, device-resident inputs, after both timed regions
            g.set_solver(1, args.anderson_depth)
            step_device()
            torch.cuda.synchronize()
            e0.record()
            it_aa, conv_aa = 0, True
            for _ in range(2):
                it, conv, _m, _v = step_device()
                it_aa += it; conv_aa &= bool(conv)
            e1.record()
            torch.cuda.synchronize()
            t_aa = e0.elapsed_time(e1) * 1e-3 / 2
            line["anderson_solver"] = {"depth": args.anderson_depth, "ms_per_step": 1e3 * t_aa, "steps_per_s": 1.0 / t_aa,
                                       "iterations_per_step": it_aa / 2, "all_converged": conv_aa,
                                       "pairs_per_s": (it_aa / 2) * N * (N - 1) / t_aa}
            g.set_solver(0)
        if args.workload.startswith("c4"):
            # BASELINE config 4: "plus an FP32 field variant" -- pass 2 alone, FP32 arithmetic, vs the FP64 kernel
            G = g.entropy_grad(v_d, w_d, s_d)
            V64 = g.pair_field(v_d, w_d, s_d, G)
            g32 = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0, precision=1)
            V32 = g32.pair_field(v_d, w_d, s_d, G)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(3):
                g32.pair_field(v_d, w_d, s_d, G)
            e1.record()
            torch.cuda.synchronize()
            t32 = e0.elapsed_time(e1) * 1e-3 / 3
            sid_t = s_d.long()
            err = [float(torch.linalg.norm((V32 - V64)[sid_t == k]) / torch.linalg.norm(V64[sid_t == k]))
                   for k in range(wl.n_species)]
            line["fp32_field_variant"] = {"kernels": g32.last_kernels(), "pairs_per_s": N * (N - 1) / t32,
                                          "ms_per_eval": 1e3 * t32, "includes": "pack + pair kernel + combine",
                                          "rel_l2_vs_fp64_per_species": err}
            del g32
        if not args.no_cpu_baseline and world == 1:
            _, info, _ = oracle_sample(wl, max(1, round(iters_total / args.steps)), args.cpu_seconds, args.workload)
            line["cpu_baseline"] = info
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
