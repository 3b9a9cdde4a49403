"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (-m gpu).

The oracle cannot evaluate a whole field at >= 1e5 markers in test time (pass 1 alone is 8e11 exponentials at
3 x 2^16), but each OUTPUT ROW is a plain sum it computes one by one (`landau_ref_*_rows`): pass 1 and pass 2 are
compared on sampled rows, the implicit step by re-evaluating Eq. (24) with oracle rows at the
midpoint the CUDA path returned, and the conservation laws (Eqs. 27, 29) hold at any size.
These tests replace the uncommitted parity report BASELINE.md section 3 used to cite; they print the measured
errors (run with -s to see them; profiles/r2_parity.md keeps the round-2 run, profiles/r3_parity.md this round's).
"""
import json
import os
from pathlib import Path

import numpy as np
import pytest

from paper_2212_00663_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_FIELD = 1e-10     # north_star: relative L2 over markers, overall and per species
TOL_DRIFT = 1e-12     # north_star: per-step relative drift of momentum and energy
REPORT = {}


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; the CUDA path has no fallback")
    from paper_2212_00663_b200 import binding
    binding.load()
    return binding


@pytest.fixture(scope="module", autouse=True)
def write_report():
    yield
    out = Path(os.environ.get("GRAFT_REPO_ROOT", Path(__file__).resolve().parent.parent)) / "gpurun_out"
    try:
        out.mkdir(exist_ok=True)
        (out / "config_size_parity.json").write_text(json.dumps(REPORT, indent=1))
    except OSError:
        pass


def rel_l2(a, b):
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def sample_rows(wl, per_species, seed):
    rng = np.random.default_rng(seed)
    return np.sort(np.concatenate([rng.choice(np.flatnonzero(wl.species_id == s), per_species, replace=False)
                                   for s in range(wl.n_species)])).astype(np.int64)


def per_species_errors(got, ref, sid, S):
    e = {"all": rel_l2(got, ref)}
    for s in range(S):
        m = sid == s
        e[f"s{s}"] = rel_l2(got[m], ref[m])
    return e


@pytest.mark.parametrize("cfg,nps", [(4, 1 << 16), (4, 1 << 17), (3, 32768), (2, 8192), (1, 4096)])
def test_pair_field_config_size_sampled_rows(B, oracle_mod, cfg, nps):
    """Pass 2 with the AUTOMATIC kernel choice (the symmetric action-reaction kernel at these sizes) at the bench
    workload 3 x 2^16, the largest single-GPU config 3 x 2^17 and configs 1-3 at full size: sampled target rows
    against the oracle's literal Eq. (23) (each row a sum over all N - 1 sources), plus Eqs. 27 and 29."""
    wl = W.make(cfg, n_per_species=nps, shuffled=True)
    g = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    o = oracle_mod.LandauRef(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    rng = np.random.default_rng(31 + cfg)
    G = rng.standard_normal((wl.n_markers, 3)) * np.sqrt(wl.mass[wl.species_id])[:, None]
    got = g.pair_field(wl.v, wl.w, wl.species_id, G).cpu().numpy()
    if wl.n_markers >= 16384:
        assert "pair=sym" in g.last_kernels()
    rows = sample_rows(wl, 64, 41 + cfg)
    ref = o.pair_field_rows(wl.v, wl.w, wl.species_id, G, rows)
    err = per_species_errors(got[rows], ref, wl.species_id[rows], wl.n_species)
    REPORT[f"pair_field c{cfg} {wl.n_species}x{nps}"] = dict(err, rows=len(rows), kernels=g.last_kernels())
    print(f"pass 2 c{cfg} {wl.n_species} x {nps}: {err} [{g.last_kernels()}]")
    assert np.all(np.isfinite(got)) and max(err.values()) <= TOL_FIELD, err
    wm = (wl.w * wl.mass[wl.species_id])[:, None]
    assert np.abs((wm * got).sum(axis=0)).max() <= 1e-13 * np.abs(wm * got).sum()          # Eq. 27
    assert abs((wm * wl.v * got).sum()) <= 1e-13 * np.abs(wm * wl.v * got).sum()             # Eq. 29


@pytest.mark.parametrize("cfg,nps", [(4, 1 << 17), (3, 32768), (2, 8192)])
def test_entropy_grad_config_size_sampled_rows(B, oracle_mod, cfg, nps):
    """Pass 1 (automatic kernel) at the sizes test_gpu_parity.py does not reach: sampled rows vs literal Eq. (22)."""
    wl = W.make(cfg, n_per_species=nps, shuffled=True)
    g = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    o = oracle_mod.LandauRef(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    G = g.entropy_grad(wl.v, wl.w, wl.species_id).cpu().numpy()
    rows = sample_rows(wl, 12 if nps > 40000 else 24, 51 + cfg)
    ref = o.entropy_grad_rows(wl.v, wl.w, wl.species_id, rows)
    err = per_species_errors(G[rows], ref, wl.species_id[rows], wl.n_species)
    REPORT[f"entropy_grad c{cfg} {wl.n_species}x{nps}"] = dict(err, rows=len(rows), kernels=g.last_kernels())
    print(f"pass 1 c{cfg} {wl.n_species} x {nps}: {err} [{g.last_kernels()}]")
    assert np.all(np.isfinite(G)) and max(err.values()) <= TOL_FIELD, err


def test_both_passes_at_one_million_markers_sampled_rows(B, oracle_mod):
    """Beyond BASELINE's largest config (393 216 markers): 3 x 349 525 = 1 048 575 markers, species sizes that are not
    multiples of any tile (ragged tails everywhere), 64-bit offsets in every partial-sum array.  Pass 2 (1.1e12 ordered
    pairs) and pass 1 (3.7e11 same-species pairs) against the oracle's literal Eqs. (23), (22) on sampled rows, plus
    Eqs. 27 and 29, which hold at any size."""
    nps = 349525
    wl = W.make(4, n_per_species=nps, shuffled=True)
    g = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    o = oracle_mod.LandauRef(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    rng = np.random.default_rng(77)
    G = rng.standard_normal((wl.n_markers, 3)) * np.sqrt(wl.mass[wl.species_id])[:, None]
    got = g.pair_field(wl.v, wl.w, wl.species_id, G).cpu().numpy()
    assert "pair=sym" in g.last_kernels()
    rows = sample_rows(wl, 12, 78)
    err = per_species_errors(got[rows], o.pair_field_rows(wl.v, wl.w, wl.species_id, G, rows), wl.species_id[rows],
                             wl.n_species)
    REPORT[f"pair_field c4 3x{nps}"] = dict(err, rows=len(rows), kernels=g.last_kernels())
    print(f"pass 2 c4 3 x {nps}: {err}")
    assert np.all(np.isfinite(got)) and max(err.values()) <= TOL_FIELD, err
    wm = (wl.w * wl.mass[wl.species_id])[:, None]
    assert np.abs((wm * got).sum(axis=0)).max() <= 1e-13 * np.abs(wm * got).sum()          # Eq. 27
    assert abs((wm * wl.v * got).sum()) <= 1e-13 * np.abs(wm * wl.v * got).sum()             # Eq. 29
    Gg = g.entropy_grad(wl.v, wl.w, wl.species_id).cpu().numpy()
    assert "entropy=mma" in g.last_kernels()
    rows = sample_rows(wl, 4, 79)
    errG = per_species_errors(Gg[rows], o.entropy_grad_rows(wl.v, wl.w, wl.species_id, rows), wl.species_id[rows],
                              wl.n_species)
    REPORT[f"entropy_grad c4 3x{nps}"] = dict(errG, rows=len(rows), kernels=g.last_kernels())
    print(f"pass 1 c4 3 x {nps}: {errG}")
    assert np.all(np.isfinite(Gg)) and max(errG.values()) <= TOL_FIELD, errG


@pytest.mark.parametrize("seed", range(16))
def test_fuzz_mid_size_clouds_sampled_rows(B, oracle_mod, seed):
    """Randomised clouds of 1e3 .. 5e4 markers: 1-4 species with random masses, charges, temperatures, drifts and ragged
    counts (no count a multiple of any tile), n_q 2..8 (one to eight node groups of the DMMA contraction), 3-V and
    native 2-V, whatever pair kernel the size selects.  Pass 1 and the whole field on sampled rows against the oracle's
    literal Eqs. (22), (23)."""
    rng = np.random.default_rng(9000 + seed)
    S = int(rng.integers(1, 5))
    mass = np.exp(rng.uniform(0.0, 9.0, S)); mass[0] = 1.0
    charge = rng.choice([-1.0, 1.0, 2.0], S)
    counts = rng.integers(1, 9000, S)
    if seed % 5 == 0:
        counts[0] = int(rng.integers(16000, 40000))
    T = rng.uniform(0.3, 2.0, S)
    vs, ws, ss = [], [], []
    for s in range(S):
        vs.append(rng.standard_normal((counts[s], 3)) * np.sqrt(T[s] / mass[s])
                  + rng.normal(0, 0.3, 3) * np.sqrt(T[s] / mass[s]))
        ws.append((0.2 + rng.random(counts[s])) / counts[s])
        ss.append(np.full(counts[s], s, dtype=np.int32))
    v, w, sid = np.concatenate(vs), np.concatenate(ws), np.concatenate(ss)
    perm = rng.permutation(len(w))
    v, w, sid = v[perm], w[perm], sid[perm]
    eps = rng.uniform(0.03, 0.2, S) * T / mass
    n_q = int(rng.integers(2, 9))
    two_v = seed % 7 == 3
    if two_v:
        v[:, 2] = 0.0
    g = B.Landau(mass, charge, eps, n_q=n_q)
    o = oracle_mod.LandauRef(mass, charge, eps, n_q=n_q)
    if two_v:
        g.set_dimension(2)
    G = g.entropy_grad(v, w, sid).cpu().numpy()
    rows = np.sort(rng.choice(len(w), min(24, len(w)), replace=False)).astype(np.int64)
    eG = rel_l2(G[rows], o.entropy_grad_rows(v, w, sid, rows))
    V = g.eval_field(v, w, sid).cpu().numpy()
    eV = rel_l2(V[rows], o.pair_field_rows(v, w, sid, G, rows))
    print(f"fuzz {seed}: S={S} N={len(w)} n_q={n_q} {'2-V' if two_v else '3-V'} [{g.last_kernels()}] G {eG:.1e} V {eV:.1e}")
    assert np.all(np.isfinite(V)) and eG <= TOL_FIELD and eV <= 10 * TOL_FIELD, (seed, eG, eV)
    if two_v:
        assert np.all(G[:, 2] == 0.0) and np.all(V[:, 2] == 0.0)


STEP_MODES = {
    # name: (setter calls on the binding object, substring expected in last_kernels())
    "jacobi": ([], "pair=sym"),
    "mixed_1e-7": ([("set_mixed_precision", (1e-7,))], "pair=sym_mixed"),
    "anderson_3": ([("set_solver", (1, 3))], "pair=sym"),
    "newton_20": ([("set_solver", (2, 20))], "pair=sym"),
    "jacobi_stiff_0.2": ([("set_stiff_pairs", (0.2,))], "pair=sym"),
    # config 4 at the survey's dt = 0.01 (reading U4), where the paper's Jacobi map no longer contracts
    "anderson_10_dt0.01": ([("set_solver", (1, 10))], "pair=sym"),
}
STEP_DT = {"anderson_10_dt0.01": 0.01}


@pytest.mark.parametrize("cfg,nps,mode", [(4, 1 << 16, "jacobi"), (3, 32768, "jacobi"),
                                          (4, 1 << 14, "mixed_1e-7"), (4, 1 << 16, "mixed_1e-7"),
                                          (4, 1 << 16, "anderson_3"), (4, 1 << 16, "newton_20"),
                                          (4, 1 << 16, "jacobi_stiff_0.2"), (4, 1 << 16, "anderson_10_dt0.01")])
def test_converged_step_config_size_satisfies_eq24_on_oracle_rows(B, oracle_mod, cfg, nps, mode):
    """One converged landau_step at the bench workload (3 x 2^16 markers, symmetric kernel, the launch sequence
    bench.py times) and at config 3's full size, checked WITHOUT a full oracle step (which would take hours):

      1. G^n of the CUDA path equals the oracle's literal Eq. (22) on sampled rows (<= 1e-10);
      2. the returned v^{n+1} solves Eq. (24): on sampled rows  v1 - v0 - dt V_oracle[(v0 + v1)/2 ; G^n]  with
         V_oracle = the oracle's literal Eq. (23) row sums at the returned midpoint.  The last Jacobi iterate
         differs from the fixed point by <= rho tol |v1| (rho < 1 the contraction factor), so the defect is
         bounded by tol = 1e-12 relative to the state in the residual's own energy norm; relative to the
         displacement |v1 - v0| ~ dt |V| (1e-3 of the state here) that is <= 1e-8;
      3. Eqs. (26)-(29): momentum and energy drift of the step <= 1e-12 (north_star).

    `mode` runs the same check, with the same bounds, on every stepping mode that solves Eq. (24): the paper's Jacobi
    loop, the mixed-precision loop (FP32 pass 2 while the residual exceeds 1e-7, FP64 after), Anderson mixing,
    Jacobian-free Newton-Krylov, and Jacobi with the exact stiff-pair treatment -- all have the same fixed point."""
    wl = W.make(cfg, n_per_species=nps, shuffled=True)
    g = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    for name, args in STEP_MODES[mode][0]:
        getattr(g, name)(*args)
    dt = STEP_DT.get(mode, wl.dt)
    o = oracle_mod.LandauRef(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    G = g.entropy_grad(wl.v, wl.w, wl.species_id).cpu().numpy()
    rowsG = sample_rows(wl, 8, 61 + cfg)
    errG = per_species_errors(G[rowsG], o.entropy_grad_rows(wl.v, wl.w, wl.species_id, rowsG), wl.species_id[rowsG],
                              wl.n_species)
    assert max(errG.values()) <= TOL_FIELD, errG
    g.set_markers(wl.v, wl.w, wl.species_id)
    m0 = g.moments(with_entropy=False)
    rc, it, res, conv = g.step(dt, wl.tol, wl.max_iter)
    assert rc == 0 and conv and res <= wl.tol, (rc, it, res)
    assert STEP_MODES[mode][1] in g.last_kernels(), g.last_kernels()
    v1 = g.get_markers().cpu().numpy()
    m1 = g.moments(with_entropy=False)
    rows = sample_rows(wl, 48, 71 + cfg)
    u = 0.5 * (wl.v + v1)
    Vo = o.pair_field_rows(u, wl.w, wl.species_id, G, rows)
    defect = v1[rows] - wl.v[rows] - dt * Vo
    disp = v1[rows] - wl.v[rows]
    wm = (wl.w * wl.mass[wl.species_id])[rows][:, None]
    rel_state = float(np.sqrt((wm * defect ** 2).sum() / (wm * v1[rows] ** 2).sum()))
    sid = wl.species_id[rows]
    rel_disp = {f"s{s}": float(np.linalg.norm(defect[sid == s]) / np.linalg.norm(disp[sid == s]))
                for s in range(wl.n_species)}
    wm_abs = float((wl.w * wl.mass[wl.species_id] * np.abs(wl.v).sum(axis=1)).sum())
    dP = float(np.abs(m1["P"].sum(axis=0) - m0["P"].sum(axis=0)).max()) / wm_abs
    dK = abs(float(m1["K"].sum() - m0["K"].sum())) / float(m0["K"].sum())
    REPORT[f"step c{cfg} {wl.n_species}x{nps} {mode}"] = dict(iterations=it, residual=res, G_rows=errG, eq24_defect_rel_state=rel_state,
                                                      eq24_defect_rel_displacement=rel_disp, momentum_drift=dP,
                                                      energy_drift=dK, kernels=g.last_kernels())
    print(f"step c{cfg} {wl.n_species} x {nps} [{mode}]: {it} iterations, residual {res:.2e}; Eq. (24) defect / state {rel_state:.2e}, "
          f"/ displacement {rel_disp}; dP {dP:.1e}, dK/K {dK:.1e}")
    assert rel_state <= 1e-12
    assert max(rel_disp.values()) <= 1e-8, rel_disp
    assert dP <= TOL_DRIFT and dK <= TOL_DRIFT


@pytest.mark.parametrize("variant", ["2v", "detect"])
def test_symmetric_kernel_generic_loop_config_size_vs_oracle_rows(B, oracle_mod, variant):
    """pair_sym_kernel's DIM = 2 and DETECT = true instantiations run the generic inner loop (`sym_step`), not the
    hand-specialised 3-V text (`sym_step3`) the headline runs: both at 3 x 2^16 markers against the oracle's literal
    Eq. (23) rows.
      2v:     landau_set_dimension(2) on v_z = 0 data (the paper's 2-V setting), supplied gradient;
      detect: the first evaluation of a step with the stiff-pair treatment on (it also looks for stiff pairs); theta is
              set so high that none is found, so v^(1) - v0 = dt V[v0 ; G^n] exactly as in the plain step."""
    wl = W.make(4, n_per_species=1 << 16, shuffled=True)
    o = oracle_mod.LandauRef(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    g = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    rows = sample_rows(wl, 32, 101)
    if variant == "2v":
        v = wl.v.copy(); v[:, 2] = 0.0
        rng = np.random.default_rng(5)
        G = rng.standard_normal((wl.n_markers, 3)) * np.sqrt(wl.mass[wl.species_id])[:, None]
        G[:, 2] = 0.0
        g.set_dimension(2)
        V = g.pair_field(v, wl.w, wl.species_id, G).cpu().numpy()
        assert "pair=sym2v" in g.last_kernels(), g.last_kernels()
        assert np.all(V[:, 2] == 0.0)
        err = per_species_errors(V[rows], o.pair_field_rows(v, wl.w, wl.species_id, G, rows), wl.species_id[rows], 3)
        bound = TOL_FIELD
    else:
        G = g.entropy_grad(wl.v, wl.w, wl.species_id).cpu().numpy()
        g.set_stiff_pairs(1e9)
        g.set_markers(wl.v, wl.w, wl.species_id)
        rc, it, res, conv = g.step(wl.dt, 0.0, 1)
        assert (rc, it, conv) == (1, 1, False) and "pair=sym" in g.last_kernels()
        assert g.stiff_pairs_last() == (0, 0)
        v1 = g.get_markers().cpu().numpy()
        err = per_species_errors(v1[rows] - wl.v[rows], wl.dt * o.pair_field_rows(wl.v, wl.w, wl.species_id, G, rows),
                                 wl.species_id[rows], 3)
        bound = 1e-9          # a displacement: dt V is added to O(1) velocities, so ~1e-16 / 1e-3 relative is lost
    REPORT[f"generic sym loop {variant} 3x65536"] = err
    print(f"symmetric kernel, generic loop [{variant}] at 3 x 2^16 vs oracle rows: {err} (bound {bound:g})")
    assert max(err.values()) <= bound, err


@pytest.mark.parametrize("solver", ["jacobi", "anderson_5"])
def test_dg_step_sym_kernel_size_satisfies_eq46_with_oracle_terms(B, oracle_mod, solver):
    """landau_step_dg (Eqs. 46-49; Gonzalez' discrete gradient, reading DG1) at 3 x 5462 = 16 386
    markers -- the symmetric pair kernel's regime, 6x the largest full-oracle DG comparison -- with the plain sweep and
    with Anderson depth 5 as on the bench line.  A full oracle DG step costs (2 pass 1 + 1 pass 2) per iteration, minutes here, so the
    converged step is checked by re-evaluating Eq. (46) with ORACLE terms only: G(u) at the returned midpoint (every
    marker, literal Eq. 22), S_eps(v0) and S_eps(v1) (Eq. 20), and the oracle's Eq. (23) rows.  Three oracle pass-1
    evaluations, ~5 s each on the GPU box's cores.

    From them lambda = [S(v1) - S(v0) - sum w G(u).dv] / sum |dv|^2 and Gbar_p = G_p(u) + lambda dv_p / w_p, and the
    defect of Eq. (46) on sampled rows is  dv - dt V_oracle[u; Gbar]: the fixed-point map's own residual at the
    returned state, in the residual's energy norm relative to the STATE over the sampled rows, with tol = 3e-12 (the
    level both implementations can still reach, reading DG2).
      anderson_5: bound 1e-11; observed 4.8e-13, below its last residual (6.2e-13).
      jacobi:     bound 3e-11; observed 1.07e-11 = 4.6x its last residual (2.3e-12).  The excess lies entirely along
                  the lambda direction: with the scalar that fits the returned step best (6e-8 relative from the
                  oracle's lambda) the defect is 1e-9 of the displacement.  The plain sweep converges slowly in lambda
                  and the difference of successive iterates under-reports it (reading DG3; DESIGN.md open items) -- a
                  property of the iteration, which the oracle's O4b shares, not of a kernel: the CUDA path's entropies
                  match the oracle's to 3e-16 here and S1 - S0 to 2e-15 (printed).
    Relative to each species' displacement the same defect is tol |v| / |dv| (the light species moves by 7e-4 of its
    speed, the heavy ones by 7e-6): bounded by 1e-6, printed.  Momentum and energy drift <= 1e-12 (Eqs. 26-29 hold for
    any lambda); the CUDA path's S_eps at v0 and v1 equal the oracle's to 1e-13; and the ORACLE's entropy of the
    returned state is not below the initial one (Eq. 49)."""
    wl = W.make(4, n_per_species=5462, shuffled=True)
    g = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    o = oracle_mod.LandauRef(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    if solver == "anderson_5":
        g.set_solver(1, 5)
    g.set_markers(wl.v, wl.w, wl.species_id)
    m0 = g.moments(with_entropy=True)
    rc, it, res, conv = g.step_dg(wl.dt, 3e-12, 100)
    assert rc == 0 and conv, (rc, it, res)
    assert "pair=sym" in g.last_kernels(), g.last_kernels()
    v1 = g.get_markers().cpu().numpy()
    m1 = g.moments(with_entropy=True)
    dv = v1 - wl.v
    u = 0.5 * (wl.v + v1)
    Gu, _ = o.entropy_grad(u, wl.w, wl.species_id, with_entropy=True)
    _, S0 = o.entropy_grad(wl.v, wl.w, wl.species_id, with_entropy=True)
    _, S1 = o.entropy_grad(v1, wl.w, wl.species_id, with_entropy=True)
    dv2 = float((dv ** 2).sum())
    remainder = float(S1.sum() - S0.sum()) - float((wl.w[:, None] * Gu * dv).sum())
    lam = remainder / dv2
    rows = sample_rows(wl, 48, 111)
    VG = o.pair_field_rows(u, wl.w, wl.species_id, Gu, rows)
    VD = o.pair_field_rows(u, wl.w, wl.species_id, dv / wl.w[:, None], rows)
    defect = dv[rows] - wl.dt * (VG + lam * VD)
    # diagnostics: the scalar that fits the returned step best, and the CUDA path's own entropies
    lam_fit = float(((dv[rows] - wl.dt * VG) * VD).sum() / (wl.dt * (VD * VD).sum()))
    defect_fit = dv[rows] - wl.dt * (VG + lam_fit * VD)
    eS0 = float(np.abs(m0["S_eps"] - S0).max() / np.abs(S0).max())
    eS1 = float(np.abs(m1["S_eps"] - S1).max() / np.abs(S1).max())
    e_dS = (float(m1["S_eps"].sum() - m0["S_eps"].sum()) - float(S1.sum() - S0.sum()))
    print(f"  lambda fit {lam_fit:.8e} vs oracle {lam:.8e} (rel {abs(lam_fit / lam - 1):.1e}); defect/disp with the fit "
          f"{ {s: float(np.linalg.norm(defect_fit[wl.species_id[rows] == s]) / np.linalg.norm(dv[rows][wl.species_id[rows] == s])) for s in range(3)} }; "
          f"S_eps CUDA vs oracle rel {eS0:.1e} / {eS1:.1e}; (S1 - S0) CUDA - oracle = {e_dS:.2e}; remainder {remainder:.3e}; sum dv^2 {dv2:.3e}")
    sid = wl.species_id[rows]
    wm = (wl.w * wl.mass[wl.species_id])[rows][:, None]
    rel_state = float(np.sqrt((wm * defect ** 2).sum() / (wm * v1[rows] ** 2).sum()))
    rel_state_s = {f"s{s}": float(np.linalg.norm(defect[sid == s]) / np.linalg.norm(v1[rows][sid == s]))
                   for s in range(wl.n_species)}
    rel_disp = {f"s{s}": float(np.linalg.norm(defect[sid == s]) / np.linalg.norm(dv[rows][sid == s]))
                for s in range(wl.n_species)}
    wm_abs = float((wl.w * wl.mass[wl.species_id] * np.abs(wl.v).sum(axis=1)).sum())
    dP = float(np.abs(m1["P"].sum(axis=0) - m0["P"].sum(axis=0)).max()) / wm_abs
    dK = abs(float(m1["K"].sum() - m0["K"].sum())) / float(m0["K"].sum())
    dS = float(S1.sum() - S0.sum())
    REPORT[f"dg step c4 3x5462 {solver}"] = dict(iterations=it, residual=res, eq46_defect_rel_state=rel_state,
                                                 eq46_defect_rel_state_per_species=rel_state_s,
                                                 eq46_defect_rel_displacement=rel_disp, lambda_oracle=lam, lambda_fit=lam_fit,
                                                 S_eps_rel_error=[eS0, eS1], dS_error=e_dS,
                                                 entropy_remainder=remainder, sum_dv2=dv2, momentum_drift=dP,
                                                 energy_drift=dK, oracle_entropy_change=dS, kernels=g.last_kernels())
    print(f"DG step 3 x 5462 [{solver}]: {it} iterations, residual {res:.2e}; Eq. (46) defect / state {rel_state:.2e} "
          f"(bound 1e-11 Anderson, 3e-11 Jacobi), per species {rel_state_s}, / displacement {rel_disp} (bound 1e-6); lambda {lam:.4e}; "
          f"dP {dP:.1e}, dK/K {dK:.1e}; oracle S1 - S0 = {dS:.3e}")
    assert rel_state <= (1e-11 if solver == "anderson_5" else 3e-11)
    assert max(rel_disp.values()) <= 1e-6, rel_disp
    assert eS0 <= 1e-13 and eS1 <= 1e-13
    assert dP <= TOL_DRIFT and dK <= TOL_DRIFT
    assert dS >= 0.0


def test_mixed_precision_gate_edges(B, oracle_mod):
    """landau_set_mixed_precision's per-iteration gate (StepCtrl::use_f32) at its two ends, 3 x 2^14 markers:

      * a switch-over residual the FP32 iterates can never reach (1e-10, the smallest accepted): every evaluation is
        FP32 except the LAST one max_iter allows, which is FP64 -- so the step ends unconverged at max_iter, but the
        committed iterate v^(K) = v0 + dt V_64[(v0 + v^(K-1))/2] is an FP64 evaluation.  v^(K-1) is rebuilt by hand
        from K-1 evaluations of the FP32 field variant (the same kernel, precision = 1); the last evaluation is then
        compared with the ORACLE's Eq. (23) rows at that midpoint to 1e-8 of the displacement -- an FP32 last
        evaluation would miss by ~3e-6, the FP32 variant's stated error;
      * a switch-over residual above every residual (1e3): only the first evaluation is FP32, and the converged state
        meets the FP64 step's to the tolerance of the stopping rule;
      * thresholds in (0, 1e-10) are refused (they would keep every step in FP32 up to max_iter)."""
    wl = W.make(4, n_per_species=1 << 14, shuffled=True)
    o = oracle_mod.LandauRef(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    K = 6
    g64 = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    G = g64.entropy_grad(wl.v, wl.w, wl.species_id).cpu().numpy()
    g32 = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0, precision=1)
    vk = wl.v.copy()
    for _ in range(K - 1):                                      # v^(1) .. v^(K-1): FP32 evaluations at the midpoint
        vk = wl.v + wl.dt * g32.pair_field(0.5 * (wl.v + vk), wl.w, wl.species_id, G).cpu().numpy()
    assert "pair=sym_f32" in g32.last_kernels()
    gm = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    with pytest.raises(B.LandauError):
        gm.set_mixed_precision(1e-12)
    gm.set_mixed_precision(1e-10)
    gm.set_markers(wl.v, wl.w, wl.species_id)
    rc, it, res, conv = gm.step(wl.dt, 1e-13, K)
    assert (rc, it, conv) == (1, K, False) and "pair=sym_mixed" in gm.last_kernels()
    assert res > 1e-10, "the FP32 iterates must not have reached the switch-over residual"
    vK = gm.get_markers().cpu().numpy()
    rows = sample_rows(wl, 32, 91)
    Vo = o.pair_field_rows(0.5 * (wl.v + vk), wl.w, wl.species_id, G, rows)
    err = per_species_errors(vK[rows] - wl.v[rows], wl.dt * Vo, wl.species_id[rows], wl.n_species)
    REPORT["mixed gate: all FP32 then FP64 last"] = dict(residual=res, last_displacement_vs_oracle_rows=err)
    print(f"mixed gate (1e-10, K = {K}): residual {res:.2e}; last (FP64) displacement vs oracle rows {err} (bound 1e-8)")
    assert max(err.values()) <= 1e-8, err
    # only the first evaluation in FP32
    gl = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    gl.set_mixed_precision(1e3)
    gl.set_markers(wl.v, wl.w, wl.species_id)
    rcl, itl, resl, convl = gl.step(wl.dt, wl.tol, wl.max_iter)
    g64.set_markers(wl.v, wl.w, wl.species_id)
    rc6, it6, res6, conv6 = g64.step(wl.dt, wl.tol, wl.max_iter)
    assert rcl == 0 and convl and rc6 == 0 and conv6
    a, b = gl.get_markers().cpu().numpy(), g64.get_markers().cpu().numpy()
    wm = (wl.w * wl.mass[wl.species_id])[:, None]
    d = float(np.sqrt((wm * (a - b) ** 2).sum() / (wm * b ** 2).sum()))
    REPORT["mixed gate: FP32 first only"] = dict(iterations=itl, iterations_fp64=it6, state_difference=d)
    print(f"mixed gate (1e3): {itl} iterations (FP64 loop {it6}); converged state differs by {d:.2e} (bound 5 tol)")
    assert d <= 5 * wl.tol


def test_one_fixed_point_iterate_config_size_vs_oracle_rows(B, oracle_mod):
    """A NON-converged step (max_iter = 2) at 3 x 2^16: the committed iterate v^(2) = v0 + dt V[(v0 + v^(1))/2],
    v^(1) = v0 + dt V[v0], is reproduced on sampled rows from oracle row sums alone (two nested evaluations of
    literal Eq. (23); the inner one needs every marker, so v^(1) is rebuilt from the CUDA path's field, itself
    compared with the oracle on the same rows)."""
    wl = W.make(4, n_per_species=1 << 16, shuffled=True)
    g = B.Landau(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    o = oracle_mod.LandauRef(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)
    G = g.entropy_grad(wl.v, wl.w, wl.species_id).cpu().numpy()
    rows = sample_rows(wl, 32, 81)
    V0 = g.pair_field(wl.v, wl.w, wl.species_id, G).cpu().numpy()
    V0o = o.pair_field_rows(wl.v, wl.w, wl.species_id, G, rows)
    assert max(per_species_errors(V0[rows], V0o, wl.species_id[rows], 3).values()) <= TOL_FIELD
    v_1 = wl.v + wl.dt * V0
    g.set_markers(wl.v, wl.w, wl.species_id)
    rc, it, res, conv = g.step(wl.dt, 0.0, 2)
    assert (rc, it, conv) == (1, 2, False)
    v2 = g.get_markers().cpu().numpy()
    V1o = o.pair_field_rows(0.5 * (wl.v + v_1), wl.w, wl.species_id, G, rows)
    err = per_species_errors(v2[rows] - wl.v[rows], wl.dt * V1o, wl.species_id[rows], 3)
    REPORT["iterate c4 3x65536"] = err
    print(f"second Jacobi iterate at 3 x 2^16 vs oracle rows: {err}")
    assert max(err.values()) <= 1e-9, err
