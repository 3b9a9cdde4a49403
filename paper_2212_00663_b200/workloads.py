"""Seeded synthetic marker workloads (BASELINE.json configs c0..c4).

This module is the ONE piece shared by the CPU oracle's tests and the CUDA path's tests /
bench: it only draws random numbers and shapes them into marker clouds.  It holds none of
the method's arithmetic (no mollifier, no quadrature, no projection tensor, no time step)
and imports neither `oracle/` nor the CUDA binding.

The paper measured on no public dataset: its own tests are grid-initialised 2-V Maxwellians
(Eqs. 34-35).  BASELINE.json's configs are 3-V stand-ins with the same
physical structure (two or three species, mass ratio 1836+, Maxwellian-type clouds whose
thermal speeds differ by sqrt(m_i/m_e) ~ 43).  Recipe (DESIGN.md
"Input recipe"):

    rng = numpy.random.default_rng(seed)          # seed = config index unless overridden
    for each species, in the listed order:
        z   = rng.standard_normal((N_s, 3))       # velocity variates
        ... = weight variates (uniform or normal)  # drawn right after the velocities
    weights rescaled so that sum_{p in s} w_p = n_s exactly (reading U3)
    eps_s = 0.05 * T_s / m_s  (reading U2; T_s = nominal, or sampled for non-Maxwellian clouds)
    marker order = species concatenated; `shuffled=True` applies one permutation drawn last
    from the same rng, to exercise species_id bucketing.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

M_E = 1.0
M_I = 1836.0
M_D = 3671.0
M_C = 22032.0


@dataclass
class Workload:
    """One synthetic marker cloud plus the run parameters BASELINE.json attaches to it."""

    name: str
    mass: np.ndarray          # [S]
    charge: np.ndarray        # [S]
    density: np.ndarray       # [S]  n_s = sum of weights of species s
    eps: np.ndarray           # [S]  mollifier covariance eps_s (velocity^2)
    v: np.ndarray             # [N,3] float64, row-major
    w: np.ndarray             # [N]   float64, > 0
    species_id: np.ndarray    # [N]   int32 in 0..S-1
    dt: float
    tol: float = 1e-12
    max_iter: int = 50
    n_steps: int = 1
    n_q: int = 4
    nu0: float = 1.0
    seed: int = 0
    notes: dict = field(default_factory=dict)

    @property
    def n_species(self) -> int:
        return int(self.mass.shape[0])

    @property
    def n_markers(self) -> int:
        return int(self.w.shape[0])

    def counts(self) -> np.ndarray:
        return np.bincount(self.species_id, minlength=self.n_species)


def _uniform_weights(rng: np.random.Generator, n: int) -> np.ndarray:
    """BASELINE config 0: w proportional to (1 + 0.5 u), u ~ U[0,1)."""
    return 1.0 + 0.5 * rng.random(n)


def _lognormal_weights(rng: np.random.Generator, n: int, sigma: float) -> np.ndarray:
    """BASELINE configs 2 and 4: lognormal weights, w proportional to exp(sigma * z_w)."""
    return np.exp(sigma * rng.standard_normal(n))


def _sampled_temperature(m: float, v: np.ndarray, w: np.ndarray) -> float:
    """Weighted sample variance times mass, averaged over the three axes (k_B = 1).

    Only used to size eps_s for clouds that are not Maxwellian by construction (reading U2).
    """
    n = w.sum()
    u = (w[:, None] * v).sum(axis=0) / n
    return float(m * (w[:, None] * (v - u) ** 2).sum() / (3.0 * n))


def _assemble(name, species, rng, shuffled, dt, n_steps, seed, eps_rule, **kw) -> Workload:
    """species: list of dicts with keys m, q, n, v, w_raw, T (nominal T or None -> sampled)."""
    mass = np.array([s["m"] for s in species], dtype=np.float64)
    charge = np.array([s["q"] for s in species], dtype=np.float64)
    density = np.array([s["n"] for s in species], dtype=np.float64)
    vs, ws, ids, eps, temps = [], [], [], [], []
    for k, s in enumerate(species):
        w = s["w_raw"]
        if w.shape[0] > 0:
            w = w * (s["n"] / w.sum())
            # one more pass: sum_{p in s} w_p = n_s to the last bit that matters
            w = w * (s["n"] / w.sum())
        T = s["T"] if (s["T"] is not None or w.shape[0] == 0) else _sampled_temperature(s["m"], s["v"], w)
        T = 1.0 if T is None else T
        temps.append(T)
        eps.append(eps_rule * T / s["m"])
        vs.append(np.ascontiguousarray(s["v"], dtype=np.float64))
        ws.append(w.astype(np.float64))
        ids.append(np.full(w.shape[0], k, dtype=np.int32))
    v = np.concatenate(vs, axis=0)
    w = np.concatenate(ws)
    sid = np.concatenate(ids)
    if shuffled:
        perm = rng.permutation(v.shape[0])
        v, w, sid = v[perm], w[perm], sid[perm]
    notes = {"T_for_eps": temps, "shuffled": bool(shuffled), "eps_rule": eps_rule}
    notes.update(kw.pop("notes", {}))
    return Workload(name=name, mass=mass, charge=charge, density=density,
                    eps=np.array(eps, dtype=np.float64),
                    v=np.ascontiguousarray(v), w=np.ascontiguousarray(w),
                    species_id=np.ascontiguousarray(sid), dt=dt, n_steps=n_steps,
                    seed=seed, notes=notes, **kw)


def config0(n_per_species: int = 256, seed: int = 0, shuffled: bool = False,
            eps_rule: float = 0.05) -> Workload:
    """c0: e (m=1,q=-1) + i (m=1836,q=+1), isotropic Maxwellians T_e=1, T_i=0.5, one step."""
    rng = np.random.default_rng(seed)
    sp = []
    for (m, q, T) in ((M_E, -1.0, 1.0), (M_I, +1.0, 0.5)):
        z = rng.standard_normal((n_per_species, 3))
        wr = _uniform_weights(rng, n_per_species)
        sp.append(dict(m=m, q=q, n=1.0, v=z * np.sqrt(T / m), w_raw=wr, T=T))
    return _assemble("c0_two_species_single_step", sp, rng, shuffled, dt=0.01, n_steps=1,
                     seed=seed, eps_rule=eps_rule, tol=1e-12, max_iter=50)


def config1(n_per_species: int = 4096, seed: int = 1, shuffled: bool = False,
            eps_rule: float = 0.05) -> Workload:
    """c1: e-i temperature relaxation, T_e=2, T_i=1, zero drift, 200 steps at dt=0.02."""
    rng = np.random.default_rng(seed)
    sp = []
    for (m, q, T) in ((M_E, -1.0, 2.0), (M_I, +1.0, 1.0)):
        z = rng.standard_normal((n_per_species, 3))
        wr = _uniform_weights(rng, n_per_species)
        sp.append(dict(m=m, q=q, n=1.0, v=z * np.sqrt(T / m), w_raw=wr, T=T))
    return _assemble("c1_ei_temperature_relaxation", sp, rng, shuffled, dt=0.02, n_steps=200,
                     seed=seed, eps_rule=eps_rule, tol=1e-12, max_iter=50)


def config2(n_per_species: int = 8192, seed: int = 2, shuffled: bool = False,
            eps_rule: float = 0.05) -> Workload:
    """c2: isotropisation; bi-Maxwellian electrons (T_par=2 along z, T_perp=1), ions T=1.5."""
    rng = np.random.default_rng(seed)
    sp = []
    z = rng.standard_normal((n_per_species, 3))
    wr = _lognormal_weights(rng, n_per_species, 0.5)
    ve = z * np.sqrt(np.array([1.0, 1.0, 2.0]) / M_E)
    sp.append(dict(m=M_E, q=-1.0, n=1.0, v=ve, w_raw=wr, T=None))
    z = rng.standard_normal((n_per_species, 3))
    wr = _lognormal_weights(rng, n_per_species, 0.5)
    sp.append(dict(m=M_I, q=+1.0, n=1.0, v=z * np.sqrt(1.5 / M_I), w_raw=wr, T=None))
    return _assemble("c2_isotropisation", sp, rng, shuffled, dt=0.01, n_steps=500,
                     seed=seed, eps_rule=eps_rule, tol=1e-12, max_iter=50)


def config3(n_per_species: int = 32768, seed: int = 3, shuffled: bool = False,
            eps_rule: float = 0.05) -> Workload:
    """c3: thermalisation; electrons on a shell |v|=1.5 (jitter 0.05), Maxwellian ions T=1."""
    rng = np.random.default_rng(seed)
    sp = []
    z = rng.standard_normal((n_per_species, 3))
    zr = rng.standard_normal(n_per_species)
    wr = _uniform_weights(rng, n_per_species)
    direction = z / np.linalg.norm(z, axis=1, keepdims=True)
    ve = direction * (1.5 + 0.05 * zr)[:, None]
    sp.append(dict(m=M_E, q=-1.0, n=1.0, v=ve, w_raw=wr, T=None))
    z = rng.standard_normal((n_per_species, 3))
    wr = _uniform_weights(rng, n_per_species)
    sp.append(dict(m=M_I, q=+1.0, n=1.0, v=z * np.sqrt(1.0 / M_I), w_raw=wr, T=None))
    return _assemble("c3_shell_thermalisation", sp, rng, shuffled, dt=0.01, n_steps=300,
                     seed=seed, eps_rule=eps_rule, tol=1e-12, max_iter=50)


def config4(n_per_species: int = 1 << 14, seed: int = 4, shuffled: bool = False,
            eps_rule: float = 0.05) -> Workload:
    """c4: scaling sweep; e, D+ (m=3671,q=+1,n=0.7), C6+ (m=22032,q=+6,n=0.05), T=1 each."""
    rng = np.random.default_rng(seed)
    sp = []
    for (m, q, n) in ((M_E, -1.0, 1.0), (M_D, +1.0, 0.7), (M_C, +6.0, 0.05)):
        z = rng.standard_normal((n_per_species, 3))
        wr = _lognormal_weights(rng, n_per_species, 1.0)
        sp.append(dict(m=m, q=q, n=n, v=z * np.sqrt(1.0 / m), w_raw=wr, T=1.0))
    # reading U4: BASELINE gives c4 no dt.  dt = 0.001: with the C6+ species (nu up to 36^2) and the
    # close pairs of 2^16-marker clouds the Jacobi fixed point of Eq. (24) does not contract at
    # dt = 0.01 (measured: no convergence in 60 iterations); at 0.001 it takes 9..16 iterations.
    return _assemble("c4_three_species_scaling", sp, rng, shuffled, dt=0.001, n_steps=1,
                     seed=seed, eps_rule=eps_rule, tol=1e-12, max_iter=50)


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}


def make(config: int, n_per_species: Optional[int] = None, seed: Optional[int] = None,
         shuffled: bool = False, eps_rule: float = 0.05) -> Workload:
    """Build BASELINE.json config `config` (0..4), optionally at a reduced marker count."""
    fn = CONFIGS[config]
    kw = dict(shuffled=shuffled, eps_rule=eps_rule)
    if n_per_species is not None:
        kw["n_per_species"] = int(n_per_species)
    if seed is not None:
        kw["seed"] = int(seed)
    return fn(**kw)


def random_cloud(n_per_species, mass, charge, temperature, seed, drift=None,
                 density=None, eps_rule: float = 0.05, shuffled: bool = True) -> Workload:
    """Generic Maxwellian multi-species cloud for edge-case tests (ragged counts, S up to 16)."""
    rng = np.random.default_rng(seed)
    S = len(mass)
    density = [1.0] * S if density is None else density
    drift = [(0.0, 0.0, 0.0)] * S if drift is None else drift
    sp = []
    for k in range(S):
        n_k = int(n_per_species[k])
        z = rng.standard_normal((n_k, 3))
        wr = _uniform_weights(rng, n_k)
        vk = z * np.sqrt(temperature[k] / mass[k]) + np.asarray(drift[k], dtype=np.float64)
        sp.append(dict(m=float(mass[k]), q=float(charge[k]), n=float(density[k]), v=vk,
                       w_raw=wr, T=float(temperature[k])))
    return _assemble("random_cloud", sp, rng, shuffled, dt=0.01, n_steps=1, seed=seed,
                     eps_rule=eps_rule)


# ---------------------------------------------------------------------------------------------------
# the paper's own 2-V tests, run through the 3-V path with
# v_z = 0 (then the 3-V scheme IS the paper's 2-V scheme, reading D1).  Markers sit on an N x N mesh
# of cell centres in [-L_s, L_s]^2, L_s = 5 v_t,s, with weights w_p = (2L/N)^2 f_s(v_p) of the (anisotropic,
# drifting) Maxwellian of Eq. (34), normalised to n_s (Eq. 35); eps_s = 1.2 (L_s/N)^1.98 evaluated in SI
# (PAPER.md:208).  Computation is in normalised units: velocity v0 = sqrt(T0/m_e), mass m_e, density n0,
# time t0 = m_e^2 v0^3 (8 pi eps0^2)/(e^4 lnLambda n0), in which nu_ss' = q_s^2 q_s'^2 (reading U1) and k_B T0 = 1.
E_CHARGE = 1.602176634e-19
M_E_KG = 9.1093837015e-31
EPS0 = 8.8541878128e-12
PAPER_TESTS = {
    # name, T0 [eV], lnLambda, species: (mass/m_e, charge, Tx/T0, Ty/T0, ux/v0, uy/v0)
    1: ("E1_electron_positron", 1000.0, 16.0, [(1.0, -1.0, 1.0, 1.0, -1.0, 0.125), (1.0, +1.0, 1.0, 1.0, 0.0, -0.125)]),
    2: ("E2_ei_velocity_relaxation", 400.0, 15.0, [(1.0, -1.0, 1.0, 1.0, 0.5, 0.0), (200.0, +1.0, 1.0, 1.0, 0.0, 0.0)]),
    3: ("E3_eD_isotropisation", 400.0, 14.6, [(1.0, -1.0, 1.0, 0.75, 0.0, 0.0),
                                              (3670.48, +1.0, 0.625, 0.5, 0.0, 0.0)]),
}


def paper_time_unit(T0_eV: float, lnLambda: float, n0: float = 1e20) -> float:
    """Seconds per normalised time unit: t0 = m_e^2 v0^3 (8 pi eps0^2)/(e^4 lnLambda n0), v0 = sqrt(T0/m_e)."""
    v0 = np.sqrt(T0_eV * E_CHARGE / M_E_KG)
    return float(M_E_KG ** 2 * v0 ** 3 * 8.0 * np.pi * EPS0 ** 2 / (E_CHARGE ** 4 * lnLambda * n0))


def paper_test(test: int, n_grid: int = 32, dt_seconds: float = 1e-8, n_steps: Optional[int] = None) -> Workload:
    """One of the paper's tests 3.1-3.3 (E1-E3 of SURVEY.md section 2.4) as a Workload (deterministic: no rng)."""
    name, T0, lnL, species = PAPER_TESTS[test]
    v0 = np.sqrt(T0 * E_CHARGE / M_E_KG)
    t0 = paper_time_unit(T0, lnL)
    mass, charge, eps, vs, ws, ids = [], [], [], [], [], []
    for k, (m, q, Tx, Ty, ux, uy) in enumerate(species):
        vt = np.sqrt(0.5 * (Tx + Ty) / m)                        # thermal speed of the mean temperature, units of v0
        L = 5.0 * vt
        c = -L + (np.arange(n_grid) + 0.5) * (2.0 * L / n_grid)  # cell centres
        X, Y = np.meshgrid(c, c, indexing="ij")
        f = np.exp(-m * (X - ux) ** 2 / (2.0 * Tx) - m * (Y - uy) ** 2 / (2.0 * Ty))   # Eq. (34) up to its constant
        w = (f / f.sum()).ravel()                                 # Eq. (35), normalised to n_s = 1
        keep = w > 1e-300
        v = np.stack([X.ravel()[keep], Y.ravel()[keep], np.zeros(int(keep.sum()))], axis=1)
        w = w[keep] / w[keep].sum()
        eps_si = 1.2 * (L * v0 / n_grid) ** 1.98                  # PAPER.md:208, in (m/s)^1.98 read as (m/s)^2
        mass.append(m); charge.append(q); eps.append(eps_si / v0 ** 2)
        vs.append(v); ws.append(w); ids.append(np.full(w.shape[0], k, dtype=np.int32))
    dt = dt_seconds / t0
    return Workload(name=name, mass=np.array(mass), charge=np.array(charge), density=np.ones(len(species)),
                    eps=np.array(eps), v=np.ascontiguousarray(np.concatenate(vs)), w=np.concatenate(ws),
                    species_id=np.concatenate(ids), dt=float(dt),
                    n_steps=int(n_steps if n_steps is not None else round(1e-3 / dt_seconds)), tol=1e-12, max_iter=30,
                    notes={"t0_seconds": t0, "v0_m_per_s": float(v0), "T0_eV": T0, "lnLambda": lnL, "n_grid": n_grid,
                           "two_v": True, "species": species})


def shard_cells(cell_offset, rank: int, world: int):
    """Contiguous range [c0, c1) of collision cells for `rank` of `world` (cells are
    independent, so a batch shards over GPUs with no data-path collective).  The cut points balance the pairwise work
    sum_c n_c^2 (pass 2 dominates a cell's cost), every cell belongs to exactly one rank, order is preserved.
    Pure index arithmetic on the host: none of the method's arithmetic lives here."""
    off = np.ascontiguousarray(cell_offset, dtype=np.int64)
    n = np.diff(off).astype(np.float64)
    if world < 1 or not (0 <= rank < world):
        raise ValueError("shard_cells: need 0 <= rank < world")
    if n.size == 0:
        return 0, 0
    cum = np.concatenate([[0.0], np.cumsum(n * n)])
    total = cum[-1]
    if total == 0.0:                                   # only empty cells: split by count
        cuts = [(n.size * r) // world for r in range(world + 1)]
    else:
        # cell c goes to the rank whose share contains the midpoint of its work interval
        mid = 0.5 * (cum[:-1] + cum[1:])
        owner = np.minimum((mid * world / total).astype(np.int64), world - 1)
        owner = np.maximum.accumulate(owner)
        cuts = [int(np.searchsorted(owner, r, side="left")) for r in range(world)] + [int(n.size)]
    return cuts[rank], cuts[rank + 1]
