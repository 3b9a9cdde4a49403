"""Pins of the oracle's discrete-gradient step O4b (Eqs. 46-49; reading DG1: Gonzalez'
midpoint discrete gradient of S_eps).  None of them is the oracle checked against itself: the fixed-point
equation, Eq. (48) and Eq. (49) are re-evaluated here in numpy from the oracle's primitive passes (which have
their own pins), and the conservation / monotonicity statements are the paper's."""
import numpy as np
import pytest

from paper_2212_00663_b200 import workloads as W


def _make(oracle_mod, n=40, cfg=0):
    wl = W.make(cfg, n_per_species=n, shuffled=True)
    return wl, oracle_mod.LandauRef(wl.mass, wl.charge, wl.eps, n_q=wl.n_q, nu0=wl.nu0)


def _pair_sum_eq49(wl, u, Gbar):
    """(1/2) sum_{p,q} nu w_p w_q Gamma.Q(u_p-u_q).Gamma, Gamma = Gbar_p/m_s - Gbar_q/m_s' (Eq. 49, plain loops)."""
    m = wl.mass[wl.species_id]
    q2 = wl.charge[wl.species_id] ** 2
    g = Gbar / m[:, None]
    tot = 0.0
    for p in range(len(m)):
        z = u[p] - u
        c = g[p] - g
        r2 = (z * z).sum(1)
        ok = r2 > 0
        r = np.sqrt(r2[ok])
        quad = ((c[ok] * c[ok]).sum(1) - (z[ok] * c[ok]).sum(1) ** 2 / r2[ok]) / r
        tot += 0.5 * (wl.nu0 * q2[p] * q2[ok] * wl.w[p] * wl.w[ok] * quad).sum()
    return tot


def test_dg_step_satisfies_its_equations(oracle_mod):
    wl, o = _make(oracle_mod)
    dt = 0.01
    o.set_markers(wl.v, wl.w, wl.species_id)
    rc, it, res, conv = o.step_dg(dt, 1e-14, 200)
    assert rc == 0 and conv
    v0, v1 = wl.v, o.get_markers()
    dv = v1 - v0
    u = 0.5 * (v0 + v1)
    Gu, _ = o.entropy_grad(u, wl.w, wl.species_id, with_entropy=True)
    _, S0 = o.entropy_grad(v0, wl.w, wl.species_id, with_entropy=True)
    _, S1 = o.entropy_grad(v1, wl.w, wl.species_id, with_entropy=True)
    lin = (wl.w[:, None] * Gu * dv).sum()
    lam = (S1.sum() - S0.sum() - lin) / (dv * dv).sum()
    Gbar = Gu + lam * dv / wl.w[:, None]
    # Eq. (48): the discrete-gradient property, exact by construction
    assert abs((dv * wl.w[:, None] * Gbar).sum() - (S1.sum() - S0.sum())) <= 1e-13 * abs(S0.sum())
    # the Gonzalez correction is a third-order remainder: tiny against the gradient itself
    assert np.abs(lam * dv / wl.w[:, None]).max() <= 1e-3 * np.abs(Gu).max()
    # Eq. (46): the converged state solves v1 = v0 + dt * O3(u; Gbar)
    V = o.pair_field(u, wl.w, wl.species_id, Gbar)
    assert np.linalg.norm(v0 + dt * V - v1) <= 1e-11 * np.linalg.norm(v1)
    # Eq. (49): entropy production = positive semidefinite pair sum
    prod = _pair_sum_eq49(wl, u, Gbar)
    assert prod > 0
    assert abs((S1.sum() - S0.sum()) / dt - prod) <= 1e-9 * prod


def test_dg_step_conserves_momentum_and_energy(oracle_mod):
    """"This modification will also retain the discrete energy and momentum conservation"."""
    wl, o = _make(oracle_mod, n=32, cfg=4)
    o.set_markers(wl.v, wl.w, wl.species_id)
    m0 = o.moments()
    for _ in range(3):
        rc, it, res, conv = o.step_dg(2e-3, 1e-13, 200)
        assert rc == 0 and conv
    m1 = o.moments()
    wm_abs = (wl.w * wl.mass[wl.species_id] * np.abs(wl.v).sum(1)).sum()
    assert np.abs(m1["P"].sum(0) - m0["P"].sum(0)).max() <= 1e-13 * wm_abs
    assert abs(m1["K"].sum() - m0["K"].sum()) <= 1e-13 * m0["K"].sum()


def test_dg_step_is_second_order_close_to_eq24(oracle_mod):
    """Eq. (46) differs from Eq. (24) only in where G is evaluated (midpoint discrete gradient vs t_n):
    the two one-step results differ by O(dt^2)."""
    wl, o = _make(oracle_mod, n=24)
    diffs = []
    for dt in (4e-3, 2e-3):
        o.set_markers(wl.v, wl.w, wl.species_id)
        assert o.step(dt, 1e-14, 200)[0] == 0
        a = o.get_markers()
        o.set_markers(wl.v, wl.w, wl.species_id)
        assert o.step_dg(dt, 1e-14, 200)[0] == 0
        b = o.get_markers()
        diffs.append(np.linalg.norm(a - b))
    assert diffs[0] > 0 and 3.0 < diffs[0] / diffs[1] < 5.0


def test_dg_entropy_never_decreases_near_equilibrium(oracle_mod):
    """Eq. (49): S_eps^{n+1} >= S_eps^n in every step, also after equilibrium is approximately reached,
    where Eq. (24) may lose entropy (Fig. 6)."""
    rng = np.random.default_rng(11)
    n = 48
    v = rng.standard_normal((n, 3))
    w = np.full(n, 1.0 / n)
    sid = np.zeros(n, dtype=np.int32)
    o = oracle_mod.LandauRef([1.0], [1.0], [0.3], n_q=4, nu0=1.0)
    o.set_markers(v, w, sid)
    S = [o.moments()["S_eps"].sum()]
    for _ in range(12):
        rc, it, res, conv = o.step_dg(0.05, 1e-13, 300)
        assert rc == 0 and conv
        S.append(o.moments()["S_eps"].sum())
    assert np.all(np.diff(S) >= -1e-13 * abs(S[0])), np.diff(S)
