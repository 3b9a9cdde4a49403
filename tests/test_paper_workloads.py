"""Host-side checks of the paper's own initial data (workloads.paper_test; Eqs. 34-35)."""
import numpy as np

from paper_2212_00663_b200 import workloads as W


def test_time_unit_matches_the_papers_collision_time_scale():
    """dt = 1e-8 s is chosen against an e-e collision time "of the order of 5e-6 s": one
    normalised time unit (nu_ee = 1) must be of that order for the paper's 400 eV / 1e20 m^-3 / lnL ~ 15 plasma."""
    t0 = W.paper_time_unit(400.0, 14.6)
    assert 0.5e-6 < t0 < 5e-6
    assert abs(W.paper_time_unit(400.0, 14.6) / W.paper_time_unit(400.0, 29.2) - 2.0) < 1e-12   # ~ 1/lnLambda
    assert abs(W.paper_time_unit(1600.0, 14.6) / t0 - 8.0) < 1e-12                               # ~ T^(3/2)


def test_grid_initialisation_reproduces_the_maxwellian_moments():
    """Eq. (35) weights on the N x N mesh of cell centres, normalised to n_s: density 1, flow and anisotropic
    temperatures of Eq. (34) to quadrature accuracy, v_z = 0 (2-V)."""
    for test in (1, 2, 3):
        wl = W.paper_test(test, n_grid=32)
        assert wl.n_species == 2 and np.all(wl.v[:, 2] == 0.0) and np.all(wl.w > 0)
        for s, (m, q, Tx, Ty, ux, uy) in enumerate(wl.notes["species"]):
            sel = wl.species_id == s
            w, v = wl.w[sel], wl.v[sel]
            assert abs(w.sum() - 1.0) < 1e-14
            u = (w[:, None] * v).sum(0)
            assert abs(u[0] - ux) < 2e-3 * np.sqrt(Tx / m) + 1e-12 and abs(u[1] - uy) < 2e-3 * np.sqrt(Ty / m) + 1e-12
            T = m * (w[:, None] * (v - u) ** 2).sum(0)
            assert abs(T[0] / Tx - 1) < 2e-3 and abs(T[1] / Ty - 1) < 2e-3
            # eps_s = 1.2 (L_s/N)^1.98: a fraction ~0.2-0.3 of the squared mesh spacing
            h = 10.0 * np.sqrt(0.5 * (Tx + Ty) / m) / 32
            assert 0.15 < wl.eps[s] / h ** 2 < 0.35
    wl = W.paper_test(3)
    assert abs(wl.dt * wl.notes["t0_seconds"] - 1e-8) < 1e-20 and wl.n_steps == 100000
