"""Pins for the analytic comparison curves (O6) against numbers printed in the paper."""
import math
from pathlib import Path

import numpy as np

from paper_2212_00663_b200 import analytic as A

GOLDEN = Path(__file__).resolve().parent / "golden"

E = 1.602176634e-19
EPS0 = 8.8541878128e-12
ME = 9.1093837015e-31
MD = 3.3435837724e-27


def printed():
    out = {}
    for line in (GOLDEN / "paper_printed_times.txt").read_text().splitlines():
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split()
            out[k] = float(v)
    return out


def test_eq41_reproduces_printed_isotropisation_times():
    """tau_i = 1.7e-4 s (match), tau_e = 5.2e-6 s (7 %, reading G2)."""
    p = printed()
    coupling = E ** 4 * 14.6 / (4 * math.pi * EPS0) ** 2
    tau_i = 1 / A.isotropisation_rate_2v(MD, 1e20, 250 * E, 200 * E, coupling)
    tau_e = 1 / A.isotropisation_rate_2v(ME, 1e20, 400 * E, 300 * E, coupling)
    assert abs(tau_i - p["tau_i"]) < 0.05e-4          # printed to two digits
    assert abs(tau_e / p["tau_e"] - 1) < 0.08


def test_eq45_vs_printed_thermalisation_time():
    """Reading G1: Eq. (45) as printed gives 2.83e-3 s = caption's 1.6e-3 s times sqrt(pi)."""
    p = printed()
    coupling = E ** 4 * 14.6 / (4 * math.pi * EPS0) ** 2
    tau = 1 / A.thermalisation_rate(ME, MD, 1e20, 350 * E, 225 * E, coupling)
    assert abs(tau / math.sqrt(math.pi) - p["tau_ei"]) < 0.05e-3


def test_bracket_limits_and_continuation():
    assert abs(A.isotropisation_bracket(0.0) - 4 / 15) < 1e-15
    for a in (1e-4, -1e-4):   # series and closed form agree where they meet
        assert abs(A.isotropisation_bracket(a * 1.0001) - A.isotropisation_bracket(a * 0.9999)) < 1e-7
    # closed form by hand at A = 1: -3 + 4 atan(1) = pi - 3
    assert abs(A.isotropisation_bracket(1.0) - (math.pi - 3)) < 1e-15
    # A = -1/2 (config 2 electrons): atanh(sqrt(.5))/sqrt(.5)
    x = math.sqrt(0.5)
    assert abs(A.isotropisation_bracket(-0.5) - 4 * (-3 + 2.5 * math.atanh(x) / x)) < 1e-14


def test_normalised_rates_for_configs_1_and_2():
    c = A.coupling_from_nu(1.0)
    assert abs(A.thermalisation_rate(1, 1836, 1, 2, 1, c) - 2.048e-4) < 1e-7
    assert abs(A.isotropisation_rate(1, 1, 2.0, 1.0, c) - 0.09266) < 1e-5
    t, Tpar, Tperp = A.integrate_isotropisation(1, 1, 2.0, 1.0, c, 5.0, 2000)
    assert abs((Tpar[-1] - Tperp[-1]) - 0.244) < 1e-3
    # Eq. (40) conserves T_par + 2 T_perp
    np.testing.assert_allclose(Tpar + 2 * Tperp, 4.0, rtol=1e-12)


def test_fit_and_temperatures():
    t = np.linspace(0, 3, 50)
    assert abs(A.fit_exponential_rate(t, 2.5 * np.exp(-0.37 * t)) + 0.37) < 1e-12
    T = A.temperatures_from_moments([2.0], [0.5], [[0.2, 0.0, 0.0]], [0.77])
    # K = n(3T/2) + |P|^2/(2 m n)
    assert abs(T["T"][0] - (2 / 3) * (0.77 - 0.04 / 2.0) / 0.5) < 1e-15


def _mc(n, seed):
    return np.random.default_rng(seed), n


def test_thermalisation_rate_equals_the_landau_energy_exchange_integral():
    """Pin of Eq. (45) that does not come from the paper: for two drift-free Maxwellians the weak form of
    the operator (Eqs. 3-4, 16-17 with G = -grad f / f) gives, with Q(z) z = 0,
        dK_a/dt = -nu_ab (1/T_b - 1/T_a) n_a n_b E[ v . Q(v - v') . v ],   v ~ N(0, T_a/m_a), v' ~ N(0, T_b/m_b),
    i.e. 1/tau^{a\\b} = 2 nu_ab n_b E[...] / (3 T_a T_b).  A Monte Carlo estimate of that expectation (1e6 samples,
    ~0.2 % noise) equals the helper to 1 %: Eq. (45) as printed is right (the Fig. 3 caption differs by sqrt(pi) = 77 %)."""
    rng = np.random.default_rng(45)
    n = 1_000_000
    for ma, mb, nb, Ta, Tb, nu in [(1.0, 1836.0, 1.0, 2.0, 1.0, 1.0), (1836.0, 1.0, 1.0, 1.0, 2.0, 1.0),
                                   (1.0, 3.0, 0.7, 1.0, 1.5, 2.5), (2.0, 2.0, 1.3, 0.5, 0.8, 1.0)]:
        v = rng.standard_normal((n, 3)) * math.sqrt(Ta / ma)
        vp = rng.standard_normal((n, 3)) * math.sqrt(Tb / mb)
        z = v - vp
        r2, zv, v2 = (z * z).sum(1), (z * v).sum(1), (v * v).sum(1)
        mc = 2.0 * nu * nb * ((r2 * v2 - zv * zv) / r2 ** 1.5).mean() / (3.0 * Ta * Tb)
        an = A.thermalisation_rate(ma, mb, nb, Ta, Tb, A.coupling_from_nu(nu))
        assert abs(mc / an - 1.0) < 0.01, (ma, mb, mc, an)


def test_isotropisation_rate_equals_the_landau_moment_integral_both_signs_of_A():
    """Pin of Eq. (41) and of its continuation to T_par > T_perp (reading U5): for a bi-Maxwellian the
    same weak form gives  dT_par/dt = (nu n/m) E[ z_z (Q(z) M z)_z ],  z = v - v',  M = diag(m/T_perp, m/T_perp, m/T_par),
    and Eq. (40) says dT_par/dt = 2 (T_perp - T_par)/tau.  Monte Carlo (1e6 samples) against the helper, 1 %."""
    rng = np.random.default_rng(41)
    n = 1_000_000
    for m, dens, Tpar, Tperp, nu in [(1.0, 1.0, 1.0, 2.0, 1.0), (1.0, 1.0, 2.0, 1.0, 1.0), (3.0, 0.7, 1.0, 1.3, 2.0)]:
        s = np.sqrt(np.array([Tperp, Tperp, Tpar]) / m)
        z = rng.standard_normal((n, 3)) * s - rng.standard_normal((n, 3)) * s
        M = np.array([m / Tperp, m / Tperp, m / Tpar])
        Mz = z * M
        r2, zMz = (z * z).sum(1), (z * Mz).sum(1)
        e = z[:, 2] * (r2 * Mz[:, 2] - z[:, 2] * zMz) / r2 ** 1.5
        mc = (nu * dens / m) * e.mean() / (2.0 * (Tperp - Tpar))
        an = A.isotropisation_rate(m, dens, Tpar, Tperp, A.coupling_from_nu(nu))
        assert abs(mc / an - 1.0) < 0.01, (Tpar, Tperp, mc, an)
