"""Analytic comparison curves the paper plots its simulations against (host helpers, numpy only).

These are NOT part of the hot path and load no native code; they turn a measured moment history
into "fitted rate / analytic rate" numbers.

Units.  The paper writes the rates in SI with the factor e_s^2 e_s'^2 lnLambda/(4 pi eps0)^2.
Because nu_ss' = e_s^2 e_s'^2 lnLambda/(8 pi eps0^2), that factor equals
nu_ss'/(2 pi); every function takes it as `coupling` so the same code serves the normalised
runs (coupling = nu0 q_s^2 q_s'^2/(2 pi), k_B = 1) and the paper's SI examples (the pins in
tests/test_analytic.py use the SI numbers printed in PAPER.md:287).
"""
from __future__ import annotations

import math

import numpy as np


def coupling_from_nu(nu_ss: float) -> float:
    """e_s^2 e_s'^2 lnLambda/(4 pi eps0)^2 expressed through nu_ss' of PAPER.md:37."""
    return nu_ss / (2.0 * math.pi)


def isotropisation_bracket(A: float) -> float:
    """A^-2 [ -3 + (A+3) atan(sqrt(A))/sqrt(A) ] of Eq. (41).

    The paper states it for T_perp > T_par (A > 0).  Reading U5: for A < 0 the same analytic
    function continues as atanh(sqrt(-A))/sqrt(-A); the A -> 0 limit is 4/15.
    """
    if abs(A) < 1e-4:
        # series: atan(x)/x = 1 - x^2/3 + x^4/5 - x^6/7 + ...,  x^2 = A
        return 4.0 / 15.0 - 8.0 * A / 35.0 + 4.0 * A * A / 21.0
    if A > 0:
        r = math.sqrt(A)
        f = math.atan(r) / r
    else:
        r = math.sqrt(-A)
        f = math.atanh(r) / r
    return (-3.0 + (A + 3.0) * f) / (A * A)


def isotropisation_rate(m: float, n: float, T_par: float, T_perp: float, coupling: float) -> float:
    """1/tau_s of Eq. (41), PAPER.md:255 (3-V form), A = T_perp/T_par - 1, k_B = 1."""
    A = T_perp / T_par - 1.0
    return (2.0 * math.sqrt(math.pi) * coupling * n / (math.sqrt(m) * T_par ** 1.5)
            * isotropisation_bracket(A))


def isotropisation_rate_2v(m: float, n: float, T_x: float, T_y: float, coupling: float) -> float:
    """2-V variant stated after Eq. (43): A = T_>/T_< - 1 and T_par -> T_<."""
    hi, lo = max(T_x, T_y), min(T_x, T_y)
    A = hi / lo - 1.0
    return (2.0 * math.sqrt(math.pi) * coupling * n / (math.sqrt(m) * lo ** 1.5)
            * isotropisation_bracket(A))


def integrate_isotropisation(m, n, T_par0, T_perp0, coupling, t_end, n_sub=20000):
    """Integrate Eq. (40): dT_perp/dt = -(1/2) dT_par/dt = -(T_perp - T_par)/tau_s.

    Returns (t, T_par, T_perp) arrays (classical RK4 with the rate re-evaluated on the fly).
    """
    def rhs(y):
        Tpar, Tperp = y
        r = isotropisation_rate(m, n, Tpar, Tperp, coupling)
        dperp = -(Tperp - Tpar) * r
        return np.array([-2.0 * dperp, dperp])

    t = np.linspace(0.0, t_end, n_sub + 1)
    h = t[1] - t[0]
    y = np.array([T_par0, T_perp0], dtype=np.float64)
    out = np.empty((n_sub + 1, 2))
    out[0] = y
    for i in range(n_sub):
        k1 = rhs(y)
        k2 = rhs(y + 0.5 * h * k1)
        k3 = rhs(y + 0.5 * h * k2)
        k4 = rhs(y + h * k3)
        y = y + (h / 6.0) * (k1 + 2 * k2 + 2 * k3 + k4)
        out[i + 1] = y
    return t, out[:, 0], out[:, 1]


def thermalisation_rate(m_s, m_sb, n_sb, T_s, T_sb, coupling) -> float:
    """1/tau-bar^{s\\s'} of Eq. (45), as printed, with the field-species density
    n_s' (reading U6).  Reading G1: the caption value of Fig. 3 (1.6e-3 s) is this formula's
    2.83e-3 s divided by sqrt(pi).  The formula, not the caption, is right: a Monte Carlo estimate of the
    Landau operator's energy-exchange integral for two Maxwellians equals it to 0.1 %
    (tests/test_analytic.py::test_thermalisation_rate_equals_the_landau_energy_exchange_integral).
    """
    return ((8.0 / 3.0) * math.sqrt(2.0 * math.pi * m_s * m_sb) * coupling * n_sb
            / (m_s * T_sb + m_sb * T_s) ** 1.5)


def temperature_gap_rate(m_a, m_b, n_a, n_b, T_a, T_b, coupling) -> float:
    """d ln(T_a - T_b)/dt = -(1/tau^{a\\b} + 1/tau^{b\\a}) from Eq. (44)."""
    return -(thermalisation_rate(m_a, m_b, n_b, T_a, T_b, coupling)
             + thermalisation_rate(m_b, m_a, n_a, T_b, T_a, coupling))


def fit_exponential_rate(t, y) -> float:
    """Least-squares slope of ln|y| against t (the decay rate of a gap history)."""
    t = np.asarray(t, dtype=np.float64)
    ly = np.log(np.abs(np.asarray(y, dtype=np.float64)))
    tm, lm = t.mean(), ly.mean()
    return float(((t - tm) * (ly - lm)).sum() / ((t - tm) ** 2).sum())


def temperatures_from_moments(mass, n, P, K, stress=None):
    """3-V forms of Eqs. (30)-(33), from landau_moments outputs (k_B = 1).

    u_s = P_s/(m_s n_s);  T_s = (2/3)(K_s - |P_s|^2/(2 m_s n_s))/n_s;
    per-axis T_s^i = (stress_ii - P_i^2/(m_s n_s))/n_s when `stress` (S x 6) is given.
    """
    mass = np.asarray(mass, dtype=np.float64)
    n = np.asarray(n, dtype=np.float64)
    P = np.asarray(P, dtype=np.float64)
    K = np.asarray(K, dtype=np.float64)
    u = P / (mass * n)[:, None]
    T = (2.0 / 3.0) * (K - (P ** 2).sum(axis=1) / (2.0 * mass * n)) / n
    out = dict(u=u, T=T)
    if stress is not None:
        stress = np.asarray(stress, dtype=np.float64)
        out["T_axis"] = (stress[:, :3] - P ** 2 / (mass * n)[:, None]) / n[:, None]
    return out
