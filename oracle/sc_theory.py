"""ORACLE (test infrastructure, not product code) -- the Kramers-adiabatic switching-current distribution the paper
compares Fig. 11(b) with ("the adiabatic approximation used in [39] that, neglecting non-equilibrium
corrections to the Kramers' theory, gives a formula for the SC cumulative distribution only valid in the limit of vanishingly
small bias ramp speed"; ref. [39] = Fulton and Dunkleberger).

In the library's units (time in 1/omega_p0, energies in E_J; R2) the washboard U(phi) = -cos phi - gamma phi has,
for 0 <= gamma < 1,
    barrier           Delta U(gamma) = 2 [ sqrt(1 - gamma^2) - gamma arccos gamma ]          (oracle/kramers.barrier)
    well = barrier frequency   omega(gamma) = (1 - gamma^2)^(1/4)
and Kramers' escape rate for moderate-to-strong damping alpha is
    Gamma(gamma) = a_t * omega / (2 pi) * exp(-Delta U / T),   a_t = sqrt(1 + (alpha / (2 omega))^2) - alpha / (2 omega).
Ramping gamma(t) = gamma0 + nu t so slowly that the well stays in equilibrium (adiabatic), the probability of having switched
below the bias gamma is
    P(gamma) = 1 - exp( -(1/nu) * integral_{gamma0}^{gamma} Gamma(g) dg ).
Plain numpy, fp64, composite trapezoid on a uniform grid (the integrand is smooth; the grid is fine enough that halving it
changes no returned digit the tests look at).
"""
from __future__ import annotations

import math

import numpy as np

from . import kramers


def rate(gamma: float, alpha: float, temperature: float, prefactor: str = "moderate") -> float:
    """Kramers' escape rate at fixed bias.  prefactor: "moderate" (a_t above) or "tst" (transition-state theory, a_t = 1)."""
    if not 0.0 <= gamma < 1.0:
        raise ValueError("a metastable well exists only for 0 <= gamma < 1")
    omega = (1.0 - gamma * gamma) ** 0.25
    a_t = 1.0
    if prefactor == "moderate":
        x = alpha / (2.0 * omega)
        a_t = math.sqrt(1.0 + x * x) - x
    elif prefactor != "tst":
        raise ValueError(prefactor)
    return a_t * omega / (2.0 * math.pi) * math.exp(-kramers.barrier(gamma) / temperature)


def switching_cdf(alpha: float, temperature: float, nu: float, gamma0: float = 0.0, n_grid: int = 200001, prefactor: str = "moderate"):
    """(gamma grid on [gamma0, 1), P(gamma) on it)."""
    g = np.linspace(gamma0, 1.0, n_grid, endpoint=False)
    r = np.array([rate(float(x), alpha, temperature, prefactor) for x in g])
    h = g[1] - g[0]
    integral = np.concatenate([[0.0], np.cumsum(0.5 * (r[1:] + r[:-1])) * h])
    return g, 1.0 - np.exp(-integral / nu)


def quantile(g, cdf, q: float) -> float:
    """gamma with P(gamma) = q, linear interpolation on the grid."""
    i = int(np.searchsorted(cdf, q))
    if i == 0 or i >= len(g):
        raise ValueError("quantile outside the grid")
    t = (q - cdf[i - 1]) / (cdf[i] - cdf[i - 1])
    return float(g[i - 1] + t * (g[i] - g[i - 1]))


def moments(g, cdf):
    """(mean, standard deviation) of the switching bias; the mass still in the well at gamma -> 1 switches there."""
    p = np.diff(cdf)
    mid = 0.5 * (g[1:] + g[:-1])
    rest = 1.0 - cdf[-1]
    mean = float(np.sum(p * mid) + rest * 1.0)
    var = float(np.sum(p * (mid - mean) ** 2) + rest * (1.0 - mean) ** 2)
    return mean, math.sqrt(var)
