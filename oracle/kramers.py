"""ORACLE (test infrastructure, not product code) -- the Arrhenius / Kramers relations of PAPER.md:357-379.

  barrier(gamma, v0)   Delta U of the tilted washboard U(phi) = -v0 (cos phi + gamma phi) between the well bottom
                       phi_min = arcsin(gamma) and the barrier top phi_max = pi - arcsin(gamma):
                       Delta U = v0 * 2 [sqrt(1 - gamma^2) - gamma arccos(gamma)].  The paper prints 0.0342 for gamma = 0.5 (Fig. 10).
  arrhenius_slope      Eq. (12):  <tau> ~ exp(Delta U / theta)           =>  Delta U = slope of ln <tau> against 1/theta
  kramers_slope        Eqs. (13)-(14): <tau> ~ (1/theta) exp(Delta U / theta) => Delta U = slope of ln(theta <tau>) against 1/theta
                       (the printed "Delta theta" in Eqs. (12)-(14) is a garble for theta, G3)
Slopes are ordinary least squares written out from the normal equations.  fp64, plain Python / numpy.
"""
from __future__ import annotations

import math

import numpy as np


def potential(phi: float, gamma: float, v0: float = 1.0) -> float:
    return -v0 * (math.cos(phi) + gamma * phi)


def barrier(gamma: float, v0: float = 1.0) -> float:
    if not 0.0 <= gamma <= 1.0:
        raise ValueError("the washboard has a barrier only for 0 <= gamma <= 1")
    return v0 * 2.0 * (math.sqrt(1.0 - gamma * gamma) - gamma * math.acos(gamma))


def _ols_slope(x, y) -> float:
    x = np.asarray(x, dtype=np.float64)
    y = np.asarray(y, dtype=np.float64)
    n = len(x)
    if n < 2 or len(y) != n:
        raise ValueError("need at least two points")
    sx, sy, sxx, sxy = x.sum(), y.sum(), (x * x).sum(), (x * y).sum()
    return float((n * sxy - sx * sy) / (n * sxx - sx * sx))


def arrhenius_slope(theta, mean_tau) -> float:
    theta = np.asarray(theta, dtype=np.float64)
    return _ols_slope(1.0 / theta, np.log(np.asarray(mean_tau, dtype=np.float64)))


def kramers_slope(theta, mean_tau) -> float:
    theta = np.asarray(theta, dtype=np.float64)
    return _ols_slope(1.0 / theta, np.log(theta * np.asarray(mean_tau, dtype=np.float64)))
