"""Host-side post-processing of a parameter sweep (the paper's L2 layer): mean escape time per set and
the barrier estimate from its temperature dependence, Eqs. (12)-(14).  Plain numpy on results already copied back;
nothing here is on the hot path."""
from __future__ import annotations

import numpy as np


def mean_escape_time(fpt, status):
    """Per set (rows): mean of the escape times of the ESCAPED trajectories, its standard error, and the censored count.
    A set with censored trajectories has a biased mean (the cap cut the tail): the caller must look at the count."""
    fpt = np.asarray(fpt, dtype=np.float64)
    status = np.asarray(status)
    esc = status == 0
    n = esc.sum(axis=-1)
    safe = np.maximum(n, 1)
    mean = np.where(esc, fpt, 0.0).sum(axis=-1) / safe
    var = np.where(esc, (fpt - mean[..., None]) ** 2, 0.0).sum(axis=-1) / np.maximum(n - 1, 1)
    return mean, np.sqrt(var / safe), (status == 1).sum(axis=-1)


def barrier_from_sweep(theta, mean_tau, prefactor="kramers") -> float:
    """Delta U from <tau>(theta): slope of ln(<tau>) (prefactor="arrhenius", Eq. (12)) or of ln(theta <tau>)
    (prefactor="kramers", Eqs. (13)-(14)) against 1/theta."""
    theta = np.asarray(theta, dtype=np.float64)
    y = np.log(np.asarray(mean_tau, dtype=np.float64))
    if prefactor == "kramers":
        y = y + np.log(theta)
    elif prefactor != "arrhenius":
        raise ValueError("prefactor must be 'arrhenius' or 'kramers'")
    return float(np.polyfit(1.0 / theta, y, 1)[0])
