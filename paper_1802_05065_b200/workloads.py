"""The five BASELINE.json configs as plain data.  No arithmetic of the method lives here: only
parameter values (`asin` for the well bottom phi0) -- the random inputs are generated inside the kernels / the oracle by
Philox from (seed, trajectory id), so a "seeded synthetic input" is (params, seed, first_id, n_traj).

This module is the one thing shared by the CUDA path's callers and the oracle's callers (tests, bench): both
`paper_1802_05065_b200.make_params(**w["params"])` and `oracle.make_params(**w["params"])` accept these dicts.
"""
from __future__ import annotations

import math

_TWO_PI = 2.0 * math.pi

CONFIGS = {
    # C1: drifted Brownian motion, inverse-Gaussian first-passage law (textbook pin; not in the paper)
    "c1": dict(params=dict(model="overdamped", scheme="em", precision="fp64", alpha=0.0, temperature=0.1, amp=0.0,
                           gamma0=1.0, nu=0.0, phi0=0.0, v0=0.0, threshold=1.0, dt=1e-3),
               n_traj=10**4, seed=1, t_max=100.0, n64_ref=39, hist=None),
    # C2: Alg. 1 ESCAPETIME, constant bias
    "c2": dict(params=dict(model="underdamped", scheme="heun", precision="fp64", alpha=0.1, temperature=0.05, amp=1.0,
                           gamma0=0.9, nu=0.0, phi0=math.asin(0.9), v0=0.0, threshold=math.asin(0.9) + _TWO_PI, dt=0.01),
               n_traj=10**5, seed=2, t_max=1e4, n64_ref=83, hist=None),
    # C3: Alg. 3 SWITCHINGCURRENT, slow ramp from gamma = 0; histogram of gamma at escape
    "c3": dict(params=dict(model="underdamped", scheme="heun", precision="fp64", alpha=0.1, temperature=0.01, amp=1.0,
                           gamma0=0.0, nu=1e-6, phi0=0.0, v0=0.0, threshold=_TWO_PI, dt=0.02),
               n_traj=10**6, seed=3, t_max=1.05 / 1e-6, n64_ref=83, hist=("gamma", 0.0, 1.05, 1000)),
    # C4: experiment-time-scale sweep, fp32 state + Kahan-compensated time
    "c4": dict(params=dict(model="underdamped", scheme="heun", precision="fp32", alpha=0.05, temperature=0.005, amp=1.0,
                           gamma0=0.5, nu=1e-9, phi0=math.asin(0.5), v0=0.0, threshold=math.asin(0.5) + _TWO_PI, dt=0.05),
               n_traj=65536, seed=4, t_max=(1.05 - 0.5) / 1e-9, n64_ref=63, hist=("gamma", 0.5, 1.05, 1000)),
    # C5: strongly imbalanced rare-event escape, overdamped washboard (Appendix A)
    "c5": dict(params=dict(model="overdamped", scheme="em", precision="fp64", alpha=0.0, temperature=0.03, amp=1.0,
                           gamma0=0.7, nu=0.0, phi0=math.asin(0.7), v0=0.0, threshold=math.asin(0.7) + _TWO_PI, dt=5e-3),
               n_traj=4 * 10**6, seed=5, t_max=1e8 * 5e-3, n64_ref=56, hist=None),
}


def workload(name: str, **overrides) -> dict:
    """A copy of a config; keyword overrides go into the top level (n_traj, seed, t_max) or into params."""
    base = CONFIGS[name]
    w = dict(base)
    w["params"] = dict(base["params"])
    for k, val in overrides.items():
        if k in w and k != "params":
            w[k] = val
        else:
            w["params"][k] = val
    w["name"] = name
    return w
