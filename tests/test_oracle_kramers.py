"""Pins for oracle/kramers.py and the host post-processing of sweeps (Fig. 10)."""
import math

import numpy as np
import pytest
from scipy import optimize

from oracle import kramers
from paper_1802_05065_b200 import analysis


def test_barrier_value_printed_in_the_paper():
    # Fig. 10 caption: Delta U = 0.0342 at gamma = 0.5; the run used V0 = 0.05
    assert round(kramers.barrier(0.5, 0.05), 4) == 0.0342
    assert kramers.barrier(0.7) == pytest.approx(0.314727, abs=1e-6)
    assert kramers.barrier(0.0) == pytest.approx(2.0) and kramers.barrier(1.0) == pytest.approx(0.0, abs=1e-15)


def test_barrier_is_the_potential_difference_between_its_extrema():
    for g in (0.1, 0.5, 0.7, 0.9, 0.99):
        lo = optimize.minimize_scalar(lambda x: kramers.potential(x, g), bounds=(-1.0, math.pi / 2), method="bounded",
                                      options=dict(xatol=1e-12)).x
        hi = optimize.minimize_scalar(lambda x: -kramers.potential(x, g), bounds=(math.pi / 2, math.pi + 0.5), method="bounded",
                                      options=dict(xatol=1e-12)).x
        assert lo == pytest.approx(math.asin(g), abs=1e-6) and hi == pytest.approx(math.pi - math.asin(g), abs=1e-6)
        assert kramers.barrier(g, 0.3) == pytest.approx(0.3 * (kramers.potential(hi, g) - kramers.potential(lo, g)), rel=1e-9)


def test_slopes_recover_the_barrier_from_exact_laws():
    theta = np.array([0.02, 0.025, 0.03, 0.04, 0.05])
    du = 0.0342
    tau_k = 7.0 / theta * np.exp(du / theta)
    tau_a = 3.0 * np.exp(du / theta)
    assert kramers.kramers_slope(theta, tau_k) == pytest.approx(du, rel=1e-10)
    assert kramers.arrhenius_slope(theta, tau_a) == pytest.approx(du, rel=1e-10)
    # the two readings of the same data differ by d ln(theta) / d(1/theta) = -theta: Arrhenius slope = Kramers slope + ~theta
    diff = kramers.arrhenius_slope(theta, tau_k) - kramers.kramers_slope(theta, tau_k)
    assert theta.min() < diff < theta.max()
    # the product's numpy post-processing agrees with the oracle's normal equations
    assert analysis.barrier_from_sweep(theta, tau_k, "kramers") == pytest.approx(kramers.kramers_slope(theta, tau_k), rel=1e-9)
    assert analysis.barrier_from_sweep(theta, tau_k, "arrhenius") == pytest.approx(kramers.arrhenius_slope(theta, tau_k), rel=1e-9)


def test_mean_escape_time_ignores_censored_entries():
    f = np.array([[1.0, 3.0, -1.0, 2.0], [5.0, -1.0, -1.0, 7.0]])
    s = np.array([[0, 0, 1, 0], [0, 1, 1, 0]])
    mean, sem, cens = analysis.mean_escape_time(f, s)
    assert np.allclose(mean, [2.0, 6.0]) and list(cens) == [1, 2]
    assert sem[0] == pytest.approx(np.std([1.0, 3.0, 2.0], ddof=1) / math.sqrt(3))
