"""Pins of oracle/sc_theory.py, the Kramers-adiabatic switching-current distribution of ref. [39] that the paper compares
Fig. 11(b) with, and of the oracle's ramped underdamped path against it.

  * SURVEY.md 8(c) P7, computed in the survey session by an independent script: config 3 at nu = 1e-4: mean 0.9375, sigma
    0.0166; config 3 as stated (nu = 1e-6): mean 0.884 (lower end of "0.884...0.907"), sigma 0.0127; config 4: 0.890, 0.0066.
  * the independent numpy Heun sample of tests/golden/ramp_numpy_sample.txt (numpy's own RNG): the theory is "0.4 % low in
    mean, 5 % in width" against it.
  * limits: rate -> TST when alpha -> 0; Arrhenius slope of ln Gamma against 1/T is -Delta U; P is a distribution function.
  * the oracle's integrator on the paper's device (alpha = 0.283, T = 0.0673) at a ramp 10^5 times faster than
    the experiment: empirical CDF within 1.5 % + sampling noise of the theory, as the paper found at the true rate."""
import math

import numpy as np
import pytest

import oracle
import ref_mp
from oracle import kramers, sc_theory as sc, units as ou


def test_reproduces_the_survey_probe_numbers():
    for (alpha, T, nu, g0), (mean, sigma) in {(0.1, 0.01, 1e-4, 0.0): (0.9375, 0.0166), (0.1, 0.01, 1e-6, 0.0): (0.884, 0.0127),
                                              (0.05, 0.005, 1e-9, 0.5): (0.890, 0.0066)}.items():
        g, cdf = sc.switching_cdf(alpha, T, nu, gamma0=g0)
        m, s = sc.moments(g, cdf)
        assert m == pytest.approx(mean, abs=6e-4) and s == pytest.approx(sigma, rel=0.01), (alpha, T, nu)   # printed to 3-4 digits
    # grid independence
    g2, cdf2 = sc.switching_cdf(0.1, 0.01, 1e-4, n_grid=50001)
    assert sc.moments(g2, cdf2)[0] == pytest.approx(0.9375, abs=6e-4)


def test_against_the_independent_numpy_sample():
    gold = {r[0]: float(r[1]) for r in ref_mp.read_golden("ramp_numpy_sample.txt")}
    g, cdf = sc.switching_cdf(0.1, 0.01, 1e-4)
    m, s = sc.moments(g, cdf)
    assert m / gold["mean_gamma_sw"] - 1 == pytest.approx(-0.004, abs=0.0015)          # "0.4 % low in mean"
    assert s / gold["std_gamma_sw"] - 1 == pytest.approx(-0.05, abs=0.02)              # "5 % in width"
    for q, key in ((0.01, "q01"), (0.5, "q50"), (0.99, "q99")):
        assert sc.quantile(g, cdf, q) == pytest.approx(gold[key], abs=0.006)


def test_rate_limits_and_cdf_properties():
    # weak damping: the moderate-damping prefactor tends to transition-state theory; strong damping: to omega/alpha (Smoluchowski)
    assert sc.rate(0.5, 1e-6, 0.05) == pytest.approx(sc.rate(0.5, 0.0, 0.05, prefactor="tst"), rel=1e-6)
    om = (1 - 0.25) ** 0.25
    assert sc.rate(0.5, 50.0, 0.05) == pytest.approx(sc.rate(0.5, 0.0, 0.05, "tst") * om / 50.0, rel=2e-3)
    # Arrhenius: d ln Gamma / d(1/T) = -Delta U (the paper prints Delta U = 0.0342 for V0 = 0.05, gamma = 0.5: 0.68485 here)
    slope = (math.log(sc.rate(0.5, 0.1, 0.02)) - math.log(sc.rate(0.5, 0.1, 0.04))) / (1 / 0.02 - 1 / 0.04)
    assert -slope == pytest.approx(kramers.barrier(0.5), rel=1e-12) and kramers.barrier(0.5) * 0.05 == pytest.approx(0.0342, abs=5e-5)
    g, cdf = sc.switching_cdf(0.283, 0.0673, 1e-6)
    assert cdf[0] == 0.0 and np.all(np.diff(cdf) >= 0) and cdf[-1] == pytest.approx(1.0, abs=1e-12)
    # slower ramps switch earlier, by about T ln(10) / |dU/dgamma| per decade
    meds = [sc.quantile(*sc.switching_cdf(0.283, 0.0673, nu), 0.5) for nu in (1e-4, 1e-5, 1e-6)]
    assert meds[0] > meds[1] > meds[2]
    dU = lambda x: 2 * math.acos(x)                                                     # -d(Delta U)/d gamma
    assert meds[0] - meds[1] == pytest.approx(0.0673 * math.log(10) / dU(0.5 * (meds[0] + meds[1])), rel=0.1)


def test_oracle_switching_currents_of_the_papers_device_follow_the_adiabatic_theory():
    """PAPER.md:399 device through the paper's own normalisation (oracle/units.py), ramp rate 1e-4 per unit time (the experiment:
    1.24e-9), stochastic Heun, threshold at the next well.  The empirical CDF of 2500 oracle trajectories stays within the
    paper's 1.5 % of the theory plus the 99 % Kolmogorov band of the sample; the median within 1.5 %."""
    p = ou.library_parameters(250.0, 88e-15, 0.748e-6, 1.2)
    nu, n = 1e-4, 2500
    kw = dict(model="underdamped", scheme="heun", alpha=p["alpha"], temperature=p["temperature"], gamma0=0.0, nu=nu, phi0=0.0,
              threshold=2 * math.pi, dt=0.02)
    r = oracle.simulate(oracle.make_params(**kw), n, 42, 1.05 / nu)
    assert np.all(r["status"] == 0)
    g, cdf = sc.switching_cdf(p["alpha"], p["temperature"], nu)
    xs = np.sort(r["gamma"])
    emp = (np.arange(n) + 0.5) / n
    dev = np.max(np.abs(emp - np.interp(xs, g, cdf)))
    assert dev < 0.015 + 1.63 / math.sqrt(n), dev
    assert np.median(xs) / sc.quantile(g, cdf, 0.5) - 1 == pytest.approx(0.0, abs=0.015)
    assert xs.std() / sc.moments(g, cdf)[1] - 1 == pytest.approx(0.0, abs=0.08)
