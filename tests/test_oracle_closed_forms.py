"""Pins P3, P4, P5: the oracle's integrator against closed forms.

P3  drifted Brownian motion to a level: inverse-Gaussian first-passage law (config 1), with the discrete-monitoring
    (Broadie-Glasserman-Kou) barrier shift, and Wald's identity which holds exactly for the sampled walk.
P4  zero noise, gamma > 1: overdamped passage over 2*pi takes exactly 2*pi/sqrt(gamma^2-1); underdamped case against
    scipy's ODE solver; gamma < 1 with zero noise never escapes (censored, fpt = -1).
P5  overdamped washboard at finite T: exact mean first-passage time by quadrature of the textbook double integral, and
    Kramers/Arrhenius scaling of ln(tau) against 1/T (Eqs. 12-14).
"""
import math

import numpy as np
import pytest
from scipy import integrate, stats

import oracle
from ref_mp import read_golden

TWO_PI = 2 * math.pi


# ---------------------------------------------------------------- P3 -------------------------------------------
def ig_cdf(t, a, mu, D):
    t = np.asarray(t, dtype=np.float64)
    s = np.sqrt(2 * D * t)
    return stats.norm.cdf((mu * t - a) / s) + np.exp(mu * a / D) * stats.norm.cdf(-(mu * t + a) / s)


@pytest.fixture(scope="module")
def config1():
    p = oracle.make_params(model="overdamped", scheme="em", amp=0.0, gamma0=1.0, temperature=0.1, phi0=0.0,
                           threshold=1.0, dt=1e-3)
    return oracle.simulate(p, 10_000, 1, 100.0, with_state=True)


def test_config1_inverse_gaussian(config1):
    r = config1
    a, mu, D, dt = 1.0, 1.0, 0.1, 1e-3
    assert np.all(r["status"] == 0)                         # none reaches the 1e5-step cap
    assert r["k"].max() < 20_000
    fpt = r["fpt"]
    assert np.array_equal(fpt, r["k"].astype(np.float64) * dt)
    a_eff = a + 0.5826 * math.sqrt(2 * D * dt)               # BGK continuity correction: -zeta(1/2)/sqrt(2 pi) = 0.5826
    n = fpt.size
    assert abs(fpt.mean() - a_eff / mu) < 4 * math.sqrt(2 * D * a / mu**3 / n)
    assert abs(fpt.var() - 2 * D * a_eff / mu**3) < 0.02     # IG variance 0.2017; s.e. of the sample variance ~0.005
    ks = stats.kstest(fpt, lambda t: ig_cdf(t, a_eff, mu, D))
    assert ks.pvalue > 0.01
    # the uncorrected law is measurably worse at this dt (guards against testing with too loose a bar)
    assert stats.kstest(fpt, lambda t: ig_cdf(t, a, mu, D)).statistic > ks.statistic


def test_config1_wald_identity_and_overshoot(config1):
    r = config1
    mu, D, dt = 1.0, 0.1, 1e-3
    resid = mu * r["fpt"] - r["phi_end"]                     # E[mu*tau - x(tau)] = 0 exactly (optional stopping)
    assert abs(resid.mean()) < 4 * resid.std() / math.sqrt(resid.size)
    assert abs(resid.std() - math.sqrt(2 * D * 1.0)) < 0.02  # Var = 2 D E[tau]
    over = r["phi_end"] - 1.0
    assert np.all(over >= 0)
    assert abs(over.mean() - 0.5826 * math.sqrt(2 * D * dt)) < 6e-4


def test_driftless_cap_and_sentinels():
    # mu = 0 far below the level with a short cap: nobody escapes -> all censored with the paper's sentinel
    p = oracle.make_params(model="overdamped", scheme="em", amp=0.0, gamma0=0.0, temperature=0.1, phi0=0.0,
                           threshold=50.0, dt=1e-3)
    r = oracle.simulate(p, 64, 3, 0.2)
    assert np.all(r["status"] == 1) and np.all(r["fpt"] == -1.0) and np.all(r["k"] == 200)
    # threshold at the initial point -> escape at k = 0
    p = oracle.make_params(model="overdamped", scheme="em", amp=0.0, gamma0=1.0, temperature=0.1, phi0=1.0,
                           threshold=1.0, dt=1e-3)
    r = oracle.simulate(p, 4, 3, 1.0)
    assert np.all(r["status"] == 0) and np.all(r["fpt"] == 0.0) and np.all(r["k"] == 0)


# ---------------------------------------------------------------- P4 -------------------------------------------
def test_deterministic_overdamped():
    for row in read_golden("deterministic.txt"):
        if row[0] != "od":
            continue
        scheme, gamma, dt, k_want = row[1], float(row[2]), float(row[3]), int(row[4])
        p = oracle.make_params(model="overdamped", scheme=scheme, amp=1.0, gamma0=gamma, temperature=0.0, phi0=0.0,
                               threshold=TWO_PI, dt=dt)
        r = oracle.simulate(p, 3, 99, 100.0)
        exact = TWO_PI / math.sqrt(gamma**2 - 1)
        assert np.all(r["status"] == 0)
        assert np.all(r["k"] == r["k"][0])                    # no noise: every id identical
        assert int(r["k"][0]) == k_want
        tol = 4 * dt if scheme == "em" else 1.5 * dt          # EM is O(dt) accurate, Heun O(dt^2) + the grid
        assert abs(r["fpt"][0] - exact) < tol
    # any phi0: the passage time over one period does not depend on the starting phase
    p = oracle.make_params(model="overdamped", scheme="heun", amp=1.0, gamma0=1.5, temperature=0.0, phi0=0.7,
                           threshold=0.7 + TWO_PI, dt=1e-3)
    r = oracle.simulate(p, 1, 1, 100.0)
    assert abs(r["fpt"][0] - TWO_PI / math.sqrt(1.25)) < 2e-3


def test_deterministic_underdamped_vs_ode_solver():
    rows = {r[1] if r[0] == "ud" else r[0]: r for r in read_golden("deterministic.txt") if r[0].startswith("ud")}
    alpha, gamma = 0.1, 1.2
    ev = lambda t, y: y[0] - TWO_PI
    ev.terminal = True
    sol = integrate.solve_ivp(lambda t, y: [y[1], gamma - math.sin(y[0]) - alpha * y[1]], [0, 50], [0.0, 0.0],
                              events=ev, rtol=1e-12, atol=1e-14)
    t_exact = sol.t_events[0][0]
    assert abs(t_exact - float(rows["ud_event_time"][1])) < 1e-5
    for scheme in ("em", "heun"):
        p = oracle.make_params(model="underdamped", scheme=scheme, alpha=alpha, amp=1.0, gamma0=gamma, temperature=0.0,
                               phi0=0.0, v0=0.0, threshold=TWO_PI, dt=0.01)
        r = oracle.simulate(p, 1, 5, 100.0)
        assert int(r["k"][0]) == int(rows[scheme][2])
        assert abs(r["fpt"][0] - t_exact) < (0.03 if scheme == "em" else 0.011)
    # Heun converges at second order: halving dt brings the grid time within dt of the event
    p = oracle.make_params(model="underdamped", scheme="heun", alpha=alpha, amp=1.0, gamma0=gamma, temperature=0.0,
                           threshold=TWO_PI, dt=0.001)
    assert 0 <= oracle.simulate(p, 1, 5, 100.0)["fpt"][0] - t_exact < 0.00101


def test_zero_noise_below_critical_bias_never_escapes():
    phi0 = math.asin(0.9)
    for model, scheme in (("overdamped", "em"), ("underdamped", "heun"), ("underdamped", "em"), ("overdamped", "heun")):
        p = oracle.make_params(model=model, scheme=scheme, alpha=0.1, amp=1.0, gamma0=0.9, temperature=0.0, phi0=phi0,
                               threshold=phi0 + TWO_PI, dt=0.01)
        r = oracle.simulate(p, 2, 1, 50.0)
        assert np.all(r["status"] == 1) and np.all(r["fpt"] == -1.0) and np.all(r["k"] == 5000)
        assert np.allclose(r["gamma"], 0.9)


def test_deterministic_ramp_gamma_at_escape():
    # zero noise, slow overdamped ramp from gamma = 0: the phase follows asin(gamma) and runs away just after gamma = 1
    # (paper: "the bias current is increased from zero to 1"; Alg. 3 stores gamma_k at the crossing)
    nu, dt = 1e-3, 0.01
    p = oracle.make_params(model="overdamped", scheme="heun", amp=1.0, gamma0=0.0, nu=nu, temperature=0.0, phi0=0.0,
                           threshold=TWO_PI, dt=dt)
    r = oracle.simulate(p, 1, 1, 2000.0)
    assert r["status"][0] == 0
    g = r["gamma"][0]
    assert abs(g - nu * r["fpt"][0]) < 1e-12
    assert 1.0 < g < 1.06                                   # delay past gamma=1 scales as nu^(2/3): ~2.9*nu^(2/3)=0.029..0.05


# ---------------------------------------------------------------- P5 -------------------------------------------
def mfpt_quadrature(gamma, T):
    """tau = (1/T) int_{phi0}^{b} dy e^{U(y)/T} int_{-inf}^{y} dz e^{-U(z)/T},  U = -cos(phi) - gamma*phi."""
    phi0 = math.asin(gamma)
    b = phi0 + TWO_PI
    U = lambda x: -math.cos(x) - gamma * x

    def inner(y):
        val, _ = integrate.quad(lambda z: math.exp((U(y) - U(z)) / T), y - 60.0, y, limit=400, epsabs=0, epsrel=1e-10)
        return val

    val, _ = integrate.quad(inner, phi0, b, limit=400, epsabs=0, epsrel=1e-8)
    return val / T


@pytest.fixture(scope="module")
def od_escape():
    gamma, dt, n = 0.7, 5e-3, 4000
    phi0 = math.asin(gamma)
    out = {}
    for T in (0.2, 0.15, 0.1):
        p = oracle.make_params(model="overdamped", scheme="em", amp=1.0, gamma0=gamma, temperature=T, phi0=phi0,
                               threshold=phi0 + TWO_PI, dt=dt)
        out[T] = oracle.simulate(p, n, 5, 5e5)
    return out


def test_overdamped_mfpt_vs_quadrature(od_escape):
    table = {float(r[0]): float(r[1]) for r in read_golden("mfpt_overdamped.txt")}
    for T, r in od_escape.items():
        tau_q = mfpt_quadrature(0.7, T)
        assert abs(tau_q - table[T]) < 2e-3 * table[T]        # the stored table is the same integral
        assert np.all(r["status"] == 0)
        fpt = r["fpt"]
        sem = fpt.std() / math.sqrt(fpt.size)
        assert abs(fpt.mean() - tau_q) < 3 * sem + 0.01 * tau_q, (T, fpt.mean(), tau_q)
        assert 0.85 < fpt.std() / fpt.mean() < 1.05           # near-exponential law (rare-event regime)


def test_kramers_arrhenius_slope(od_escape):
    gamma = 0.7
    dU = 2 * (math.sqrt(1 - gamma**2) - gamma * math.acos(gamma))     # washboard barrier, = 0.314727
    assert abs(dU - 0.314727) < 1e-6
    Ts = sorted(od_escape)
    lt = [math.log(od_escape[T]["fpt"].mean()) for T in Ts]
    slope = (lt[0] - lt[-1]) / (1 / Ts[0] - 1 / Ts[-1])                # d ln(tau) / d(1/T)  (Eq. 12)
    lq = [math.log(mfpt_quadrature(gamma, T)) for T in (Ts[0], Ts[-1])]
    slope_q = (lq[0] - lq[1]) / (1 / Ts[0] - 1 / Ts[-1])
    assert abs(slope - slope_q) < 0.012                                # statistical: 2 means of 4000, CV~1, over d(1/T)=5
    assert abs(slope_q - dU) < 0.1 * dU                                # prefactor correction at these T (table ratio 1.22->1.14)
    # Kramers prefactor: tau -> 2*pi/sqrt(1-gamma^2) * exp(dU/T) from above as T decreases
    kr = lambda T: TWO_PI / math.sqrt(1 - gamma**2) * math.exp(dU / T)
    ratios = [mfpt_quadrature(gamma, T) / kr(T) for T in (0.2, 0.1, 0.06)]
    assert ratios[0] > ratios[1] > ratios[2] > 1.0 and ratios[2] < 1.09
