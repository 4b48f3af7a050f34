"""Pins of the paper-faithful variant, scheme 2 = Alg. 1 / Alg. 3 AS PRINTED (R17):
Euler, the bias gamma_k = gamma0 + dgamma*k taken BEFORE the step (Alg. 3 line 13 precedes lines 14-15; the textbook scheme 0
uses gamma_{k-1}), the strict test phi_k > th (Alg. 1 line 12, Alg. 3 line 16; schemes 0 and 1 use >=), and the paper's own
threshold th = pi - phi0 (Alg. 1 line 5) passed as the parameter.

What a plausible mistake would break: gamma_{k-1} instead of gamma_k (the enumeration with a large ramp step, the closed form
of the deterministic ramp), >= instead of > (the path that lands exactly on the threshold), new-state instead of old-state
updates (the enumeration: every state against 50-digit arithmetic)."""
import itertools
import math

import numpy as np
import pytest

import oracle
import ref_mp

CASES = [
    dict(model=1, scheme=2, alpha=0.3, temperature=0.8, amp=1.0, gamma0=0.9, nu=0.4, phi0=1.0, v0=0.2, threshold=1.8, dt=0.25),
    dict(model=1, scheme=2, alpha=0.3, temperature=0.8, amp=1.0, gamma0=0.9, nu=0.0, phi0=1.0, v0=0.2, threshold=1.8, dt=0.25),
    dict(model=0, scheme=2, alpha=0.0, temperature=0.08, amp=1.0, gamma0=0.8, nu=0.5, phi0=0.9, v0=0.0, threshold=1.3, dt=0.1),
]


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("case", CASES, ids=lambda c: f"m{c['model']}nu{c['nu']}")
def test_enumerate_sign_paths_of_the_paper_scheme(case, precision):
    """All 2^10 sign paths: every state and every escape index against the printed recurrences in 50-digit arithmetic.  The
    ramp step is large (nu*dt = 0.1 / 0.05), so using gamma_{k-1} for gamma_k moves states by ~1e-2: far above the bars."""
    n = 10
    p = oracle.make_params(precision=precision, **case)
    t_max = n * case["dt"]
    tol = 4e-16 if precision == "fp64" else 3e-7
    n_esc = 0
    differs_from_textbook = 0
    for signs in itertools.product((-1.0, 1.0), repeat=n):
        phi, v, st, ke = oracle.trace(p, 0, 0, t_max, n + 1, normals=signs)
        st_mp, k_mp, states, margin = ref_mp.run(n_cap=n, normals=signs, **case)
        assert margin > 1e-5
        assert (st, ke) == (st_mp, k_mp)
        for k, (ph_mp, v_mp) in enumerate(states):
            assert abs(float(ph_mp) - phi[k]) <= tol * (k + 1) * max(1.0, abs(phi[k]))
            if case["model"] == 1:
                assert abs(float(v_mp) - v[k]) <= tol * (k + 1) * max(1.0, abs(v[k]))
        n_esc += st == 0
        st0, k0, _, _ = ref_mp.run(n_cap=n, normals=signs, **dict(case, scheme=0))
        differs_from_textbook += (st0, k0) != (st_mp, k_mp)
    assert 50 < n_esc < 2**n - 50
    if case["nu"] != 0.0:
        assert differs_from_textbook > 0          # the ordering of the bias update is visible in the escape indices


def test_strict_comparison_on_a_path_that_lands_on_the_threshold():
    """Noise off, no sine, mu = 0.5, dt = 0.5: phi_k = 0.25 k exactly in binary.  th = 1: '>=' (scheme 0) escapes at k = 4,
    the paper's '>' (scheme 2) at k = 5.  Same for the initial state: phi0 = th is an escape at k = 0 only with '>='."""
    base = dict(model="overdamped", alpha=0.0, temperature=0.0, amp=0.0, gamma0=0.5, nu=0.0, phi0=0.0, threshold=1.0, dt=0.5)
    for precision in ("fp64", "fp32"):
        r0 = oracle.simulate(oracle.make_params(scheme="em", precision=precision, **base), 3, 1, 10.0)
        r2 = oracle.simulate(oracle.make_params(scheme="paper", precision=precision, **base), 3, 1, 10.0)
        assert list(r0["k"]) == [4, 4, 4] and list(r2["k"]) == [5, 5, 5]
        assert list(r0["fpt"]) == [2.0] * 3 and list(r2["fpt"]) == [2.5] * 3
        at = dict(base, phi0=1.0)
        assert list(oracle.simulate(oracle.make_params(scheme="em", precision=precision, **at), 2, 1, 10.0)["k"]) == [0, 0]
        assert list(oracle.simulate(oracle.make_params(scheme="paper", precision=precision, **at), 2, 1, 10.0)["k"]) == [1, 1]


def test_deterministic_ramp_closed_form_tells_gamma_k_from_gamma_k_minus_1():
    """No sine, no noise, overdamped: phi_n = dt * sum_{k=1..n} gamma_j with j = k (paper) or k - 1 (textbook), i.e.
    phi_n = dt*(n*gamma0 + dgamma*n(n+1)/2) against dt*(n*gamma0 + dgamma*n(n-1)/2)."""
    g0, nu, dt, n = 0.125, 0.5, 0.25, 12                    # all exactly representable; dgamma = 0.125
    for scheme, shift in (("paper", +1), ("em", -1)):
        p = oracle.make_params(model="overdamped", scheme=scheme, temperature=0.0, amp=0.0, gamma0=g0, nu=nu, phi0=0.0,
                               threshold=1e9, dt=dt)
        phi, _, st, ke = oracle.trace(p, 0, 0, n * dt, n + 1)
        for k in range(n + 1):
            assert phi[k] == dt * (k * g0 + nu * dt * k * (k + shift) / 2)
        assert st == 1 and ke == n


def test_paper_threshold_escape_comes_before_the_next_well():
    """Alg. 1 line 5: th = pi - phi0, the barrier top; configs use phi0 + 2 pi, the next well (the two differ by the
    slide-down time, mean 5067 against 5690 steps on config 2 in an independent numpy probe).  Same noise, same path: the
    barrier-top crossing of every trajectory comes first, and the mean is near the probe's."""
    phi0 = math.asin(0.9)
    base = dict(model="underdamped", alpha=0.1, temperature=0.05, gamma0=0.9, phi0=phi0, dt=0.01)
    n = 4000
    top = oracle.simulate(oracle.make_params(scheme="paper", threshold=math.pi - phi0, **base), n, 2, 1e4)
    well = oracle.simulate(oracle.make_params(scheme="paper", threshold=phi0 + 2 * math.pi, **base), n, 2, 1e4)
    assert np.all(top["status"] == 0) and np.all(well["status"] == 0)
    assert np.all(top["k"] < well["k"])
    slide = (well["k"] - top["k"]).astype(float)
    assert 350 < slide.mean() < 900                         # 5690 - 5067 = 623 steps in the probe
    assert abs(top["k"].mean() - 5067) < 5 * 4300 / math.sqrt(n) + 120
    # with nu = 0 the ordering of the bias update is immaterial: scheme 2 differs from scheme 0 only where a state equals th
    em = oracle.simulate(oracle.make_params(scheme="em", threshold=phi0 + 2 * math.pi, **base), n, 2, 1e4)
    assert np.array_equal(em["k"], well["k"])


def test_switching_current_of_the_paper_scheme_is_one_increment_ahead():
    """Alg. 3 with a ramp: the paper's ordering sees the bias one increment (dgamma) early, so its switching currents are
    statistically indistinguishable from the textbook ordering at dgamma = 2e-5 ('differs by dgamma, far below
    any tolerance') -- but the paths are not identical."""
    base = dict(model="underdamped", alpha=0.1, temperature=0.01, gamma0=0.0, nu=1e-3, phi0=0.0, threshold=math.pi, dt=0.02)
    n = 600
    a = oracle.simulate(oracle.make_params(scheme="paper", **base), n, 3, 1050.0)
    b = oracle.simulate(oracle.make_params(scheme="em", **base), n, 3, 1050.0)
    assert np.all(a["status"] == 0) and np.all(b["status"] == 0)
    assert not np.array_equal(a["k"], b["k"])
    assert abs(a["gamma"].mean() - b["gamma"].mean()) < 4 * a["gamma"].std() / math.sqrt(n)
    assert 0.9 < a["gamma"].mean() < 1.0
    assert np.allclose(a["gamma"], 2e-5 * a["k"].astype(float), rtol=0, atol=1e-15)      # Gamma_e = gamma_k at the crossing step
