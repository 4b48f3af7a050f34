"""Pins P6 and P10: brute force on tiny inputs and whole-path recomputation in 50-digit arithmetic.

(i)  inject normals from {-1,+1}: all 2^n paths, n = 10, for each of the four recurrences; every state of every path and
     every escape index must agree with the definitions evaluated in mpmath (tests/ref_mp.py).
(ii) the real Philox -> Box-Muller -> step chain for a few steps, recomputed in mpmath: states to a few ulp.
(iii) the worked examples of SURVEY.md P10 (tests/golden/worked_examples.txt): escape indices of whole runs.
"""
import itertools
import math

import numpy as np
import pytest

import oracle
import ref_mp

CASES = [
    # model, scheme, params chosen so that a fair share of the 1024 sign paths cross within 10 steps
    dict(model=0, scheme=0, alpha=0.0, temperature=0.08, amp=1.0, gamma0=0.8, nu=0.02, phi0=0.9, v0=0.0, threshold=1.3, dt=0.1),
    dict(model=0, scheme=1, alpha=0.0, temperature=0.08, amp=1.0, gamma0=0.8, nu=0.02, phi0=0.9, v0=0.0, threshold=1.3, dt=0.1),
    dict(model=1, scheme=0, alpha=0.3, temperature=0.8, amp=1.0, gamma0=0.9, nu=0.01, phi0=1.0, v0=0.2, threshold=1.8, dt=0.25),
    dict(model=1, scheme=1, alpha=0.3, temperature=0.8, amp=1.0, gamma0=0.9, nu=0.01, phi0=1.0, v0=0.2, threshold=1.8, dt=0.25),
    dict(model=0, scheme=0, alpha=0.0, temperature=0.05, amp=0.0, gamma0=0.5, nu=0.0, phi0=0.0, v0=0.0, threshold=0.63, dt=0.1),
]


@pytest.mark.parametrize("case", CASES, ids=lambda c: f"m{c['model']}s{c['scheme']}a{c['amp']}")
def test_enumerate_sign_paths(case):
    n = 10
    p = oracle.make_params(**case)
    t_max = n * case["dt"]
    assert oracle.n_cap(p, t_max) == n
    hist_oracle = np.zeros(n + 2, int)
    hist_exact = np.zeros(n + 2, int)
    for signs in itertools.product((-1.0, 1.0), repeat=n):
        phi, v, st, ke = oracle.trace(p, 0, 0, t_max, n + 1, normals=signs)
        st_mp, k_mp, states, margin = ref_mp.run(n_cap=n, normals=signs, **case)
        assert margin > 1e-9                                   # the enumeration has no borderline crossing
        assert (st, ke) == (st_mp, k_mp)
        for k, (ph_mp, v_mp) in enumerate(states):
            assert abs(float(ph_mp) - phi[k]) <= 4e-16 * (k + 1) * max(1.0, abs(phi[k]))
            if case["model"] == 1:
                assert abs(float(v_mp) - v[k]) <= 4e-16 * (k + 1) * max(1.0, abs(v[k]))
        hist_oracle[ke if st == 0 else n + 1] += 1
        hist_exact[k_mp if st_mp == 0 else n + 1] += 1
    assert np.array_equal(hist_oracle, hist_exact)
    assert 50 < hist_exact[:n + 1].sum() < 2**n - 50            # both outcomes well represented


def test_short_philox_paths_vs_mpmath():
    phi0 = math.asin(0.9)
    cases = [
        (dict(model=1, scheme=1, alpha=0.1, temperature=0.05, amp=1.0, gamma0=0.9, nu=0.0, phi0=phi0, v0=0.0,
              threshold=phi0 + 2 * math.pi, dt=0.01), 2, 0),
        (dict(model=1, scheme=0, alpha=0.1, temperature=0.05, amp=1.0, gamma0=0.9, nu=1e-3, phi0=phi0, v0=0.0,
              threshold=phi0 + 2 * math.pi, dt=0.01), 2, 12345),
        (dict(model=0, scheme=1, alpha=0.0, temperature=0.03, amp=1.0, gamma0=0.7, nu=1e-4, phi0=0.77, v0=0.0,
              threshold=7.0, dt=5e-3), 5, 2**40 + 7),
        (dict(model=0, scheme=0, alpha=0.0, temperature=0.1, amp=0.0, gamma0=1.0, nu=0.0, phi0=0.0, v0=0.0,
              threshold=1.0, dt=1e-3), 1, 0),
    ]
    for case, seed, tid in cases:
        p = oracle.make_params(**case)
        nst = 40
        phi, v, st, ke = oracle.trace(p, seed, tid, 1e3, nst + 1)
        _, _, states, _ = ref_mp.run(n_cap=10**6, seed=seed, tid=tid, max_steps=nst, **case)
        for k, (ph_mp, v_mp) in enumerate(states):
            assert abs(float(ph_mp) - phi[k]) < 5e-15, (case, k)
            if case["model"] == 1:
                assert abs(float(v_mp) - v[k]) < 5e-15, (case, k)


def golden():
    return {r[0]: r[1:] for r in ref_mp.read_golden("worked_examples.txt")}


def test_worked_examples_config1():
    g = golden()
    p = oracle.make_params(model="overdamped", scheme="em", amp=0.0, gamma0=1.0, temperature=0.1, phi0=0.0,
                           threshold=1.0, dt=1e-3)
    r = oracle.simulate(p, 8, 1, 100.0)
    assert [int(k) for k in r["k"]] == [int(x) for x in g["c1_kesc"]]
    phi, _, _, _ = oracle.trace(p, 1, 0, 100.0, 4)
    assert np.allclose(phi[1:4], [float(x) for x in g["c1_path_id0"]], rtol=0, atol=1e-15)
    # and an independent 50-digit run of id 4 (the shortest) gives the same index with a wide margin
    st, k, _, margin = ref_mp.run(0, 0, 0, 0.1, 0.0, 1.0, 0.0, 0.0, 0.0, 1.0, 1e-3, 10**5, seed=1, tid=4)
    assert (st, k) == (0, int(g["c1_kesc"][4]))


def test_worked_examples_config2():
    g = golden()
    phi0 = math.asin(0.9)
    p = oracle.make_params(model="underdamped", scheme="heun", alpha=0.1, temperature=0.05, gamma0=0.9, phi0=phi0,
                           threshold=phi0 + 2 * math.pi, dt=0.01)
    r = oracle.simulate(p, 4, 2, 1e4)
    assert [int(k) for k in r["k"]] == [int(x) for x in g["c2_kesc"]]
    phi, _, _, _ = oracle.trace(p, 2, 0, 1e4, 4)
    assert np.allclose(phi[1:4], [float(x) for x in g["c2_path_id0"]], rtol=0, atol=1e-15)


def test_worked_examples_config5_family_and_fast_ramp():
    g = golden()
    phi0 = math.asin(0.7)
    p = oracle.make_params(model="overdamped", scheme="em", temperature=0.2, gamma0=0.7, phi0=phi0,
                           threshold=phi0 + 2 * math.pi, dt=5e-3)
    assert [int(k) for k in oracle.simulate(p, 4, 5, 5e5)["k"]] == [int(x) for x in g["c5T02_kesc"]]
    p = oracle.make_params(model="underdamped", scheme="heun", alpha=0.1, temperature=0.01, gamma0=0.0, nu=1e-3,
                           threshold=2 * math.pi, dt=0.02)
    r = oracle.simulate(p, 2, 3, 1.05e3)
    assert [int(k) for k in r["k"]] == [int(x) for x in g["c3fast_kesc"]]
    assert np.allclose(r["gamma"], [float(x) for x in g["c3fast_gamma"]], rtol=0, atol=1e-12)
    assert np.allclose(r["fpt"], r["k"].astype(float) * 0.02)
