"""Independent CPU pins for the fp32 pieces of the oracle (R14).

Nothing here calls an oracle function to produce its own expected value:

(a) normal_quad_f -- WHICH Philox word is the uniform, which the angle, and the order (cosA, sinA, cosB, sinB): the four
    words come from the pure-Python Philox of tests/ref_mp.py, the uniform is the one IEEE int->float rounding of the
    spec done by numpy, and Box-Muller is evaluated in 50-digit mpmath.  A swapped word or a swapped cos/sin is an O(1)
    error.
(b) run_f32 -- the Euler-Maruyama / overdamped / Heun branches: 64-step paths (nu != 0) against the 50-digit definition
    of tests/ref_mp.run driven by the mpmath normals of (a); and all 2^8 sign paths of injected +-1 normals per
    recurrence: escape indices against exact arithmetic.
(c) the status-2 rule R14 (phi_k NaN at some k before any crossing): which k and which outputs, fp64 and fp32.
"""
import itertools
import math

import numpy as np
import pytest
from mpmath import mp, mpf

import oracle
import ref_mp

TWO_PI = 2 * math.pi


def mp_normal_quad(seed, tid, block):
    """DESIGN.md 4.7 from the definition: pair A from words (o0, o1), pair B from (o2, o3); u = RN_f((float) o) * 2^-32
    + 2^-33 (the int->float conversion is the spec's one rounding; the fma is exact-scale), theta = 2 pi o / 2^32."""
    o = ref_mp.philox_block(seed, tid, block)
    out = []
    for h in range(2):
        of = float(np.float32(np.uint32(o[2 * h])))                     # IEEE round-to-nearest conversion, by numpy
        u = float(np.float32(of * 2.0**-32 + 2.0**-33))                 # single rounding of the exact sum (fmaf)
        theta = 2 * mp.pi * mpf(o[2 * h + 1]) / mpf(2) ** 32
        r = mp.sqrt(-2 * mp.log(mpf(u)))
        out += [r * mp.cos(theta), r * mp.sin(theta)]
    return out


def test_normal_quad_word_assignment_and_order():
    rng = np.random.default_rng(4)
    worst = 0.0
    for _ in range(300):
        seed, tid, b = (int(x) for x in rng.integers(0, 2**62, 3))
        got = oracle.normals_f32(seed, tid, b, 1).astype(np.float64)
        want = mp_normal_quad(seed, tid, b)
        for g, w in zip(got, want):
            err = abs(mpf(float(g)) - w)
            worst = max(worst, float(err) / max(1.0, abs(float(w))))
            assert err <= 2e-6 * max(1.0, abs(float(w))), (seed, tid, b, got, [float(x) for x in want])
    assert worst > 0.0                                                   # the comparison is not vacuous (fp32 rounds)
    # consecutive blocks of one stream: block index b0 + i, four normals each, in stream order
    got = oracle.normals_f32(7, 3, 2**32 - 1, 3).astype(np.float64)
    want = [float(x) for i in range(3) for x in mp_normal_quad(7, 3, 2**32 - 1 + i)]
    assert np.allclose(got, want, rtol=0, atol=3e-6)


def test_step_to_normal_assignment_fp32():
    # steps 4b+1 .. 4b+4 use (cosA, sinA, cosB, sinB) of block b: a mu = 0 walk exposes the normals as increments
    p = oracle.make_params(model="overdamped", scheme="em", precision="fp32", amp=0.0, gamma0=0.0, temperature=0.5,
                           phi0=0.0, threshold=1e9, dt=1.0)
    phi, _, _, _ = oracle.trace(p, 77, 5, 1e3, 13)
    want = [float(x) for b in range(3) for x in mp_normal_quad(77, 5, b)]
    assert np.allclose(np.diff(phi), want, rtol=0, atol=2e-5)            # partial sums are rounded to float each step


F32_CASES = [
    dict(model=0, scheme=0, alpha=0.0, temperature=0.03, amp=1.0, gamma0=0.7, nu=2e-3, phi0=0.77, v0=0.0, threshold=7.0, dt=0.02),
    dict(model=0, scheme=1, alpha=0.0, temperature=0.03, amp=1.0, gamma0=0.7, nu=2e-3, phi0=0.77, v0=0.0, threshold=7.0, dt=0.02),
    dict(model=1, scheme=0, alpha=0.05, temperature=0.005, amp=1.0, gamma0=0.5, nu=1e-3, phi0=0.52, v0=0.1, threshold=6.8, dt=0.05),
    dict(model=1, scheme=1, alpha=0.05, temperature=0.005, amp=1.0, gamma0=0.5, nu=1e-3, phi0=0.52, v0=0.1, threshold=6.8, dt=0.05),
]


@pytest.mark.parametrize("case", F32_CASES, ids=lambda c: f"m{c['model']}s{c['scheme']}")
def test_run_f32_branches_vs_definition(case):
    """Every recurrence of run_f32, ramp on (the Kahan clock feeds gamma), 64 Philox-driven steps: each state within a
    few float ulps of the 50-digit definition driven by the mpmath normals above."""
    nst = 64
    for seed, tid in [(4, 9), (11, 2**33 + 5)]:
        p = oracle.make_params(precision="fp32", **case)
        phi, v, st, ke = oracle.trace(p, seed, tid, 1e3, nst + 1)
        zs = [z for b in range(nst // 4) for z in mp_normal_quad(seed, tid, b)]
        kw = dict(case, phi0=float(np.float32(case["phi0"])), v0=float(np.float32(case["v0"])))
        _, _, states, _ = ref_mp.run(n_cap=10**6, normals=zs, max_steps=nst, **kw)
        assert ke > nst                                                    # no crossing inside the window
        for k, (ph_mp, v_mp) in enumerate(states):
            assert abs(float(ph_mp) - phi[k]) < 2e-6, (case, k, float(ph_mp), phi[k])
            if case["model"] == 1:
                assert abs(float(v_mp) - v[k]) < 2e-6, (case, k, float(v_mp), v[k])
        # teeth: the same comparison fails by far more than the bar if the ramp is dropped or the noise sign flipped
        _, _, wrong, _ = ref_mp.run(n_cap=10**6, normals=[-z for z in zs], max_steps=nst, **kw)
        assert abs(float(wrong[nst][0]) - phi[nst]) > 1e-4


ENUM_CASES = [
    dict(model=0, scheme=0, alpha=0.0, temperature=0.08, amp=1.0, gamma0=0.8, nu=0.02, phi0=0.9, v0=0.0, threshold=1.3, dt=0.1),
    dict(model=0, scheme=1, alpha=0.0, temperature=0.08, amp=1.0, gamma0=0.8, nu=0.02, phi0=0.9, v0=0.0, threshold=1.3, dt=0.1),
    dict(model=1, scheme=0, alpha=0.3, temperature=0.8, amp=1.0, gamma0=0.9, nu=0.01, phi0=1.0, v0=0.2, threshold=1.8, dt=0.25),
    dict(model=1, scheme=1, alpha=0.3, temperature=0.8, amp=1.0, gamma0=0.9, nu=0.01, phi0=1.0, v0=0.2, threshold=1.8, dt=0.25),
]


@pytest.mark.parametrize("case", ENUM_CASES, ids=lambda c: f"m{c['model']}s{c['scheme']}")
def test_enumerate_sign_paths_fp32(case):
    """All 2^8 paths of injected +-1 normals through the fp32 integrator: escape index and status equal exact arithmetic
    wherever the exact path stays clear of the threshold by more than fp32 rounding can move it; states within 1e-5."""
    n = 8
    p = oracle.make_params(precision="fp32", **case)
    t_max = n * case["dt"]
    assert oracle.n_cap(p, t_max) == n
    compared = escaped = 0
    for signs in itertools.product((-1.0, 1.0), repeat=n):
        phi, v, st, ke = oracle.trace(p, 0, 0, t_max, n + 1, normals=signs)
        st_mp, k_mp, states, margin = ref_mp.run(n_cap=n, normals=signs, **case)
        if margin < 1e-4:
            continue                                                       # borderline in single precision: not a pin
        compared += 1
        escaped += st_mp == 0
        assert (st, ke) == (st_mp, k_mp), (signs, st, ke, st_mp, k_mp)
        for k, (ph_mp, v_mp) in enumerate(states):
            assert abs(float(ph_mp) - phi[k]) < 1e-5
            if case["model"] == 1:
                assert abs(float(v_mp) - v[k]) < 1e-5
    assert compared > 200 and 20 < escaped < compared - 20


@pytest.mark.parametrize("precision,big,dt", [("fp64", 1e300, 1e300), ("fp32", 1e40, 1e38)])
def test_status2_rule_which_step_and_outputs(precision, big, dt):
    """R14: status 2 <=> phi_k is NaN at some k <= n_cap with no crossing at any earlier step; k_end is that k and
    out_fpt = out_gamma = NaN.  sigma = sqrt(2 T dt) overflows to +inf in the working precision (dt itself stays finite
    there, so the drift term f*dt = 0*dt is 0 at phi = 0), and the first kick decides:
      z1 > 0: phi_1 = +inf >= threshold -> escaped at k = 1 (a crossing wins over everything after it);
      z1 < 0: phi_1 = -inf (not NaN, not a crossing); phi_2 needs sin(-inf) = NaN -> status 2 at k = 2;
      z1 = 0: inf * 0 = NaN -> status 2 at k = 1."""
    kw = dict(model="overdamped", scheme="em", precision=precision, temperature=big, amp=1.0, gamma0=0.0, nu=0.0, phi0=0.0,
              threshold=1e10, dt=dt)
    p = oracle.make_params(**kw)
    t_max = 100 * dt
    phi, _, st, ke = oracle.trace(p, 0, 0, t_max, 4, normals=[-1.0, 1.0, 1.0])
    assert (st, ke) == (2, 2) and phi[0] == 0.0 and phi[1] == -np.inf and np.isnan(phi[2]) and np.isnan(phi[3])
    phi, _, st, ke = oracle.trace(p, 0, 0, t_max, 4, normals=[1.0, -1.0])
    assert (st, ke) == (0, 1) and phi[1] == np.inf
    phi, _, st, ke = oracle.trace(p, 0, 0, t_max, 4, normals=[0.0, 1.0])
    assert (st, ke) == (2, 1) and np.isnan(phi[1])
    # through the simulate entry point with the Philox stream: the sign of the first normal (cos branch of block 0,
    # from the pure-Python Philox + mpmath) decides status, step and outputs of every id
    n = 64
    r = oracle.simulate(p, n, 3, t_max)
    for i in range(n):
        z1 = mp_normal_quad(3, i, 0)[0] if precision == "fp32" else ref_mp.normal_pair(3, i, 0)[0]
        assert abs(z1) > 1e-6
        if z1 > 0:
            assert (r["status"][i], r["k"][i]) == (0, 1) and r["fpt"][i] == 1.0 * dt and r["gamma"][i] == 0.0
        else:
            assert (r["status"][i], r["k"][i]) == (2, 2) and np.isnan(r["fpt"][i]) and np.isnan(r["gamma"][i])
    assert 10 < int(np.sum(r["status"] == 2)) < n - 10
