"""Pin P7 -- the noisy underdamped path (configs 2-4) has no closed form; it is pinned statistically:
equipartition in a deep well, the Smoluchowski (large damping) limit against the exact overdamped MFPT, agreement of
Euler and Heun as dt -> 0, and an independent numpy sample of the ramped escape (tests/golden/ramp_numpy_sample.txt).
Plus the fp32 + Kahan-time variant (O10) against the fp64 path."""
import math

import numpy as np
from scipy import stats

import oracle
from ref_mp import read_golden

TWO_PI = 2 * math.pi


def test_equipartition_in_a_deep_well():
    # gamma = 0, T << barrier 2: the phase stays in the well and <v^2> = T, <(phi)^2> ~ T (harmonic, amp = 1)
    T, alpha = 0.05, 0.5
    n = 400_000
    for scheme, tol in (("heun", 0.08), ("em", 0.12)):
        p = oracle.make_params(model="underdamped", scheme=scheme, alpha=alpha, temperature=T, gamma0=0.0, phi0=0.0,
                               v0=0.0, threshold=100.0, dt=0.02)
        v2, x2 = [], []
        for tid in range(4):
            phi, v, st, ke = oracle.trace(p, 31, tid, (n - 1) * 0.02, n)
            assert st == 1 or ke >= n - 1
            v2.append(np.mean(v[2000:] ** 2)); x2.append(np.mean(phi[2000:] ** 2))
        assert abs(np.mean(v2) / T - 1) < tol, (scheme, np.mean(v2))
        assert abs(np.mean(x2) / T - 1) < 0.15, (scheme, np.mean(x2))   # anharmonic correction ~ +T/4... small


def test_smoluchowski_limit():
    # alpha >> 1: MFPT_UD(alpha) -> alpha * tau_OD (time rescaling of the overdamped equation), O(1/alpha^2) corrections
    table = {float(r[0]): float(r[1]) for r in read_golden("mfpt_overdamped.txt")}
    alpha, T, gamma = 10.0, 0.2, 0.7
    phi0 = math.asin(gamma)
    p = oracle.make_params(model="underdamped", scheme="heun", alpha=alpha, temperature=T, gamma0=gamma, phi0=phi0,
                           v0=0.0, threshold=phi0 + TWO_PI, dt=0.02)
    r = oracle.simulate(p, 3000, 41, 1e6)
    assert np.all(r["status"] == 0)
    m, sem = r["fpt"].mean(), r["fpt"].std() / math.sqrt(3000)
    assert abs(m - alpha * table[T]) < 3 * sem + 0.03 * alpha * table[T], (m, alpha * table[T])


def test_euler_and_heun_agree_as_dt_shrinks():
    phi0 = math.asin(0.9)
    base = dict(model="underdamped", alpha=0.1, temperature=0.05, gamma0=0.9, phi0=phi0, v0=0.0, threshold=phi0 + TWO_PI)
    n = 6000
    means = {}
    for scheme, dt, seed in (("heun", 0.01, 2), ("heun", 0.005, 102), ("em", 0.0025, 202)):
        r = oracle.simulate(oracle.make_params(scheme=scheme, dt=dt, **base), n, seed, 1e4)
        assert np.all(r["status"] == 0)
        means[(scheme, dt)] = (r["fpt"].mean(), r["fpt"].std() / math.sqrt(n), r["fpt"])
    # config 2's mean is ~56.9 time units (5690 steps at dt=0.01) -- SURVEY.md P7
    assert abs(means[("heun", 0.01)][0] - 56.9) < 3.0
    a, b, c = means[("heun", 0.01)], means[("heun", 0.005)], means[("em", 0.0025)]
    assert abs(a[0] - b[0]) < 4 * math.hypot(a[1], b[1])
    assert abs(a[0] - c[0]) < 4 * math.hypot(a[1], c[1]) + 0.02 * a[0]
    assert stats.ks_2samp(a[2], b[2]).pvalue > 0.01


def test_ramped_escape_vs_independent_numpy_sample():
    g = {r[0]: float(r[1]) for r in read_golden("ramp_numpy_sample.txt")}
    n = 1000
    p = oracle.make_params(model="underdamped", scheme="heun", alpha=0.1, temperature=0.01, gamma0=0.0, nu=1e-4,
                           phi0=0.0, v0=0.0, threshold=TWO_PI, dt=0.02)
    r = oracle.simulate(p, n, 3, 1.05e4)
    assert np.all(r["status"] == 0)
    gs = r["gamma"]
    assert np.allclose(gs, 1e-4 * r["fpt"], rtol=1e-12)
    sem = math.hypot(g["mean_stderr"], g["std_gamma_sw"] / math.sqrt(n))
    assert abs(gs.mean() - g["mean_gamma_sw"]) < 3 * sem
    assert abs(gs.std() / g["std_gamma_sw"] - 1) < 0.12
    q = np.quantile(gs, [0.01, 0.5, 0.99])
    assert abs(q[1] - g["q50"]) < 0.003 and abs(q[0] - g["q01"]) < 0.012 and abs(q[2] - g["q99"]) < 0.006


# ------------------------------------------------------------ fp32 + Kahan time (O10, config 4) ---------------------
def test_fp32_distribution_matches_fp64():
    phi0 = math.asin(0.9)
    base = dict(model="underdamped", scheme="heun", alpha=0.1, temperature=0.05, gamma0=0.9, phi0=phi0, v0=0.0,
                threshold=phi0 + TWO_PI, dt=0.01)
    n = 6000
    r64 = oracle.simulate(oracle.make_params(precision="fp64", **base), n, 2, 1e4)
    r32 = oracle.simulate(oracle.make_params(precision="fp32", **base), n, 302, 1e4)
    assert np.all(r32["status"] == 0)
    assert stats.ks_2samp(r64["fpt"], r32["fpt"]).pvalue > 0.01
    assert abs(r64["fpt"].mean() - r32["fpt"].mean()) < 4 * r64["fpt"].std() * math.sqrt(2 / n)


def test_fp32_kahan_time_keeps_a_slow_ramp_exact():
    # zero noise, slow ramp: escape happens just past gamma = 1, at t ~ 1e5 after 2e6 steps.  A float accumulator
    # t += dt would stall/drift by per cent at this length ("requires a particular care"); the Kahan pair
    # keeps gamma(t) right, so the fp32 escape step agrees with the fp64 one to ~1e-6.
    base = dict(model="underdamped", scheme="heun", alpha=0.5, temperature=0.0, gamma0=0.0, nu=1e-5, phi0=0.0, v0=0.0,
                threshold=TWO_PI, dt=0.05)
    k64 = int(oracle.simulate(oracle.make_params(precision="fp64", **base), 1, 1, 1.2e5)["k"][0])
    r32 = oracle.simulate(oracle.make_params(precision="fp32", **base), 1, 1, 1.2e5)
    k32 = int(r32["k"][0])
    assert r32["status"][0] == 0 and 1.0 < r32["gamma"][0] < 1.02
    assert abs(k32 - k64) / k64 < 2e-5, (k32, k64)
    # outputs are computed in fp64 from the integer step index in both precisions
    assert r32["fpt"][0] == k32 * 0.05
    # a naive float accumulation of the same dt is far off at this length -- shows the test has teeth
    t = np.float32(0.0)
    acc = np.cumsum(np.full(200_000, np.float32(0.05), dtype=np.float32), dtype=np.float32)[-1]
    assert abs(float(acc) - 200_000 * 0.05) / (200_000 * 0.05) > 1e-4


def test_fp32_short_path_tracks_definition():
    # first steps of an fp32 run against the same recurrence evaluated in float64 numpy from the oracle's own fp32
    # normals: differences are a few float ulps per step
    phi0 = math.asin(0.5)
    p = oracle.make_params(model="underdamped", scheme="heun", precision="fp32", alpha=0.05, temperature=0.005,
                           gamma0=0.5, nu=1e-3, phi0=phi0, v0=0.0, threshold=phi0 + TWO_PI, dt=0.05)
    nst = 64
    phi, v, st, ke = oracle.trace(p, 4, 9, nst * 0.05, nst + 1)
    z = oracle.normals_f32(4, 9, 0, nst // 4).astype(np.float64)
    sig = math.sqrt(2 * 0.05 * 0.005 * 0.05)
    x, w = float(np.float32(phi0)), 0.0
    for k in range(1, nst + 1):
        g1, g2 = 0.5 + 1e-3 * (k - 1) * 0.05, 0.5 + 1e-3 * k * 0.05
        a1 = g1 - math.sin(x) - 0.05 * w
        xp = x + w * 0.05
        wp = w + a1 * 0.05 + sig * z[k - 1]
        a2 = g2 - math.sin(xp) - 0.05 * wp
        x, w = x + 0.025 * (w + wp), w + 0.025 * (a1 + a2) + sig * z[k - 1]
        assert abs(x - phi[k]) < 2e-6 and abs(w - v[k]) < 2e-6, k
