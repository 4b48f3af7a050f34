"""Pin P2(i): each transcendental of the oracle against mpmath (<= 4 ulp, the spec's sanity bar)
and against x87 long double on millions of arguments, including the reduction boundaries."""
import math

import numpy as np
import pytest
from mpmath import mp, mpf

import oracle

mp.dps = 50
PI_L = np.longdouble("3.14159265358979323846264338327950288")


def ulp_err(got, ref_mp):
    ref = float(ref_mp)
    u = math.ulp(abs(ref)) if ref != 0 else 5e-324
    return abs(mpf(got) - ref_mp) / mpf(u)


def test_sin_drift_vs_mpmath():
    rng = np.random.default_rng(1)
    xs = list(rng.uniform(-10, 10, 4000)) + list(rng.uniform(-1e-3, 1e-3, 200))
    # reduction boundaries: odd multiples of pi/2, multiples of pi, and their neighbours
    for n in range(-7, 8):
        for d in (0.0, 1e-12, -1e-12, 1e-7, -1e-7):
            xs.append(n * math.pi / 2 + d)
    xs += [0.0, -0.0, 5e-324, 1e-300, 1.0, -1.0, 100.0, -250.5, 1e4]
    x = np.array(xs)
    y = oracle.sin_drift(x)
    worst = 0.0
    for xi, yi in zip(x, y):
        ref = mp.sin(mpf(float(xi)))
        if abs(xi) <= 12:
            worst = max(worst, float(ulp_err(float(yi), ref)))
        # absolute accuracy near multiples of pi, where the relative error of any 2-term reduction degrades
        assert abs(mpf(float(yi)) - ref) < mpf(5e-16) * max(1.0, abs(xi)), xi
    assert worst <= 4.0, worst
    assert oracle.sin_drift(np.array([0.0]))[0] == 0.0


def test_sin_drift_vs_longdouble_bulk():
    rng = np.random.default_rng(2)
    x = rng.uniform(-10, 10, 2_000_000)
    y = oracle.sin_drift(x)
    ref = np.sin(x.astype(np.longdouble))
    err = np.abs(y.astype(np.longdouble) - ref) / np.spacing(np.abs(ref.astype(np.float64)))
    assert err.max() <= 4.0
    assert np.all(np.abs(y) <= 1.0)
    # odd symmetry is exact by construction
    assert np.array_equal(oracle.sin_drift(-x[:10000]), -y[:10000])


def test_uniform_open_exact():
    rng = np.random.default_rng(3)
    for X in [0, 1, 2**12 - 1, 2**12, 2**63, 2**64 - 1] + [int(v) for v in rng.integers(0, 2**63, 500)]:
        u = oracle.uniform_open(X)
        assert mpf(u) == mpf(2 * (X >> 12) + 1) / mpf(2) ** 53
        assert 0.0 < u < 1.0


def test_neg2log_vs_mpmath():
    rng = np.random.default_rng(4)
    js = [0, 1, 2, 3, 2**52 - 1, 2**52 - 2, 2**51, 2**51 - 1, 2**51 + 1] + [int(v) for v in rng.integers(0, 2**52, 3000)]
    js += [int(v) for v in rng.integers(0, 2**20, 300)]           # tiny u
    # mantissas around 1/sqrt2 and sqrt2 (the split point of the reduction)
    for e in range(1, 10):
        c = int(2**52 * 2**-e * math.sqrt(0.5) * 2)
        js += [c // 2 + d for d in (-2, -1, 0, 1, 2)]
    worst = 0.0
    for j in js:
        u = (2 * j + 1) * 2.0**-53
        w = float(oracle.neg2log(np.array([u]))[0])
        ref = -2 * mp.log(mpf(2 * j + 1) / mpf(2) ** 53)
        worst = max(worst, float(ulp_err(w, ref)))
        assert w > 0.0
    assert worst <= 4.0, worst


def test_neg2log_vs_longdouble_bulk():
    rng = np.random.default_rng(5)
    j = rng.integers(0, 2**52, 2_000_000, dtype=np.uint64)
    u = (j.astype(np.float64) * 2 + 1) * 2.0**-53
    w = oracle.neg2log(u)
    ref = -2 * np.log(u.astype(np.longdouble))
    err = np.abs(w.astype(np.longdouble) - ref) / np.spacing(np.abs(ref.astype(np.float64)))
    assert err.max() <= 4.0


def test_sincos_turns_vs_mpmath():
    rng = np.random.default_rng(6)
    Ys = [0, 2**64 - 1, 2**63, 2**62, 3 * 2**62, 2**61, 2**61 - 2**11, 2**61 + 2**11, 7 * 2**61, 7 * 2**61 - 2**11]
    Ys += [int(v) for v in rng.integers(0, 2**63, 3000)] + [int(v) + 2**63 for v in rng.integers(0, 2**63, 3000)]
    c, s = oracle.sincos_turns(np.array(Ys, dtype=np.uint64))
    for Y, ci, si in zip(Ys, c, s):
        ang = 2 * mp.pi * mpf(Y >> 11) / mpf(2) ** 53
        assert abs(mpf(float(ci)) - mp.cos(ang)) < 3e-16
        assert abs(mpf(float(si)) - mp.sin(ang)) < 3e-16
    assert abs(float(c[0]) - 1.0) == 0.0 and float(s[0]) == 0.0        # f = 0


def test_sincos_turns_bulk():
    rng = np.random.default_rng(7)
    Y = rng.integers(0, 2**64, 2_000_000, dtype=np.uint64)
    c, s = oracle.sincos_turns(Y)
    ang = 2 * PI_L * (Y >> np.uint64(11)).astype(np.longdouble) * np.longdouble(2.0) ** -53
    assert np.max(np.abs(c.astype(np.longdouble) - np.cos(ang))) < 3e-16
    assert np.max(np.abs(s.astype(np.longdouble) - np.sin(ang))) < 3e-16
    assert np.max(np.abs(c * c + s * s - 1.0)) < 1e-15


# ---- fp32 variant (O10): same shapes in float, bar <= 4 float ulp ----------------------------------------------

def test_fp32_sin_drift():
    rng = np.random.default_rng(8)
    x = rng.uniform(-10, 10, 1_000_000).astype(np.float32)
    y = oracle.sin_drift_f(x)
    ref = np.sin(x.astype(np.float64))
    err = np.abs(y.astype(np.float64) - ref) / np.spacing(np.abs(ref).astype(np.float32)).astype(np.float64)
    # near multiples of pi the 2-term float reduction loses relative accuracy; bound those absolutely
    far = np.abs(ref) > 0.05
    assert err[far].max() <= 4.0
    assert np.max(np.abs(y.astype(np.float64) - ref)) < 5e-7


def test_fp32_uniform_and_log():
    for o, want in [(0, 2.0**-33), (1, 2.0**-32 + 2.0**-33), (2**31, 0.5 + 2.0**-33), (2**32 - 1, 1.0), (2**32 - 127, 1.0), (2**32 - 129, 1.0 - 2.0**-24)]:
        assert oracle.uniform_open_f(o) == np.float32(want)
    assert oracle.uniform_open_f(2**32 - 1) == 1.0
    rng = np.random.default_rng(9)
    o = rng.integers(0, 2**32, 1_000_000, dtype=np.uint64)
    u = (o.astype(np.float32) * np.float32(2.0**-32) + np.float32(2.0**-33)).astype(np.float32)
    u = np.minimum(u, np.float32(1.0))
    w = oracle.neg2log_f(u)
    ref = -2 * np.log(u.astype(np.float64))
    ok = ref > 1e-3
    err = np.abs(w.astype(np.float64) - ref)[ok] / np.spacing(ref[ok].astype(np.float32)).astype(np.float64)
    assert err.max() <= 4.0
    assert np.all(w >= 0.0)
    assert oracle.neg2log_f(np.array([1.0], np.float32))[0] == 0.0
    assert abs(float(oracle.neg2log_f(np.array([2.0**-33], np.float32))[0]) - 66 * math.log(2)) < 1e-5


def test_fp32_sincos_turns():
    rng = np.random.default_rng(10)
    o = np.concatenate([rng.integers(0, 2**32, 1_000_000, dtype=np.uint64).astype(np.uint32),
                        np.array([0, 2**29 - 1, 2**29, 2**29 + 1, 2**30, 2**31, 3 * 2**30, 2**32 - 1, 2**32 - 2**29,
                                  2**32 - 2**29 - 1], dtype=np.uint32)])
    c, s = oracle.sincos_turns_f(o)
    ang = 2 * np.pi * o.astype(np.float64) * 2.0**-32
    assert np.max(np.abs(c.astype(np.float64) - np.cos(ang))) < 3e-7
    assert np.max(np.abs(s.astype(np.float64) - np.sin(ang))) < 3e-7
