"""From-definition references used ONLY by the tests to pin the oracle (never by the product, never by the oracle).

Pure-Python Philox4x32-10 on Python ints, and the Box-Muller / Euler / Heun definitions evaluated in 50-digit
mpmath arithmetic -- i.e. the mathematics the oracle's double-precision code approximates, with none of its
polynomial approximations, bit tricks or rounding.  (DESIGN.md section 4 gives the definitions.)
"""
from __future__ import annotations

import os

from mpmath import mp, mpf

mp.dps = 50
MASK = 0xFFFFFFFF


def philox4x32_10(ctr, key):
    c0, c1, c2, c3 = ctr
    k0, k1 = key
    for _ in range(10):
        p0 = 0xD2511F53 * c0
        p1 = 0xCD9E8D57 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & MASK, p1 & MASK, ((p0 >> 32) ^ c3 ^ k1) & MASK, p0 & MASK
        k0 = (k0 + 0x9E3779B9) & MASK
        k1 = (k1 + 0xBB67AE85) & MASK
    return c0, c1, c2, c3


def philox_block(seed, tid, block):
    return philox4x32_10((block & MASK, block >> 32, tid & MASK, tid >> 32), (seed & MASK, seed >> 32))


def uniforms(o):
    X = (o[0] << 32) | o[1]
    Y = (o[2] << 32) | o[3]
    u1 = mpf(2 * (X >> 12) + 1) / mpf(2) ** 53
    f = mpf(Y >> 11) / mpf(2) ** 53
    return u1, f


def normal_pair(seed, tid, block):
    u1, f = uniforms(philox_block(seed, tid, block))
    r = mp.sqrt(-2 * mp.log(u1))
    return r * mp.cos(2 * mp.pi * f), r * mp.sin(2 * mp.pi * f)


def normal_for_step(seed, tid, k, cache):
    b = (k - 1) // 2
    if b not in cache:
        cache.clear()
        cache[b] = normal_pair(seed, tid, b)
    return cache[b][(k - 1) % 2]


def run(model, scheme, alpha, temperature, amp, gamma0, nu, phi0, v0, threshold, dt, n_cap, seed=None, tid=None,
        normals=None, max_steps=None):
    """Integrate one trajectory in mp arithmetic. Returns (status, k_end, states list [(phi,v)], min |phi-thr|)."""
    alpha, temperature, amp, gamma0, nu = mpf(alpha), mpf(temperature), mpf(amp), mpf(gamma0), mpf(nu)
    phi, v, thr, dt = mpf(phi0), mpf(v0), mpf(threshold), mpf(dt)
    sigma = mp.sqrt(2 * alpha * temperature * dt) if model == 1 else mp.sqrt(2 * temperature * dt)
    dgamma = nu * dt
    h2 = dt / 2
    gam = lambda j: gamma0 + dgamma * j
    F = lambda ph, j: gam(j) - amp * mp.sin(ph)
    states = [(phi, v)]
    margin = abs(phi - thr)
    # scheme 2 = the paper's Alg. 1 / Alg. 3 as printed: Euler with gamma_k (line 13 of
    # Alg. 3 comes before the update) and the strict test phi_k > th
    crossed = (lambda x: x > thr) if scheme == 2 else (lambda x: x >= thr)
    if crossed(phi):
        return 0, 0, states, margin
    cache = {}
    limit = n_cap if max_steps is None else min(n_cap, max_steps)
    for k in range(1, limit + 1):
        z = mpf(normals[k - 1]) if normals is not None else normal_for_step(seed, tid, k, cache)
        if scheme == 2:
            if model == 0:
                phi = phi + F(phi, k) * dt + sigma * z
            else:
                a = F(phi, k) - alpha * v
                phi, v = phi + v * dt, v + a * dt + sigma * z
        elif model == 0:
            if scheme == 0:
                phi = phi + F(phi, k - 1) * dt + sigma * z
            else:
                f1 = F(phi, k - 1)
                php = phi + f1 * dt + sigma * z
                phi = phi + h2 * (f1 + F(php, k)) + sigma * z
        else:
            if scheme == 0:
                a = F(phi, k - 1) - alpha * v
                phi, v = phi + v * dt, v + a * dt + sigma * z
            else:
                a1 = F(phi, k - 1) - alpha * v
                php = phi + v * dt
                vp = v + a1 * dt + sigma * z
                a2 = F(php, k) - alpha * vp
                phi, v = phi + h2 * (v + vp), v + h2 * (a1 + a2) + sigma * z
        states.append((phi, v))
        margin = min(margin, abs(phi - thr))
        if crossed(phi):
            return 0, k, states, margin
    return 1, limit, states, margin


def read_golden(name):
    """Parse tests/golden/<name>: returns list of token lists, comments and blanks dropped."""
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    rows = []
    with open(path) as fh:
        for line in fh:
            line = line.split("#", 1)[0].strip()
            if line:
                rows.append(line.split())
    return rows
