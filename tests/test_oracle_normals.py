"""Pins P2(iii,iv) and the first lines of P10: Box-Muller normals of the oracle -- worked values, mpmath recomputation,
moments, one-sample KS against the normal law, and absence of correlation within and across blocks."""
import numpy as np
from mpmath import mpf
from scipy import stats

import oracle
from ref_mp import normal_pair as mp_pair, read_golden


def golden():
    return {r[0]: r[1:] for r in read_golden("worked_examples.txt")}


def test_worked_block_values():
    g = golden()
    z, u, f = oracle.normals_f64(1, 0, 0, 2, with_uniforms=True)
    assert u[0] == float.fromhex(g["uniform_u1"][0])
    assert f[0] == float.fromhex(g["uniform_f"][0])
    want = [float(x) for x in g["normals_b0"] + g["normals_b1"]]
    assert np.allclose(z, want, rtol=0, atol=2e-15)


def test_normals_vs_mpmath():
    rng = np.random.default_rng(21)
    for _ in range(300):
        seed, tid, b = (int(x) for x in rng.integers(0, 2**62, 3))
        z = oracle.normals_f64(seed, tid, b, 1)
        za, zb = mp_pair(seed, tid, b)
        assert abs(mpf(float(z[0])) - za) < 6e-15 and abs(mpf(float(z[1])) - zb) < 6e-15


def test_step_to_normal_assignment():
    # R4: step k (1-based) uses block (k-1) div 2; cos branch for odd k, sin branch for even k.  Checked through the
    # integrator: drifted Brownian motion with mu = 0, sigma = 1 exposes the normals as state increments.
    p = oracle.make_params(model="overdamped", scheme="em", amp=0.0, gamma0=0.0, temperature=0.5, phi0=0.0,
                           threshold=1e9, dt=1.0)
    phi, _, _, _ = oracle.trace(p, 77, 5, 1e3, 9)
    z = oracle.normals_f64(77, 5, 0, 4)
    assert np.allclose(np.diff(phi), z, rtol=0, atol=1e-14)
    for b in range(4):
        za, zb = mp_pair(77, 5, b)
        assert abs(float(za) - (phi[2 * b + 1] - phi[2 * b])) < 1e-13
        assert abs(float(zb) - (phi[2 * b + 2] - phi[2 * b + 1])) < 1e-13


def test_moments_and_ks():
    z = oracle.normals_f64(12345, 3, 0, 2_000_000)          # 4e6 normals of one stream
    n = z.size
    assert abs(z.mean()) < 4 / np.sqrt(n)
    assert abs(z.var() - 1) < 4 * np.sqrt(2 / n)
    assert abs(np.mean(z**3)) < 4 * np.sqrt(15 / n)
    assert abs(np.mean(z**4) - 3) < 4 * np.sqrt(96 / n)
    assert np.abs(z).max() < 8.58
    assert stats.kstest(z[:1_000_000], "norm").pvalue > 0.01
    za, zb = z[0::2], z[1::2]
    assert abs(np.corrcoef(za, zb)[0, 1]) < 4 / np.sqrt(za.size)                 # within a block
    assert abs(np.corrcoef(z[:-1], z[1:])[0, 1]) < 4 / np.sqrt(n)                # lag 1
    assert abs(np.corrcoef(za[:-1], za[1:])[0, 1]) < 4 / np.sqrt(za.size)        # across blocks


def test_across_ids_independent():
    z = oracle.normals_ids_f64(9, 0, 1_000_000)             # block 0 of 1e6 different trajectory ids
    assert abs(z.mean()) < 4 / np.sqrt(z.size)
    assert abs(z.var() - 1) < 4 * np.sqrt(2 / z.size)
    assert stats.kstest(z[::2], "norm").pvalue > 0.01
    assert abs(np.corrcoef(z[0:-2:2], z[2::2])[0, 1]) < 4 / np.sqrt(z.size / 2)  # neighbouring ids


def test_fp32_normals():
    z = oracle.normals_f32(4, 17, 0, 1_000_000).astype(np.float64)   # 4e6 normals
    n = z.size
    assert abs(z.mean()) < 4 / np.sqrt(n)
    assert abs(z.var() - 1) < 4 * np.sqrt(2 / n)
    assert abs(np.mean(z**4) - 3) < 4 * np.sqrt(96 / n)
    assert np.abs(z).max() < 6.77
    assert stats.kstest(z[:1_000_000], "norm").pvalue > 0.01
    q = z.reshape(-1, 4)
    for i in range(4):
        for j in range(i + 1, 4):
            assert abs(np.corrcoef(q[:, i], q[:, j])[0, 1]) < 4 / np.sqrt(q.shape[0])
