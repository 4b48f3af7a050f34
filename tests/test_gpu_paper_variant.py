"""GPU parity of SURVEY.md 8(f) item 4, the paper-faithful variant: FPT_SCHEME_PAPER = Alg. 1 / Alg. 3 as printed
(Euler, bias gamma_k before the step, strict phi_k > th, threshold pi - phi0) against the oracle's
scheme 2, bit for bit, in fp64 and fp32, on both integrator kernels; and FPT_PREC_FP32_FAST (the hardware sine of the
paper's single-precision kernels), which has no CPU twin and is compared statistically only."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
import paper_1802_05065_b200 as fpt

pytestmark = pytest.mark.gpu


def _np(t):
    return t.detach().cpu().numpy()


def _gpu(w, n, opts=None, first_id=0):
    p = fpt.make_params(**dict(w["params"], first_id=first_id))
    st = fpt.alloc_stats()
    f, g, s = fpt.simulate_ex(p, n, w["seed"], w["t_max"], opts=opts, stats=st)
    torch.cuda.synchronize()
    return (_np(f), _np(g), _np(s)), fpt.read_stats(st)


def _ora(w, n, first_id=0):
    return oracle.simulate(oracle.make_params(**dict(w["params"], first_id=first_id)), n, w["seed"], w["t_max"])


PHI0 = math.asin(0.9)
PAPER_ALG1 = dict(model="underdamped", scheme="paper", alpha=0.1, temperature=0.05, amp=1.0, gamma0=0.9, nu=0.0, phi0=PHI0, v0=0.0,
                  threshold=math.pi - PHI0, dt=0.01)                                       # Alg. 1 with its own threshold
PAPER_ALG3 = dict(model="underdamped", scheme="paper", alpha=0.1, temperature=0.01, amp=1.0, gamma0=0.0, nu=2e-3, phi0=0.0, v0=0.0,
                  threshold=math.pi, dt=0.02)                                              # Alg. 3: phi0 = asin(0) = 0, th = pi
CASES = [
    ("alg1 fp64", dict(params=dict(PAPER_ALG1, precision="fp64"), seed=2, t_max=400.0), 3001),
    ("alg1 fp32", dict(params=dict(PAPER_ALG1, precision="fp32"), seed=2, t_max=400.0), 3001),
    ("alg3 fp64", dict(params=dict(PAPER_ALG3, precision="fp64"), seed=3, t_max=1.05 / 2e-3), 1500),
    ("alg3 fp32", dict(params=dict(PAPER_ALG3, precision="fp32"), seed=3, t_max=1.05 / 2e-3), 1500),
    ("overdamped ramp fp64", dict(params=dict(model="overdamped", scheme="paper", precision="fp64", temperature=0.1, amp=1.0, gamma0=0.5,
                                              nu=1e-3, phi0=math.asin(0.5), threshold=math.pi - math.asin(0.5), dt=5e-3), seed=5,
                                  t_max=400.0), 2000),
    ("no sine, ramp, fp64", dict(params=dict(model="underdamped", scheme="paper", precision="fp64", alpha=0.4, temperature=0.2, amp=0.0,
                                             gamma0=0.0, nu=0.05, phi0=0.0, threshold=2.0, dt=0.01), seed=9, t_max=30.0), 1000),
]


@pytest.mark.parametrize("name,w,n", CASES, ids=[c[0] for c in CASES])
def test_paper_scheme_bit_exact_on_both_kernels(name, w, n):
    ora = _ora(w, n)
    assert 0 < np.sum(ora["status"] == 0)
    for opts in (fpt.launch_opts(specialise=False), fpt.launch_opts(specialise=True), None,
                 fpt.launch_opts(block=64, blocks_per_sm=1, max_blocks=5, specialise=False)):
        (f, g, s), st = _gpu(w, n, opts)
        assert np.array_equal(s, ora["status"])
        assert np.array_equal(f, ora["fpt"]) and np.array_equal(g, ora["gamma"])
        assert st["useful_steps"] == int(np.sum(ora["k"]))
        if w["params"]["amp"] != 0.0 and opts is not None and opts.specialise == 1:
            assert st["kernel"] == 2
    # the ordering of the bias update is visible: the textbook scheme gives other escape steps on the ramped cases
    if w["params"]["nu"] != 0.0:
        (f0, _, _), _ = _gpu(dict(w, params=dict(w["params"], scheme="em")), n)
        assert not np.array_equal(f0, f)


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
@pytest.mark.parametrize("model", ["overdamped", "underdamped"])
def test_paper_scheme_traces_bit_exact(model, precision):
    """Every state of 3000 steps, through the same State specialisation the production launch picks (ramp and no ramp)."""
    for nu in (0.0, 3e-4):
        kw = dict(model=model, scheme="paper", precision=precision, alpha=0.2, temperature=0.07, amp=1.0, gamma0=0.6, nu=nu, phi0=0.6,
                  v0=0.1, threshold=1e9, dt=0.01)
        n = 3000
        phi, v, st, ke = fpt.dbg_trace(fpt.make_params(**kw), 11, 12345, n * 0.01, n + 1)
        torch.cuda.synchronize()
        ophi, ov, ost, oke = oracle.trace(oracle.make_params(**kw), 11, 12345, n * 0.01, n + 1)
        assert np.array_equal(_np(phi), ophi) and int(st[0]) == ost and int(ke[0]) == oke
        if model == "underdamped":
            assert np.array_equal(_np(v), ov)


def test_strict_comparison_and_initial_state():
    """phi_k = 0.25 k exactly (no sine, no noise): '>=' escapes at k = 4, the paper's '>' at k = 5; phi0 == th escapes at
    k = 0 only with '>=' (the fill kernel's host-side test uses the same comparator)."""
    base = dict(model="overdamped", alpha=0.0, temperature=0.0, amp=0.0, gamma0=0.5, nu=0.0, phi0=0.0, threshold=1.0, dt=0.5)
    for precision in ("fp64", "fp32"):
        for scheme, k_want, k0_want in (("em", 4, 0), ("paper", 5, 1)):
            w = dict(params=dict(base, scheme=scheme, precision=precision), seed=1, t_max=10.0)
            (f, g, s), st = _gpu(w, 70)
            assert np.all(s == 0) and np.all(f == 0.5 * k_want)
            w0 = dict(params=dict(base, scheme=scheme, precision=precision, phi0=1.0), seed=1, t_max=10.0)
            (f0, _, s0), st0 = _gpu(w0, 70)
            assert np.all(s0 == 0) and np.all(f0 == 0.5 * k0_want) and st0["kernel"] == (0 if k0_want == 0 else 1)
            o = _ora(w0, 70)
            assert np.array_equal(f0, o["fpt"])


def test_hardware_sine_variant_is_statistically_the_fp32_paper_scheme():
    """FPT_PREC_FP32_FAST: sin.approx (absolute error ~1e-6 near the well) instead of the 2-ulp polynomial.  Paths decorrelate
    from the oracle's after a few thousand steps, so the comparison is statistical: two-sample KS (p > 0.01, BASELINE.json
    north_star) of escape times (Alg. 1) and switching currents (Alg. 3) against the fp32 oracle on OTHER ids, and the first
    steps of a trace within the sine's error."""
    from scipy import stats
    n = 4000
    w1 = dict(params=dict(PAPER_ALG1, precision="fp32_fast"), seed=2, t_max=1e4)
    (f, g, s), st = _gpu(w1, n)
    o = oracle.simulate(oracle.make_params(**dict(PAPER_ALG1, precision="fp32", first_id=10**6)), n, 2, 1e4)
    assert np.all(s == 0) and st["kernel"] == 1
    assert stats.ks_2samp(f, o["fpt"]).pvalue > 0.01
    assert abs(f.mean() - o["fpt"].mean()) < 5 * o["fpt"].std() / math.sqrt(n)
    w3 = dict(params=dict(PAPER_ALG3, precision="fp32_fast"), seed=3, t_max=1.05 / 2e-3)
    (f3, g3, s3), _ = _gpu(w3, n)
    o3 = oracle.simulate(oracle.make_params(**dict(PAPER_ALG3, precision="fp32", first_id=10**6)), n, 3, 1.05 / 2e-3)
    esc, oesc = s3 == 0, o3["status"] == 0                 # a few paths are still sliding down when the ramp ends (censored)
    assert np.all(s3 != 2) and esc.mean() > 0.9 and abs(esc.mean() - oesc.mean()) < 0.03
    assert stats.ks_2samp(g3[esc], o3["gamma"][oesc]).pvalue > 0.01
    # same ids: not bit-identical (it IS another sine), but the first hundred states track the oracle's to ~1e-5
    kw = dict(PAPER_ALG1, precision="fp32_fast", threshold=1e9)
    phi, v, _, _ = fpt.dbg_trace(fpt.make_params(**kw), 2, 7, 1.0, 101)
    ophi, ov, _, _ = oracle.trace(oracle.make_params(**dict(kw, precision="fp32")), 2, 7, 1.0, 101)
    assert np.max(np.abs(_np(phi) - ophi)) < 1e-4 and np.max(np.abs(_np(v) - ov)) < 1e-4
    (fx, _, _), _ = _gpu(dict(w1, params=dict(PAPER_ALG1, precision="fp32")), 512)
    assert not np.array_equal(fx, f[:512])
