"""Parameter-sweep batches: fpt_simulate_sweep against per-set fpt_simulate
calls, the oracle, the exact mean first-passage times of tests/golden/mfpt_overdamped.txt, and the barrier fit."""
import os

import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from oracle import kramers
import paper_1802_05065_b200 as fpt
from paper_1802_05065_b200 import analysis

pytestmark = pytest.mark.gpu

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "mfpt_overdamped.txt")


def _table():
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    return {float(a): float(b) for a, b in rows}


def test_sweep_equals_separate_calls_and_the_oracle():
    # heterogeneous sets: different models, schemes, precisions, caps; ragged size; more sets than pool streams
    base = fpt.workload("c2")
    sets, caps = [], []
    for i in range(11):
        kw = dict(base["params"], temperature=0.05 + 0.01 * i, first_id=1000 * i)
        if i % 4 == 1:
            kw.update(model="overdamped", scheme="em", temperature=0.2 + 0.02 * i)
        if i % 4 == 2:
            kw.update(scheme="em")
        if i % 4 == 3:
            kw.update(precision="fp32", nu=1e-4)
        sets.append(kw)
        caps.append(40.0 + 5.0 * i)
    n = 333
    f, g, s = fpt.simulate_sweep([fpt.make_params(**kw) for kw in sets], n, 9, caps)
    torch.cuda.synchronize()
    assert f.shape == (11, n)
    saw_cens = saw_esc = False
    for i, kw in enumerate(sets):
        f1, g1, s1 = fpt.simulate(fpt.make_params(**kw), n, 9, caps[i])
        torch.cuda.synchronize()
        assert torch.equal(f[i], f1) and torch.equal(g[i], g1) and torch.equal(s[i], s1), i
        o = oracle.simulate(oracle.make_params(**kw), n, 9, caps[i])
        assert np.array_equal(s[i].cpu().numpy(), o["status"]), i
        assert np.array_equal(f[i].cpu().numpy(), o["fpt"]) and np.array_equal(g[i].cpu().numpy(), o["gamma"]), i
        saw_cens |= bool((o["status"] == 1).any())
        saw_esc |= bool((o["status"] == 0).any())
    assert saw_cens and saw_esc


def test_sweep_edge_cases():
    p = fpt.make_params(**fpt.workload("c1")["params"])
    f, g, s = fpt.simulate_sweep([], 10, 1, 1.0)
    assert f.numel() == 0
    f, g, s = fpt.simulate_sweep([p, p], 0, 1, 1.0)
    assert f.shape == (2, 0)
    bad = fpt.make_params(**dict(fpt.workload("c1")["params"], dt=-1.0))
    out = fpt.binding._alloc_outputs(20)
    out[2].fill_(77)
    with pytest.raises(fpt.FptError):
        fpt.simulate_sweep([p, bad], 10, 1, 1.0, out=out)
    torch.cuda.synchronize()
    assert bool((out[2] == 77).all())                    # nothing was launched for the valid set either
    with pytest.raises(ValueError):
        fpt.simulate_sweep([p, p], 10, 1, [1.0])


def test_temperature_sweep_reproduces_exact_mfpt_and_barrier():
    """Overdamped washboard at gamma = 0.7: mean escape time against the exact quadrature values and the
    barrier from the Arrhenius slope (Eq. (12); the overdamped prefactor has no 1/theta) against the same fit on the exact values."""
    table = _table()
    temps = [0.2, 0.15, 0.1, 0.08]
    w = fpt.workload("c5")
    n = 20000
    sets = [fpt.make_params(**dict(w["params"], temperature=T, first_id=i * n)) for i, T in enumerate(temps)]
    f, g, s = fpt.simulate_sweep(sets, n, 5, 5e-3 * 4e6)
    torch.cuda.synchronize()
    mean, sem, cens = analysis.mean_escape_time(f.cpu().numpy(), s.cpu().numpy())
    assert list(cens) == [0, 0, 0, 0]
    for T, m, e in zip(temps, mean, sem):
        assert abs(m - table[T]) < 3.0 * e + 0.01 * table[T], (T, m, e, table[T])       # 3 sigma + 1 % Euler bias
    du_sim = analysis.barrier_from_sweep(temps, mean, "arrhenius")
    du_exact_law = kramers.arrhenius_slope(temps, [table[T] for T in temps])
    assert du_sim == pytest.approx(du_exact_law, abs=0.01)
    assert du_sim == pytest.approx(kramers.barrier(0.7), rel=0.15)          # finite-T prefactor drift: Kramers ratio 1.22 -> 1.11
