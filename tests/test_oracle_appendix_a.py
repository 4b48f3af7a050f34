"""Pins for oracle/appendix_a.py (the paper's Appendix A speed-up model)."""
import numpy as np
import pytest

from oracle import appendix_a as A


def test_one_run_per_thread_is_the_harmonic_number():
    # max of N iid exponential(1) has mean H_N = 1 + 1/2 + ... + 1/N (textbook): efficiency of the paper's own kernel
    for n in (1, 2, 20, 32, 512):
        h = float(np.sum(1.0 / np.arange(1, n + 1)))
        assert A.mean_parallel_time(1, n) == pytest.approx(h, rel=1e-10)
        assert A.efficiency(1, n) == pytest.approx(1.0 / h, rel=1e-10)
    assert A.efficiency(1, 32) == pytest.approx(0.24640, abs=1e-5)


def test_single_thread_is_perfect_and_cdf_is_a_cdf():
    for nl in (1, 7, 1000):
        assert A.efficiency(nl, 1) == pytest.approx(1.0, rel=1e-10)          # mean of Erlang(N_L,1) is N_L
    x = np.linspace(0.0, 200.0, 2001)
    c = A.parallel_time_cdf(x, 50, 20)
    assert c[0] == 0.0 and c[-1] == pytest.approx(1.0) and np.all(np.diff(c) >= 0)
    assert A.parallel_time_cdf(3.0, 2, 2) == pytest.approx((1.0 - np.exp(-3.0) * (1.0 + 3.0)) ** 2)   # Erlang(2) CDF by hand


def test_two_threads_two_runs_closed_form():
    # E[max(X, Y)] for X, Y ~ Erlang(2, 1): 2*E[X] - E[min]; P(min > x) = (e^-x (1+x))^2 -> E[min] = int = 1/2 + 1/2 + 1/4 = 5/4
    assert A.mean_parallel_time(2, 2) == pytest.approx(4.0 - 1.25, rel=1e-10)


def test_brute_force_monte_carlo():
    rng = np.random.default_rng(7)
    for nl, nt in ((1, 32), (5, 32), (10, 20), (50, 8)):
        loads = rng.exponential(1.0, size=(40000, nt, nl)).sum(axis=2)       # (A.1)-(A.2) per thread
        ep = loads.max(axis=1)                                               # (A.3)
        se = ep.std() / np.sqrt(len(ep))
        assert abs(ep.mean() - A.mean_parallel_time(nl, nt)) < 4.5 * se
        assert A.speedup(nl, nt) == pytest.approx(nl * nt / A.mean_parallel_time(nl, nt))


def test_limits_stated_in_the_paper():
    # efficiency -> 1 as N_r grows at fixed N_tpb; worse for more threads at fixed N_r
    e = [A.efficiency(nl, 20) for nl in (1, 2, 5, 10, 50, 100, 1000, 10000)]
    assert all(b > a for a, b in zip(e, e[1:])) and e[-1] > 0.98
    assert e[0] == pytest.approx(0.27795, abs=1e-4)
    n_r = 10240
    by_threads = [A.efficiency(n_r // nt, nt) for nt in (20, 32, 128, 512)]
    assert all(b < a for a, b in zip(by_threads, by_threads[1:]))
    # survey-session table, N_tpb = 32
    for nl, want in ((2, 0.334), (5, 0.466), (10, 0.566), (50, 0.760), (100, 0.821), (1000, 0.938)):
        assert A.efficiency(nl, 32) == pytest.approx(want, abs=1.5e-3)
