"""ORACLE (test infrastructure, not product code) -- the paper's Appendix A speed-up model, written out as defined.

PAPER.md:409-438.  N_r runs with iid exponential(1) lengths are split statically over N_tpb threads, N_L = N_r / N_tpb
runs each (A.2: a thread's load is Erlang(N_L, 1)).  The parallel time is the maximum over the threads (A.3), whose CDF
is the Erlang CDF to the power N_tpb (A.4); the speed-up is S = <E_t> / <E_p> (A.5; the printed denominator <E_n> is a
garble for <E_p>, G7) and the speed-up efficiency is S / N_tpb (Fig. 9).

Plain numpy/scipy, fp64:  <E_p> = int_0^inf (1 - F(x)^N_tpb) dx  with  F = regularised lower incomplete gamma P(N_L, x).
Pins (tests/test_oracle_appendix_a.py): N_L = 1 gives the harmonic number H_N exactly; N_tpb = 1 gives efficiency 1;
brute-force Monte Carlo of (A.1)-(A.3); monotone limits of PAPER.md:341.
"""
from __future__ import annotations

import numpy as np
from scipy import integrate, special


def mean_sequential_time(n_runs: int) -> float:
    """<E_t> of (A.1)-(A.2): mean of Erlang(N_r, 1) = N_r (unit mean run length)."""
    return float(n_runs)


def parallel_time_cdf(x, n_per_thread: int, n_threads: int):
    """(A.4): CDF[E_p, x] = CDF[Erlang(N_L, 1), x] ** N_tpb."""
    return special.gammainc(n_per_thread, np.asarray(x, dtype=np.float64)) ** n_threads


def mean_parallel_time(n_per_thread: int, n_threads: int) -> float:
    """<E_p> = int_0^inf (1 - CDF[E_p, x]) dx, by adaptive quadrature split at the bulk of the Erlang law."""
    if n_per_thread < 1 or n_threads < 1:
        raise ValueError("n_per_thread and n_threads must be >= 1")
    f = lambda x: 1.0 - parallel_time_cdf(x, n_per_thread, n_threads)   # noqa: E731
    sd = np.sqrt(n_per_thread)
    hi = n_per_thread + 12.0 * sd + 12.0 * np.log(n_threads + 1.0) + 40.0
    pts = [max(0.0, n_per_thread - 8.0 * sd), float(n_per_thread), n_per_thread + 8.0 * sd]
    val, _ = integrate.quad(f, 0.0, hi, points=pts, limit=400, epsabs=1e-12, epsrel=1e-12)
    return float(val)


def speedup(n_per_thread: int, n_threads: int) -> float:
    """(A.5): S = <E_t> / <E_p> with N_r = N_L * N_tpb."""
    return mean_sequential_time(n_per_thread * n_threads) / mean_parallel_time(n_per_thread, n_threads)


def efficiency(n_per_thread: int, n_threads: int) -> float:
    """Speed-up efficiency S / N_tpb (Fig. 9) = N_L / <max of N_tpb Erlang(N_L, 1)>."""
    return speedup(n_per_thread, n_threads) / n_threads
