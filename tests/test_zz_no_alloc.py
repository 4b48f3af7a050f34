"""fpt_simulate_noalloc (include/fpt.h): the entry point for callers that must not allocate -- the persistent kernel with all
its scratch memory (global id counter, statistics, time-slicing parking slots and rings) in one file-scope device array of the
library.  Its outputs must be those of the existing, allocating path bit for bit (this suite's tolerance everywhere: the outputs
are a function of (params, seed, id) only), on calls made one after the other that share the array and find the previous call's
contents in it.  Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the others.
"""
import numpy as np
import pytest

import paper_1802_05065_b200 as fpt

pytestmark = pytest.mark.gpu


def _np(t):
    return t.detach().cpu().numpy()


def _existing(w, n):
    """the existing path: fpt_simulate (pool-allocated workspace, the library's own kernel choice)"""
    import torch
    f, g, s = fpt.simulate(fpt.make_params(**w["params"]), n, w["seed"], w["t_max"])
    torch.cuda.synchronize()
    return _np(f), _np(g), _np(s)


def _noalloc(w, n, out, stats):
    import torch
    fpt.simulate_noalloc(fpt.make_params(**w["params"]), n, w["seed"], w["t_max"], out, stats=stats)
    torch.cuda.synchronize()
    return tuple(_np(t).copy() for t in out), fpt.read_stats(stats)


def test_noalloc_entry_point_matches_the_existing_path_on_calls_in_a_row():
    import torch
    torch.cuda.set_device(0)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    n_max = fpt.binding.NOALLOC_MAX_TRAJ
    # caller-owned outputs and statistics block, allocated once, reused by every call (poisoned in between)
    out = (torch.empty(n_max, dtype=torch.float64, device="cuda"), torch.empty(n_max, dtype=torch.float64, device="cuda"),
           torch.empty(n_max, dtype=torch.int32, device="cuda"))
    stats = fpt.alloc_stats()
    ramp64 = fpt.workload("c3", nu=1e-3, t_max=1050.0)           # fp64 ramp: equal lengths, more trajectories than lanes -> sliced
    const64 = fpt.workload("c2", t_max=90.0)                     # constant bias: refill through the array's id counter; some censored
    ramp32 = fpt.workload("c4", nu=2e-4, t_max=2750.0)           # fp32 + Kahan time, sliced
    calls = [(ramp64, min(n_max, 5 * 128 * sms)), (const64, 20000), (ramp32, min(n_max, 6 * 128 * sms)), (ramp64, min(n_max, 5 * 128 * sms)),
             (const64, 777), (ramp64, 3 * 128 * sms + 5)]
    refs = {}
    sliced = 0
    for w, n in calls:
        key = (id(w), n)
        if key not in refs:
            refs[key] = _existing(w, n)
        for t in out:
            t.fill_(-7)
        got, st = _noalloc(w, n, tuple(t[:n] for t in out), stats)
        ref = refs[key]
        assert np.array_equal(got[2], ref[2]) and np.array_equal(got[0], ref[0]) and np.array_equal(got[1], ref[1]), (w["params"], n)
        assert st["kernel"] == 1 and st["n_traj"] == n and st["n_escaped"] + st["n_censored"] == n
        assert st["n_censored"] == int(np.sum(ref[2] == 1))
        assert np.all(_np(out[2][n:n + 64]) == -7)                       # nothing written past the caller's n
        sliced += st["time_slices"] > 0
    assert sliced >= 3                                                   # the slots and rings of the array were really used
    assert 0 < np.sum(refs[(id(const64), 20000)][2] == 1) < 20000
    # every trajectory decided at k = 0: the fill path, counters in the array
    w0 = fpt.workload("c2", threshold=-1.0)
    got, st = _noalloc(w0, 1000, tuple(t[:1000] for t in out), stats)
    ref = _existing(w0, 1000)
    assert all(np.array_equal(a, b) for a, b in zip(got, ref)) and st["kernel"] == 0 and st["n_escaped"] == 1000


def test_noalloc_entry_point_rejects_sizes_beyond_its_maximum():
    import torch
    torch.cuda.set_device(0)
    n = fpt.binding.NOALLOC_MAX_TRAJ + 1
    out = (torch.zeros(n, dtype=torch.float64, device="cuda"), None, torch.zeros(n, dtype=torch.int32, device="cuda"))
    w = fpt.workload("c2", t_max=5.0)
    with pytest.raises(fpt.FptError, match=r"beyond the fixed maximum.*code -3"):
        fpt.simulate_noalloc(fpt.make_params(**w["params"]), n, w["seed"], w["t_max"], out)
    torch.cuda.synchronize()
    assert int(out[2].abs().sum().item()) == 0 and float(out[0].abs().sum().item()) == 0.0      # nothing was enqueued
    fpt.simulate_noalloc(fpt.make_params(**w["params"]), n - 1, w["seed"], w["t_max"], tuple(None if t is None else t[:n - 1] for t in out))
    torch.cuda.synchronize()                                             # the maximum itself is accepted
    ref = _existing(w, n - 1)
    assert np.array_equal(_np(out[0][:n - 1]), ref[0]) and np.array_equal(_np(out[2][:n - 1]), ref[2])
