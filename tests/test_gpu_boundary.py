"""GPU tests of the boundary (include/fpt.h): fpt_simulate_ex with per-call launch options and per-call statistics, the
warp-specialised kernel in every layout, and the corner cases of the shared-memory budget and the hand-over counters.

Everything is compared bit for bit with the oracle or with the plain call of the same job: outputs are a function of
(params, seed, id) only (fpt.h "Determinism")."""
import threading

import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
import paper_1802_05065_b200 as fpt

pytestmark = pytest.mark.gpu


def _np(t):
    return t.detach().cpu().numpy()


def _ex(w, n, opts=None, hist=False, first_id=0, check_every=0, seed=None):
    p = fpt.make_params(**dict(w["params"], first_id=first_id, check_every=check_every))
    st = fpt.alloc_stats()
    h = None
    if hist:
        of, lo, hi, nb = w["hist"]
        cnt = torch.zeros(nb + 2, dtype=torch.int64, device="cuda")
        h = (of, lo, hi, nb, cnt)
    f, g, s = fpt.simulate_ex(p, n, w["seed"] if seed is None else seed, w["t_max"], hist=h, opts=opts, stats=st)
    torch.cuda.synchronize()
    out = (_np(f), _np(g), _np(s)) + ((_np(cnt).astype(np.uint64),) if hist else ())
    return out, fpt.read_stats(st)


def _oracle(w, n, first_id=0, seed=None):
    return oracle.simulate(oracle.make_params(**dict(w["params"], first_id=first_id)), n, w["seed"] if seed is None else seed, w["t_max"])


def _assert_oracle(out, ora, w=None):
    f, g, s = out[:3]
    assert np.array_equal(s, ora["status"])
    ok = s != 2
    assert np.array_equal(f[ok], ora["fpt"][ok]) and np.array_equal(g[ok], ora["gamma"][ok])
    if len(out) > 3:
        of, lo, hi, nb = w["hist"]
        assert np.array_equal(out[3], oracle.histogram(ora["gamma"] if of == "gamma" else ora["fpt"], ora["status"], lo, hi, nb))


CASES = [
    ("c2 fp64 heun ud", fpt.workload("c2", t_max=300.0), 3001),
    ("c3 fp64 ramp + histogram", fpt.workload("c3", nu=2e-3, t_max=1.05 / 2e-3), 1500),
    ("c5 fp64 em od", fpt.workload("c5", temperature=0.1, t_max=1500.0), 2500),
    ("c4 fp32 kahan ramp + histogram", fpt.workload("c4", nu=2e-5, t_max=0.55 / 2e-5), 1200),
    ("fp64 em ud censored", fpt.workload("c2", scheme="em", t_max=40.0), 2000),
    ("fp32 heun od", dict(params=dict(model="overdamped", scheme="heun", precision="fp32", temperature=0.3, gamma0=0.6, phi0=0.5,
                                      threshold=5.0, dt=0.01, amp=1.0), seed=33, t_max=400.0, hist=None), 1100),
]


@pytest.mark.parametrize("name,w,n", CASES, ids=[c[0] for c in CASES])
def test_specialised_kernel_every_layout_matches_the_oracle(name, w, n):
    """Consumers integrate, producers generate the normals (csrc/fpt_specialised.cuh): every (consumers, producers) layout,
    one and two blocks per SM, a grid capped to a few blocks (every lane refills many times, then the block drains and
    its consumers park / adopt), with and without the fused histogram -- all equal to the oracle, bit for bit."""
    ora = _oracle(w, n)
    hist = w.get("hist") is not None
    saw_migration = False
    for nc, np_ in [(1, 1), (1, 2), (1, 3), (2, 1), (2, 2), (2, 3), (3, 1), (3, 2), (3, 3), (4, 1), (4, 2)]:
        for kw in (dict(), dict(max_blocks=3), dict(blocks_per_sm=2, max_blocks=5)):
            out, st = _ex(w, n, fpt.launch_opts(specialise=True, consumers=nc, producers=np_, **kw), hist=hist)
            _assert_oracle(out, ora, w)
            assert st["kernel"] == 2 and st["block"] == 32 * nc * (1 + np_), st
            assert st["useful_steps"] == int(np.sum(ora["k"])) and st["helper_lane_steps"] > 0
            assert st["n_escaped"] == int(np.sum(ora["status"] == 0)) and st["n_censored"] == int(np.sum(ora["status"] == 1))
            saw_migration |= st["migrations"] > 0
    assert saw_migration, "drain compaction between consumers never triggered"


def test_time_slicing_rotates_trajectories_without_changing_results():
    """fpt_launch_opts.time_slice: with fewer lanes than trajectories, a lane sets its trajectory aside in device memory every
    quantum (2048 steps or more) while others of its block's wait and takes the one that has waited longest.  A set-aside trajectory resumes from (phi, v[, t, c],
    k) with its Philox position, ramp registers and Kahan pair rebuilt: results stay the oracle's bit for bit -- narrow and wide
    spreads of the trajectory lengths, Heun and Euler, fp64 and fp32, with the fused histogram -- and the rotation really happens.
    The slicing variant of the kernel exists for the ramped-bias states only: for a constant bias the option is ignored."""
    cases = [
        (fpt.workload("c3", nu=2e-4, t_max=1.05 / 2e-4), 700, True),                         # fp64 ramp, ~2.4e5 steps each
        (fpt.workload("c4", nu=2e-5, t_max=0.55 / 2e-5), 900, True),                         # fp32 + Kahan time, ~3.6e5 steps
        (fpt.workload("c2", nu=1e-4, t_max=120.0), 3000, False),                             # hot, slow ramp: widely spread lengths, so finishes,
                                                                                             # refills and preemptions mix; some censored
        (fpt.workload("c5", temperature=0.1, nu=2e-5, t_max=1000.0), 2500, False),           # EM overdamped, ramped, some censored
    ]
    for w, n, hist in cases:
        ora = _oracle(w, n)
        for geo in (dict(block=64, blocks_per_sm=1, max_blocks=5), dict(block=128, blocks_per_sm=1, max_blocks=2),
                    dict(block=256, blocks_per_sm=1, max_blocks=1)):
            out, st = _ex(w, n, fpt.launch_opts(specialise=False, time_slice=True, **geo), hist=hist)
            _assert_oracle(out, ora, w)
            assert st["kernel"] == 1 and st["time_slices"] > 0, st
            assert st["useful_steps"] == int(np.sum(ora["k"])) and st["n_censored"] == int(np.sum(ora["status"] == 1))
        out, st = _ex(w, n, fpt.launch_opts(specialise=False, time_slice=False, block=64, blocks_per_sm=1, max_blocks=5), hist=hist)
        _assert_oracle(out, ora, w)
        assert st["time_slices"] == 0
    # a quantum of 64 steps (test hook): tens of hand-overs per trajectory, every poll of a K = 64 launch
    w, n, hist = cases[2]
    ora = _oracle(w, n)
    fpt.dbg_set_slice_quantum(64)
    try:
        out, st = _ex(w, n, fpt.launch_opts(specialise=False, time_slice=True, block=96, blocks_per_sm=1, max_blocks=3), hist=hist)
    finally:
        fpt.dbg_set_slice_quantum(0)
    _assert_oracle(out, ora, w)
    assert st["time_slices"] > 20 * n, st
    # constant bias: ignored (no slicing variant of those kernels), same results
    wc = fpt.workload("c2", t_max=60.0)
    out, st = _ex(wc, 2000, fpt.launch_opts(specialise=False, time_slice=True, block=64, blocks_per_sm=1, max_blocks=5))
    _assert_oracle(out, _oracle(wc, 2000), None)
    assert st["time_slices"] == 0
    # all trajectories resident: nothing ever waits, nothing is set aside
    w = fpt.workload("c3", nu=2e-3, t_max=1.05 / 2e-3)
    out, st = _ex(w, 256, fpt.launch_opts(specialise=False, time_slice=True, block=128, blocks_per_sm=1))
    _assert_oracle(out, _oracle(w, 256), None)
    assert st["time_slices"] == 0


def test_time_slicing_is_the_default_where_equal_length_trajectories_leave_a_ragged_wave():
    """The library's own choice (fpt_launch_opts.time_slice = 0): ramped fp32 jobs of 3 to 3.8 blocks of 128 per SM -- config 4's
    65 536 trajectories on 148 SMs -- run 3 blocks per SM with slicing; ramped jobs of 1 to 3 ragged waves slice at full
    occupancy; constant-bias jobs and short caps never do.  Same bits as without."""
    import torch
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    w4 = fpt.workload("c4", nu=1.5e-4, t_max=0.5 / 1.5e-4)                                    # ~6.7e4 steps each, cap 2^16 or more
    n = int(3.46 * 128 * sms)
    out, st = _ex(w4, n)
    assert st["kernel"] == 1 and st["grid"] == 3 * sms and st["block"] == 128 and st["time_slices"] > 0, st
    out0, st0 = _ex(w4, n, fpt.launch_opts(time_slice=False))
    assert st0["time_slices"] == 0 and st0["grid"] > 3 * sms
    assert all(np.array_equal(a, b) for a, b in zip(out, out0))
    w3 = fpt.workload("c3", nu=1e-3, t_max=1050.0)                                            # fp64, 1.5 waves
    _, full = _ex(fpt.workload("c3", nu=1e-1, t_max=10.5), 1 << 19)
    lanes = full["grid"] * full["block"]
    out, st = _ex(w3, lanes * 3 // 2)
    assert st["time_slices"] > 0 and st["grid"] * st["block"] == lanes, st
    out0, st0 = _ex(w3, lanes * 3 // 2, fpt.launch_opts(time_slice=False))
    assert st0["time_slices"] == 0 and all(np.array_equal(a, b) for a, b in zip(out, out0))
    _, st = _ex(w3, lanes * 5)                                                               # five waves: blends by itself
    assert st["time_slices"] == 0
    _, st = _ex(fpt.workload("c2", t_max=2000.0), lanes * 3 // 2)                            # constant bias: refill balances
    assert st["time_slices"] == 0


def test_default_poll_interval_follows_what_the_host_knows_about_the_trajectory_length():
    """check_every = 0: 64; 128 from long caps (2^21 steps fp64, 2^16 fp32); 512 when the bias is ramped and the ramp reaches
    the critical tilt (or the cap) only after 2^22 steps or more -- the length of a ramped trajectory is known in advance.
    Never changes results."""
    persistent = fpt.launch_opts(specialise=False)
    w = fpt.workload("c3", t_max=4.3e6 * 0.02)                         # config 3's own ramp (nu = 1e-6), cut at 4.3e6 steps: all censored
    out, st = _ex(w, 32, persistent)
    assert st["check_every"] == 512 and st["n_censored"] == 32, st
    _assert_oracle(out, _oracle(w, 32), None)
    out128, st128 = _ex(w, 32, persistent, check_every=128)
    assert st128["check_every"] == 128 and all(np.array_equal(a, b) for a, b in zip(out, out128))
    _, st = _ex(fpt.workload("c3", nu=1e-3, t_max=1050.0), 64, persistent)                  # 5e4 steps to the critical tilt
    assert st["check_every"] == 64
    _, st = _ex(fpt.workload("c3", nu=1e-5, t_max=50.0), 64, persistent)                    # long ramp, short cap
    assert st["check_every"] == 64
    _, st = _ex(fpt.workload("c2", t_max=5.0), 64, persistent)                              # constant bias, cap 500 steps
    assert st["check_every"] == 64
    _, st = _ex(fpt.workload("c4", nu=1e-4, t_max=5500.0), 64, persistent)                  # fp32, cap 1.1e5 steps
    assert st["check_every"] == 128


def test_specialised_kernel_is_the_default_for_small_jobs_only():
    w = fpt.workload("c2", t_max=60.0)
    out, st = _ex(w, 4000)
    assert st["kernel"] == 2                                     # cannot fill the GPU: specialised
    out2, st2 = _ex(w, 4000, fpt.launch_opts(specialise=False))
    assert st2["kernel"] == 1 and all(np.array_equal(a, b) for a, b in zip(out, out2))
    _, st3 = _ex(w, 4000, fpt.launch_opts(schedule="static"))    # the static split of Appendix A is a persistent-kernel mode
    assert st3["kernel"] == 1
    _, st4 = _ex(fpt.workload("c1"), 4000)                        # no sine: a step is a handful of operations, nothing to split
    assert st4["kernel"] == 1
    _, st5 = _ex(fpt.workload("c2", t_max=5.0), 1 << 20)          # fills the GPU
    assert st5["kernel"] == 1
    _, st6 = _ex(fpt.workload("c2", threshold=1.0), 100)          # decided at k = 0
    assert st6["kernel"] == 0 and st6["n_escaped"] == 100


def test_per_call_options_and_statistics_from_six_threads():
    """No state outside a call: six host threads, each on its own stream with its own launch options and its own device
    statistics block, get the outputs AND the counters of the same calls made one after the other."""
    jobs = [(fpt.workload("c2", t_max=80.0), 3001, 11, fpt.launch_opts(block=64, blocks_per_sm=1, max_blocks=9)),
            (fpt.workload("c5", temperature=0.15, t_max=600.0), 2000, 12, fpt.launch_opts(specialise=True, consumers=2, producers=2)),
            (fpt.workload("c3", nu=4e-3, t_max=1.05 / 4e-3), 1500, 13, fpt.launch_opts(schedule="static", block=96, blocks_per_sm=1, max_blocks=4)),
            (fpt.workload("c4", nu=5e-5, t_max=0.55 / 5e-5), 900, 14, fpt.launch_opts(tail_helper=False, block=128, blocks_per_sm=1, max_blocks=2)),
            (fpt.workload("c1"), 4000, 15, None),
            (fpt.workload("c2", t_max=30.0, scheme="em"), 2500, 16, fpt.launch_opts(specialise=True, consumers=4, producers=1, max_blocks=2))]
    ref = [_ex(w, n, o, seed=seed) for w, n, seed, o in jobs]
    streams = [torch.cuda.Stream() for _ in jobs]
    stats = fpt.alloc_stats(len(jobs))
    outs = [None] * len(jobs)
    last = [None] * len(jobs)

    def work(i):
        w, n, seed, o = jobs[i]
        p = fpt.make_params(**w["params"])
        with torch.cuda.stream(streams[i]):                      # torch allocates the outputs on the stream they are written on
            for _ in range(3):                                   # back to back on the same stream as well
                outs[i] = fpt.simulate_ex(p, n, seed, w["t_max"], opts=o, stats=(stats, i), stream=streams[i])
        streams[i].synchronize()
        last[i] = fpt.last_stats()                               # the deprecated shim: the calling THREAD's last call

    threads = [threading.Thread(target=work, args=(i,)) for i in range(len(jobs))]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    torch.cuda.synchronize()
    for i, ((rout, rst), out) in enumerate(zip(ref, outs)):
        assert all(np.array_equal(_np(a), b, equal_nan=True) for a, b in zip(out, rout)), i
        st = fpt.read_stats(stats, i)
        for key in ("n_traj", "n_escaped", "n_censored", "n_nan", "useful_steps", "n_cap", "grid", "block", "check_every", "kernel"):
            assert st[key] == rst[key], (i, key, st, rst)
            assert last[i][key] == rst[key], (i, key)
        if jobs[i][3] is not None and jobs[i][3].schedule == 1:   # static split: the issued lane-steps are deterministic too
            assert st["issued_lane_steps"] == rst["issued_lane_steps"]


def test_fused_histogram_of_8192_bins_next_to_the_static_shared_memory():
    """nbins = 8192 (the header's maximum) needs 32 KB of dynamic shared memory on top of the persistent kernel's 41.5 KB
    (fp64) / 17 KB (fp32) of static shared memory: above the 48 KB default, so the library has to opt in."""
    for w, n in [(fpt.workload("c3", nu=2e-3, t_max=1.05 / 2e-3), 1500), (fpt.workload("c4", nu=2e-5, t_max=0.55 / 2e-5), 1200)]:
        w = dict(w, hist=("gamma", w["hist"][1], w["hist"][2], 8192))
        ora = _oracle(w, n)
        for opts in (fpt.launch_opts(specialise=False), fpt.launch_opts(specialise=False, block=256, blocks_per_sm=1),
                     fpt.launch_opts(specialise=True), None):
            out, st = _ex(w, n, opts, hist=True)
            _assert_oracle(out, ora, w)
            assert int(out[3].sum()) == st["n_escaped"]
    # the standalone histogram agrees
    f, g, s, c = out
    c2 = fpt.histogram(torch.from_numpy(g).cuda(), torch.from_numpy(s).cuda(), w["hist"][1], w["hist"][2], 8192)
    assert np.array_equal(_np(c2).astype(np.uint64), c)


def test_tail_helper_hand_over_counters_cross_2_to_the_32():
    """The hand-over sequence counters are 64-bit (a served phase may last 2^53 steps).  Started just below 2^32 they run
    across the point where 32-bit counters would wrap; results and counters are those of the run that starts at 0."""
    w = fpt.workload("c2", t_max=400.0)
    n = 1536
    opts = fpt.launch_opts(block=128, blocks_per_sm=1, max_blocks=n // 128, specialise=False)
    ref, rst = _ex(w, n, opts, check_every=64)
    assert rst["helper_lane_steps"] > 0
    _assert_oracle(ref, _oracle(w, n))
    try:
        for seq0 in ((1 << 32) - 3, (1 << 31) - 2, (1 << 63) - 1):
            fpt.dbg_set_helper_seq0(seq0)
            out, st = _ex(w, n, opts, check_every=64)
            assert all(np.array_equal(a, b) for a, b in zip(out, ref)), seq0
            assert st["useful_steps"] == rst["useful_steps"] and st["helper_lane_steps"] > 0
    finally:
        fpt.dbg_set_helper_seq0(0)


def test_sweeps_from_two_host_threads():
    """fpt_simulate_sweep forks into a per-device stream pool: two threads sweeping at once must not interleave."""
    temps = [0.2, 0.15, 0.1, 0.08, 0.12, 0.18, 0.09, 0.11, 0.16, 0.14]
    sets = [fpt.make_params(**dict(fpt.workload("c5", temperature=T)["params"], first_id=1000 * i)) for i, T in enumerate(temps)]
    n = 700
    ref = [fpt.simulate_sweep(sets, n, seed, 900.0) for seed in (5, 6)]
    torch.cuda.synchronize()
    ref = [tuple(_np(x).copy() for x in r) for r in ref]
    outs = [None, None]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]

    def work(i):
        with torch.cuda.stream(streams[i]):
            for _ in range(4):
                outs[i] = fpt.simulate_sweep(sets, n, 5 + i, 900.0, stream=streams[i])
        streams[i].synchronize()

    threads = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    for i in range(2):
        assert all(np.array_equal(_np(a), b) for a, b in zip(outs[i], ref[i])), i
    # one set of the sweep against the oracle
    o = oracle.simulate(oracle.make_params(**dict(fpt.workload("c5", temperature=temps[3])["params"], first_id=3000)), n, 5, 900.0)
    assert np.array_equal(ref[0][0][3], o["fpt"]) and np.array_equal(ref[0][2][3], o["status"])
