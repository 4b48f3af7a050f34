"""Scheduler A/B: the static split analysed in the paper's Appendix A against
the dynamic refill scheduler, on an imbalanced (near-exponential) workload.

  * results are bit-identical under both schedulers (and equal to the oracle's);
  * the static scheduler's issued lane-steps equal, EXACTLY, what the static split predicts from the per-trajectory
    lengths (lane j of L owns runs j, j+L, ...; a warp lasts as long as its slowest lane; poll granularity K);
  * its lane efficiency follows the closed form of Appendix A, oracle/appendix_a.py, for N_tpb = 32 (a warp), within
    the few per cent by which the escape-time law differs from an exponential (PAPER.md:417 says so itself);
  * the dynamic scheduler (refill + drain compaction) stays above 85 % / 95 % with 4 / 16 runs per lane, where the static
    split sits near 43 % / 63 %.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle
from oracle import appendix_a
import paper_1802_05065_b200 as fpt

pytestmark = pytest.mark.gpu

K = 16


def _run(w, n, schedule, geom):
    fpt.set_launch(*geom)
    fpt.set_schedule(schedule)
    try:
        p = fpt.make_params(**dict(w["params"], check_every=K))
        f, g, s = fpt.simulate(p, n, w["seed"], w["t_max"])
        torch.cuda.synchronize()
        st = fpt.last_stats()
    finally:
        fpt.set_schedule("dynamic")
        fpt.set_launch(0, 0, 0)
    return f.cpu().numpy(), g.cpu().numpy(), s.cpu().numpy(), st


def _static_issued(k_end, lanes, K):
    """Issued lane-steps of the static split: per warp, 32 * K * max over its lanes of sum_j ceil(k_j / K)."""
    n = len(k_end)
    intervals = -(-k_end // K)
    per_lane = np.zeros(lanes, dtype=np.int64)
    np.add.at(per_lane, np.arange(n) % lanes, intervals)
    return int(32 * K * per_lane.reshape(-1, 32).max(axis=1).sum())


@pytest.mark.parametrize("runs_per_lane", [1, 4, 16])
def test_static_split_matches_appendix_a_and_dynamic_beats_it(runs_per_lane):
    # overdamped washboard, gamma = 0.7, T = 0.08: mean ~1e5 steps, escape times exponential to a few per cent; no cap in reach
    w = fpt.workload("c5", temperature=0.08, t_max=5e-3 * 4e7)
    blocks, block = 16, 256                                        # 8 warps per block: drain compaction has room
    lanes = blocks * block
    n = lanes * runs_per_lane
    fs, gs, ss, st_static = _run(w, n, "static", (block, 0, blocks))
    fd, gd, sd, st_dyn = _run(w, n, "dynamic", (block, 0, blocks))
    assert st_static["grid"] == blocks and st_dyn["grid"] == blocks
    assert np.array_equal(fs, fd) and np.array_equal(gs, gd) and np.array_equal(ss, sd)
    assert np.all(ss == 0)
    m = 256                                                        # oracle on a sample of the ids (cost)
    ora = oracle.simulate(oracle.make_params(**w["params"]), m, w["seed"], w["t_max"])
    assert np.array_equal(fs[:m], ora["fpt"]) and np.array_equal(ss[:m], ora["status"])

    k_end = np.rint(fs / w["params"]["dt"]).astype(np.int64)
    assert st_static["useful_steps"] == int(k_end.sum()) == st_dyn["useful_steps"]
    assert st_static["issued_lane_steps"] == _static_issued(k_end, lanes, K)
    assert st_static["migrations"] == 0 and st_static["refill_atomics"] == 0

    model = appendix_a.efficiency(runs_per_lane, 32)
    cv = k_end.std() / k_end.mean()
    assert 0.9 < cv < 1.02, cv
    assert st_static["lane_efficiency"] == pytest.approx(model, rel=0.08), (st_static["lane_efficiency"], model)
    # what the refill scheduler buys on the same trajectories
    assert st_dyn["lane_efficiency"] > st_static["lane_efficiency"]
    if runs_per_lane >= 4:
        assert st_dyn["lane_efficiency"] > (0.85 if runs_per_lane == 4 else 0.95), st_dyn
