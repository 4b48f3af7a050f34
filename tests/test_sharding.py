"""Host-side logic of the multi-GPU path without a GPU: id-range arithmetic, first_id keying and
the histogram all_reduce, run with world size 2 and 3 on the gloo backend.  The compute hooks of simulate_sharded are
pointed at the ORACLE here (tests may use it; the product default is the CUDA binding), so the test also shows that a
sharded job reproduces the single-process result id by id."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_1802_05065_b200 import sharding, workloads


def test_shard_ranges_tile_the_job():
    for n in (0, 1, 7, 64, 1000, 10**6 + 3):
        for world in (1, 2, 3, 8):
            nxt = 0
            for r in range(world):
                start, count = sharding.shard_range(n, r, world)
                assert start == nxt and count >= 0
                nxt += count
            assert nxt == n
            sizes = [sharding.shard_range(n, r, world)[1] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.shard_range(10, 2, 2)
    kw, count = sharding.shard_params(dict(dt=0.1, first_id=1000), 10, 1, 2)
    assert kw["first_id"] == 1005 and count == 5 and kw["dt"] == 0.1


def _oracle_hooks():
    def simulate(p, n, seed, t_max):
        r = oracle.simulate(p, n, seed, t_max, nthreads=1)
        return torch.from_numpy(r["fpt"]), torch.from_numpy(r["gamma"]), torch.from_numpy(r["status"])

    def simulate_hist(p, n, seed, t_max, lo, hi, nbins, hist_of="gamma"):
        f, g, s = simulate(p, n, seed, t_max)
        vals = g if hist_of in ("gamma", 0) else f
        c = oracle.histogram(vals.numpy(), s.numpy(), lo, hi, nbins)
        return f, g, s, torch.from_numpy(c.astype(np.int64))

    return dict(simulate_fn=simulate, simulate_hist_fn=simulate_hist, make_params_fn=oracle.make_params)


def _worker(rank, world, port, n_total, outdir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = workloads.workload("c3", nu=5e-3, t_max=1.05 / 5e-3)
        start, (f, g, s), counts = sharding.simulate_sharded(w["params"], n_total, w["seed"], w["t_max"], rank, world,
                                                              hist=w["hist"], **_oracle_hooks())
        np.savez(os.path.join(outdir, f"r{rank}.npz"), start=start, f=f.numpy(), g=g.numpy(), s=s.numpy(), c=counts.numpy())
        dist.barrier()
    finally:
        dist.destroy_process_group()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_job_equals_single_process(world, tmp_path):
    n_total = 101                                   # ragged over 2 and 3 ranks
    mp.spawn(_worker, args=(world, _free_port(), n_total, str(tmp_path)), nprocs=world, join=True)
    w = workloads.workload("c3", nu=5e-3, t_max=1.05 / 5e-3)
    ref = oracle.simulate(oracle.make_params(**w["params"]), n_total, w["seed"], w["t_max"])
    of, lo, hi, nb = w["hist"]
    want_counts = oracle.histogram(ref["gamma"], ref["status"], lo, hi, nb).astype(np.int64)
    parts = [np.load(tmp_path / f"r{r}.npz") for r in range(world)]
    nxt = 0
    for p in parts:
        assert int(p["start"]) == nxt
        nxt += len(p["f"])
        assert np.array_equal(p["c"], want_counts)              # every rank holds the histogram of the WHOLE job
    assert nxt == n_total
    assert np.array_equal(np.concatenate([p["f"] for p in parts]), ref["fpt"])
    assert np.array_equal(np.concatenate([p["g"] for p in parts]), ref["gamma"])
    assert np.array_equal(np.concatenate([p["s"] for p in parts]), ref["status"])
    assert want_counts.sum() == int(np.sum(ref["status"] == 0)) > 0
