"""Multi-GPU sharding of the hot path.

Trajectories are independent and the Philox stream is keyed by the GLOBAL trajectory id, so a job of `n_total`
trajectories splits into contiguous id ranges, one per rank (one process per GPU), with no data-path exchange: rank r
calls fpt_simulate with `first_id = base_id + start_r`.  The per-trajectory outputs stay on the rank that produced them.
The only reduction the method has is the switching-current histogram: nbins+2 integer counts, summed over
ranks with one all_reduce.  Results are identical to a single-GPU run of the same ids, whatever the world size.
"""
from __future__ import annotations

from . import binding


def shard_range(n_total: int, rank: int, world: int) -> tuple[int, int]:
    """(start, count) of rank's contiguous id range: the first n_total % world ranks get one extra trajectory."""
    if n_total < 0 or world < 1 or not 0 <= rank < world:
        raise ValueError(f"bad shard request n_total={n_total} rank={rank} world={world}")
    q, r = divmod(n_total, world)
    start = rank * q + min(rank, r)
    return start, q + (1 if rank < r else 0)


def shard_params(params_kw: dict, n_total: int, rank: int, world: int) -> tuple[dict, int]:
    """Keyword parameters of this rank's call (first_id advanced to the shard) and its trajectory count."""
    start, count = shard_range(n_total, rank, world)
    kw = dict(params_kw)
    kw["first_id"] = int(kw.get("first_id", 0)) + start
    return kw, count


def allreduce_counts(counts, group=None):
    """Sum the histogram counts over the ranks, in place (int64 tensor of nbins+2; exact integer sum, order independent)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(counts, op=dist.ReduceOp.SUM, group=group)
    return counts


def simulate_sharded(params_kw: dict, n_total: int, seed: int, t_max: float, rank: int, world: int, hist=None,
                     group=None, simulate_fn=None, simulate_hist_fn=None, make_params_fn=None):
    """This rank's share of a job of n_total trajectories.

    hist = (hist_of, lo, hi, nbins) additionally returns the histogram of the WHOLE job (all_reduce over `group`).
    Returns (first_index, (fpt, gamma, status), counts_or_None); outputs cover ids [first_index, first_index + count).
    The *_fn hooks default to the CUDA binding; they exist so that the host-side logic can be exercised without a GPU.
    """
    simulate_fn = simulate_fn or binding.simulate
    simulate_hist_fn = simulate_hist_fn or binding.simulate_hist
    make_params_fn = make_params_fn or binding.make_params
    kw, count = shard_params(params_kw, n_total, rank, world)
    start = kw["first_id"] - int(params_kw.get("first_id", 0))
    p = make_params_fn(**kw)
    if hist is None:
        return start, simulate_fn(p, count, seed, t_max), None
    hist_of, lo, hi, nbins = hist
    f, g, s, counts = simulate_hist_fn(p, count, seed, t_max, lo, hi, nbins, hist_of=hist_of)
    return start, (f, g, s), allreduce_counts(counts, group)
