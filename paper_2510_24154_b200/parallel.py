"""Multi-GPU sharding of the history range: one process per GPU, histories are
independent, so the only exchange step is one all-reduce(sum) of the per-bin tally moments.

The arithmetic of the path stays in the CUDA kernels (aepid_read_moments / aepid_finalize_moments);
this module only partitions indices and calls torch.distributed (NCCL on GPUs; gloo in the CPU tests).
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def shard_histories(n_total: int, rank: int, world: int):
    """Contiguous block [first, first + n) of the global history range owned by `rank`."""
    if world < 1 or not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad shard arguments")
    first = (n_total * rank) // world
    last = (n_total * (rank + 1)) // world
    return first, last - first


def allreduce_moments(moments: dict, group=None):
    """In-place all-reduce(sum) of s1 / s2 tensors and the [histories, batches] totals.

    `moments` is what Engine.read_moments returns; tensors may live on CUDA (NCCL) or CPU (gloo).
    Returns the same dict with `totals` replaced by the global totals (a float64 tensor on the CPU)."""
    keys = [k for k in ("epid_s1", "epid_s2", "phantom_s1", "phantom_s2") if moments.get(k) is not None]
    dev = moments[keys[0]].device if keys else torch.device("cpu")
    tot = torch.as_tensor(moments["totals"], dtype=torch.float64).to(dev)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        for k in keys:
            dist.all_reduce(moments[k], op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(tot, op=dist.ReduceOp.SUM, group=group)
    moments["totals"] = tot.cpu()
    return moments


def simulate_sharded(engine, n_total: int, seed: int, rank: int, world: int):
    """Reset the tallies and run this rank's block of the global history range [0, n_total)."""
    first, n = shard_histories(n_total, rank, world)
    engine.reset_tallies()
    engine.set_history_offset(first)
    engine.simulate(n, seed)
    return first, n


def global_tallies(engine, group=None, epid=True, phantom=True):
    """Mean per history and standard error over ALL ranks' batches (device tensors)."""
    m = allreduce_moments(engine.read_moments(epid=epid, phantom=phantom), group)
    n_hist, n_batches = float(m["totals"][0]), float(m["totals"][1])
    out = {"n_histories": n_hist, "n_batches": n_batches}
    if epid:
        out["epid_mean"], out["epid_sigma"] = engine.finalize_moments(m["epid_s1"], m["epid_s2"], n_hist, n_batches)
    if phantom:
        out["phantom_mean"], out["phantom_sigma"] = engine.finalize_moments(m["phantom_s1"], m["phantom_s2"], n_hist, n_batches)
    return out
