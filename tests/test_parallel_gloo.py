"""N > 1 host logic on CPU (gloo, world_size 2): history-range sharding and the one exchange step of SURVEY.md 8(e).
The per-rank moments that the CUDA kernels produce on a GPU are built here with numpy from synthetic batch sums;
what is tested is that all-reducing them and applying the finalisation formula of include/aepid.h equals the
pooled batch estimator over all ranks' batches."""
import os

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2510_24154_b200 import parallel


def test_shard_histories_partitions_the_range():
    for n, w in ((10, 3), (1_000_000_007, 8), (5, 8), (0, 2)):
        blocks = [parallel.shard_histories(n, r, w) for r in range(w)]
        assert blocks[0][0] == 0 and sum(b[1] for b in blocks) == n
        for a, b in zip(blocks[:-1], blocks[1:]):
            assert a[0] + a[1] == b[0]
        assert max(b[1] for b in blocks) - min(b[1] for b in blocks) <= 1
    with pytest.raises(ValueError):
        parallel.shard_histories(10, 2, 2)


def _rank_data(rank, nbins=1000, B=8):
    rng = np.random.default_rng(100 + rank)
    nb = rng.integers(900, 1100, size=B).astype(np.float64)           # histories per batch
    x = rng.gamma(5.0, 1.0, size=(B, nbins)) * nb[:, None] * 1e-3      # batch sums
    return x, nb


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    x, nb = _rank_data(rank)
    m = {"epid_s1": torch.from_numpy(x.sum(0)), "epid_s2": torch.from_numpy((x * x / nb[:, None]).sum(0)),
         "phantom_s1": None, "phantom_s2": None, "totals": np.array([nb.sum(), float(len(nb))])}
    m = parallel.allreduce_moments(m)
    q.put((rank, m["epid_s1"].numpy(), m["epid_s2"].numpy(), m["totals"].numpy()))
    dist.barrier()
    dist.destroy_process_group()


def test_allreduce_moments_equals_pooled_batch_estimator():
    world, port = 2, 29500 + os.getpid() % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs: p.start()
    res = [q.get(timeout=120) for _ in range(world)]
    for p in procs: p.join(timeout=60)
    xs, nbs = zip(*[_rank_data(r) for r in range(world)])
    x, nb = np.concatenate(xs), np.concatenate(nbs)
    N, B = nb.sum(), len(nb)
    mean = x.sum(0) / N
    sigma = np.sqrt((nb[:, None] * (x / nb[:, None] - mean) ** 2).sum(0) / ((B - 1) * N))   # pooled estimator
    for rank, s1, s2, tot in res:
        assert tot[0] == N and tot[1] == B
        m = s1 / tot[0]
        sg = np.sqrt(np.maximum(s2 - tot[0] * m * m, 0) / ((tot[1] - 1) * tot[0]))          # aepid_finalize_moments
        assert np.allclose(m, mean, rtol=1e-12) and np.allclose(sg, sigma, rtol=1e-8)


def test_allreduce_is_identity_without_a_process_group():
    x, nb = _rank_data(0)
    m = {"epid_s1": torch.from_numpy(x.sum(0)), "epid_s2": None, "phantom_s1": None, "phantom_s2": None, "totals": np.array([nb.sum(), 8.0])}
    ref = m["epid_s1"].clone()
    out = parallel.allreduce_moments(m)
    assert torch.equal(out["epid_s1"], ref) and float(out["totals"][0]) == nb.sum()
