"""N > 1 path on CPU: two gloo ranks shard a parameter batch, evaluate their shards independently (here with
the oracle standing in for the device, tiny C1-like vectors) and gather the per-vector results; the gathered
vector must equal the unsharded evaluation.  Also the max-over-ranks timing reduction."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import gen
import oracle as o
from paper_2510_07764_b200.shard import gather_vectors, max_over_ranks, shard_slice


def test_shard_slice_partitions_the_range():
    for n in (0, 1, 7, 8, 1024, 1025):
        for world in (1, 2, 3, 8):
            parts = [shard_slice(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[r][1] == parts[r + 1][0] for r in range(world - 1))
            sizes = [hi - lo for lo, hi in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_slice(4, 2, 2)


def _batch(n):
    rng = np.random.default_rng(3)
    E = gen.logspace(0.3, 3.0, 4)
    cfg = dict(n_spots=1, n_theta=4, n_phi=4, n_phase=4, n_fp=192, emission=0, oblate=0)
    P = np.stack([gen.pack_params(1.4, 12.0, 200.0, rng.uniform(0.2, 0.8), 0.2,
                                  spots=[(rng.uniform(0.5, 1.2), 0.0, 0.2, 6.5)]) for _ in range(n)])
    return cfg, E, P


def _score(cfg, E, p):
    f, st = o.evaluate(cfg, E, p)
    assert st == 0
    return float(f.sum())


def _worker(rank, world, port, n, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg, E, P = _batch(n)
    lo, hi = shard_slice(n, rank, world)
    local = torch.tensor([_score(cfg, E, P[b]) for b in range(lo, hi)], dtype=torch.float64)
    full = gather_vectors(local, n)
    tmax = max_over_ranks([float(rank + 1), 5.0 - rank])
    if rank == 0:
        out.put((full.numpy(), tmax))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_reproduce_the_unsharded_batch():
    n, world = 5, 2                                       # ragged: shards of 3 and 2
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    full, tmax = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    cfg, E, P = _batch(n)
    ref = np.array([_score(cfg, E, P[b]) for b in range(n)])
    # the oracle sums rows under OpenMP (order not fixed): equal up to summation round-off
    assert full.shape == ref.shape and np.allclose(full, ref, rtol=1e-12, atol=0)
    assert tmax == [2.0, 5.0]
