"""CPU, world_size 2, gloo: the host logic of the multi-GPU path (paper_2606_28565_b200/sharding.py).

The path shards by steps with no data-path collective; the only exchange is the all-reduce of the
per-configuration totals, and the timed region is the max over ranks.  Each rank runs the ORACLE on its
shard (this is a test: the oracle stands in for the device), and the reduced result must equal the
oracle on the unsharded workload.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import oracle as O
from paper_2606_28565_b200 import sharding as S
import workloads as W


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _oracle_steps(w):
    lats = [O.predict_bucket(b, w.specs, W.TIER_NONE)["lat"][0] for b in w.buckets]
    return O.compose(lats, [b.step_off for b in w.buckets], w.n_steps, w.step_params, w.cfg_off)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = W.config4(n_steps=41, n_layers=2, n_cfg=5)
        shard = S.shard_workload_by_steps(w, rank, world)
        step, tot = _oracle_steps(shard)
        t = torch.from_numpy(np.ascontiguousarray(tot))[None, :].clone()
        S.allreduce_cfg_totals(t, dist)
        slow = S.max_over_ranks(0.010 * (rank + 1), dist)
        val = S.aggregate_throughput(1000, 7, 0.010 * (rank + 1), world, dist)
        # weak-scaling shards: same recipe, different seed, reproducible
        a = W.config2(n=3000, seed=S.shard_seed(1, rank))
        b = W.config2(n=3000, seed=S.shard_seed(1, rank))
        same = all(np.array_equal(x, y) for ba, bb in zip(a.buckets, b.buckets) for x, y in zip(ba.cols, bb.cols))
        out[rank] = dict(step=step, tot=t.numpy()[0].copy(), slow=slow, val=val, same=same,
                         first=int(a.buckets[0].cols[0][:64].sum()), range=S.shard_range(w.n_steps, rank, world))
    finally:
        dist.destroy_process_group()


def test_step_sharding_allreduce_and_max_over_ranks_world2():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    w = W.config4(n_steps=41, n_layers=2, n_cfg=5)
    step, tot = _oracle_steps(w)
    # no collective on the per-step path: the shards' steps, concatenated, are the unsharded steps
    got = np.concatenate([out[r]["step"] for r in range(world)])
    assert np.array_equal(got, step)
    assert out[0]["range"][0] == 0 and out[0]["range"][1] == out[1]["range"][0] and out[1]["range"][1] == w.n_steps
    # the one exchange: per-configuration totals, summed over ranks, on every rank
    for r in range(world):
        assert np.allclose(out[r]["tot"], tot, rtol=1e-12, atol=0)
    # timing: max over ranks; throughput = all ranks' units / that time
    assert all(abs(out[r]["slow"] - 0.020) < 1e-12 for r in range(world))
    assert all(abs(out[r]["val"] - 2 * 1000 * 7 / 0.020) < 1e-6 for r in range(world))
    assert all(out[r]["same"] for r in range(world)) and out[0]["first"] != out[1]["first"]


def test_shard_range_is_an_exact_partition():
    for n in (0, 1, 7, 100000):
        for world in (1, 2, 3, 8):
            edges = [S.shard_range(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(edges, edges[1:]))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        S.shard_range(4, 2, 2)


def test_spec_sharding_partitions_the_sweep():
    w = W.config5(n_rows=2000, n_specs=7)
    parts = [S.shard_specs(w, r, 3).specs for r in range(3)]
    assert sum(parts, []) == list(w.specs)
