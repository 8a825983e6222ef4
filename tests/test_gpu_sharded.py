"""-m gpu: the SHARDED product path through libks: two processes on the one GPU of
the test box, gloo for the host-side reduce.  Each rank takes its shard (steps of a serving workload, or spec vectors
of a what-if sweep), runs ks_run_steps on it, and the per-configuration totals meet in ONE all-reduce; the result must
equal the unsharded GPU result and the oracle.  The ranks never wait on one another on the device.
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

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _make(kind):
    if kind == "steps":
        return W.config4(n_steps=403, n_layers=3, n_cfg=7, tier=W.TIER_A)
    return W.config5(n_rows=30011, n_specs=6, n_layers=3)


def _run(w, n_specs_total=None, spec0=0):
    """ks_run_steps on device buffers; returns (step [ns, n_steps], totals [n_specs_total, n_cfg] with this shard's rows)."""
    from paper_2606_28565_b200 import binding as B
    from paper_2606_28565_b200 import driver as D
    ctx = B.Context(0)
    try:
        D.load_models(ctx, w)
        db = D.to_device(w)
        ns, n_cfg = len(w.specs), int(w.cfg_off.shape[0]) - 1
        cfg = torch.from_numpy(np.ascontiguousarray(w.cfg_off, dtype=np.int32)).cuda()
        step = torch.empty((ns, w.n_steps), dtype=torch.float32, device="cuda")
        tot = torch.empty((ns, n_cfg), dtype=torch.float32, device="cuda")
        ctx.run_steps(db, [b.step_off for b in db], w.specs, w.tier, w.n_steps, w.step_params, cfg, n_cfg, step, tot,
                      space=B.KS_MEM_DEVICE)
        torch.cuda.synchronize()
    finally:
        ctx.close()
    full = torch.zeros((n_specs_total or ns, n_cfg), dtype=torch.float32)
    full[spec0:spec0 + ns] = tot.cpu()
    return step.cpu().numpy(), full


def _worker(rank, world, port, kind, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = _make(kind)
        if kind == "steps":
            shard = S.shard_workload_by_steps(w, rank, world)
            step, tot = _run(shard)
        else:
            shard = S.shard_specs(w, rank, world)
            a, _ = S.shard_range(len(w.specs), rank, world)
            step, tot = _run(shard, len(w.specs), a)
        S.allreduce_cfg_totals(tot, dist)            # the path's only exchange
        out[rank] = dict(step=step, tot=tot.numpy().copy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("kind", ["steps", "specs"])
def test_sharded_run_steps_equals_unsharded_and_oracle(kind):
    world = 2
    out = mp.Manager().dict()
    mp.spawn(_worker, args=(world, _free_port(), kind, out), nprocs=world, join=True)
    w = _make(kind)
    step_u, tot_u = _run(w)
    tot_u = tot_u.numpy()
    # per-step results need no exchange: the shards' outputs, put side by side, are the unsharded output, bit for bit
    step_s = np.concatenate([out[r]["step"] for r in range(world)], axis=1 if kind == "steps" else 0)
    assert np.array_equal(step_s, step_u)
    for r in range(world):
        if kind == "steps":   # a configuration that straddles the shard boundary is the sum of two partial totals
            assert np.allclose(out[r]["tot"], tot_u, rtol=2e-6, atol=0)
        else:                 # spec shards own whole rows of the totals: the reduce is a gather
            assert np.array_equal(out[r]["tot"], tot_u)
    # ... and the oracle on the unsharded workload agrees (Tier A: 1e-2; sums of Tier-A latencies likewise)
    heads = {f: O.Head(h) for f, h in w.heads.items()}
    for s, spec in enumerate(w.specs):
        lats = [O.predict_bucket(b, [spec], W.TIER_A, head=heads[b.slot])["lat"][0] for b in w.buckets]
        so, to = O.compose(lats, [b.step_off for b in w.buckets], w.n_steps, w.step_params, w.cfg_off)
        assert np.max(np.abs(step_u[s] - so) / np.abs(so)) <= 1e-2
        assert np.max(np.abs(tot_u[s] - to) / np.abs(to)) <= 1e-2
