"""Host-side sharding of the hot path over several GPUs (one process per GPU).

Every prediction and every serving step is independent, so the path shards with NO
data-path collective: a rank takes a contiguous range of steps (all buckets are step-sorted, so that
is one contiguous row range per bucket) or, for the what-if sweep, a range of hardware-spec vectors.
Only the per-configuration totals cross shard boundaries: one all-reduce(sum) of n_specs x n_cfg
floats.  ``torch.distributed`` is used for that all-reduce and for the max-over-ranks of the timed
region (backend nccl on GPUs, gloo in the CPU tests).  No method arithmetic lives here.
"""
from __future__ import annotations

import copy
from typing import Tuple

import numpy as np

from workloads import Bucket, Workload


def shard_range(n: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous, balanced split of range(n): sizes differ by at most one, the union is exact."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    return (n * rank) // world, (n * (rank + 1)) // world


def shard_seed(base_seed: int, rank: int) -> int:
    """Weak-scaling benchmark shards: every rank draws its own workload of the same recipe."""
    return base_seed + 1000 * rank


def shard_workload_by_steps(w: Workload, rank: int, world: int) -> Workload:
    """Rank's share of a step-segmented workload: steps [s0, s1), the matching row range of every
    bucket, CSR offsets rebased to the shard, configuration offsets clipped to the shard's steps (a
    configuration that straddles a shard boundary contributes a partial total on both ranks)."""
    if w.n_steps <= 0:
        raise ValueError("workload has no step segmentation")
    s0, s1 = shard_range(w.n_steps, rank, world)
    out = copy.copy(w)
    out.buckets = []
    for b in w.buckets:
        so = np.asarray(b.step_off, dtype=np.int64)
        r0, r1 = int(so[s0]), int(so[s1])
        out.buckets.append(Bucket(b.family, [np.ascontiguousarray(c[r0:r1]) for c in b.cols], b.dtype_bytes, b.hq,
                                  b.hkv, b.head_dim, (so[s0:s1 + 1] - r0).astype(np.int32),
                                  None if b.mult is None else np.ascontiguousarray(b.mult[r0:r1]), b.model_slot))
    out.n_steps = s1 - s0
    if w.cfg_off is not None:
        out.cfg_off = (np.clip(np.asarray(w.cfg_off, dtype=np.int64), s0, s1) - s0).astype(np.int32)
    out.name = f"{w.name}[steps {s0}:{s1}]"
    return out


def shard_specs(w: Workload, rank: int, world: int) -> Workload:
    """What-if sweep: rank's share of the hardware-spec vectors (descriptors are replicated)."""
    a, b = shard_range(len(w.specs), rank, world)
    out = copy.copy(w)
    out.specs = list(w.specs[a:b])
    out.name = f"{w.name}[specs {a}:{b}]"
    return out


def allreduce_cfg_totals(cfg_lat, dist=None):
    """Sum the per-configuration totals [n_specs, n_cfg] of all shards in place (the path's only
    exchange step; kilobytes, latency-bound).  ``cfg_lat`` is a torch tensor on the backend's device."""
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(cfg_lat, op=dist.ReduceOp.SUM)
    return cfg_lat


def max_over_ranks(seconds: float, dist=None, device="cpu") -> float:
    """Timed region of a multi-GPU run = the slowest rank's device time."""
    import torch
    t = torch.tensor([float(seconds)], dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(rows_per_rank: int, steps: int, seconds_local: float, world: int, dist=None, device="cpu") -> float:
    """Whole-job predictions/s: the units all ranks processed / the max-over-ranks time."""
    return world * rows_per_rank * steps / max_over_ranks(seconds_local, dist, device)
