"""Thin host driver: moves a synthetic Workload into HBM (torch tensors = device memory only),
loads its heads/grids into a libks Context and calls the C ABI through the binding.

Stands in for the paper's discrete-event scheduler, which "emits step/kernel
descriptor batches"; it performs no prediction arithmetic itself.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Optional

import numpy as np

from . import binding as B
from workloads import Workload


@dataclass
class DeviceBucket:
    family: int
    cols: list            # torch tensors on the GPU (int32 or float32), or pinned host tensors
    dtype_bytes: int
    hq: int
    hkv: int
    head_dim: int
    step_off: object = None
    mult: object = None   # optional int32 per-row multiplicities (layer-homogeneous form)
    model_slot: object = None   # efficiency-model slot (None = the family's)

    @property
    def n(self) -> int:
        return int(self.cols[0].shape[0]) if self.cols else 0


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("libks needs a CUDA device (B200, sm_100a); there is no CPU fallback")
    return torch


def to_device(w: Workload, device: str = "cuda:0") -> List[DeviceBucket]:
    torch = _torch()
    out = []
    for b in w.buckets:
        cols = [torch.from_numpy(np.ascontiguousarray(c)).to(device) for c in b.cols]
        so = torch.from_numpy(np.ascontiguousarray(b.step_off, dtype=np.int32)).to(device) if b.step_off is not None else None
        mu = torch.from_numpy(np.ascontiguousarray(b.mult, dtype=np.int32)).to(device) if b.mult is not None else None
        out.append(DeviceBucket(b.family, cols, b.dtype_bytes, b.hq, b.hkv, b.head_dim, so, mu, b.model_slot))
    return out


def to_pinned(w: Workload) -> List[DeviceBucket]:
    """Host-side (pinned) copy of the buckets for the end-to-end KS_MEM_HOST path."""
    torch = _torch()
    out = []
    for b in w.buckets:
        # one pinned block per bucket, columns back to back: the library moves adjacent columns with one copy
        if b.cols and all(c.dtype == b.cols[0].dtype and c.shape == b.cols[0].shape for c in b.cols):
            block = torch.from_numpy(np.ascontiguousarray(np.stack(b.cols))).pin_memory()
            cols = [block[k] for k in range(block.shape[0])]
        else:
            cols = [torch.from_numpy(np.ascontiguousarray(c)).pin_memory() for c in b.cols]
        so = torch.from_numpy(np.ascontiguousarray(b.step_off, dtype=np.int32)).pin_memory() if b.step_off is not None else None
        mu = torch.from_numpy(np.ascontiguousarray(b.mult, dtype=np.int32)).pin_memory() if b.mult is not None else None
        out.append(DeviceBucket(b.family, cols, b.dtype_bytes, b.hq, b.hkv, b.head_dim, so, mu, b.model_slot))
    return out


def load_models(ctx: B.Context, w: Workload) -> None:
    for fam, h in w.heads.items():
        ctx.load_heads(fam, h)
    for fam, members in getattr(w, "ensembles", {}).items():  # families whose Tier-A head is an MLP ensemble
        ctx.load_head_ensemble(fam, members)
    for fam, bh in getattr(w, "bounded", {}).items():      # families whose Tier-A head is the bounded analytical form
        ctx.load_bounded_head(fam, bh)
    for fam, g in w.grids.items():
        ctx.load_grid(fam, g)


def predict(ctx: B.Context, w: Workload, dbuckets: Optional[List[DeviceBucket]] = None, device: str = "cuda:0",
            aux: bool = True, tier: Optional[int] = None):
    """ks_predict_kernels on device-resident columns; returns per-bucket numpy outputs."""
    torch = _torch()
    db = dbuckets if dbuckets is not None else to_device(w, device)
    ns = len(w.specs)
    lat = [torch.empty((ns, b.n), dtype=torch.float32, device=device) for b in db]
    tiles = [torch.empty((ns, b.n), dtype=torch.int32, device=device) for b in db] if aux else None
    waves = [torch.empty((ns, b.n), dtype=torch.int32, device=device) for b in db] if aux else None
    troof = [torch.empty((ns, b.n), dtype=torch.float32, device=device) for b in db] if aux else None
    ctx.predict_kernels(db, w.specs, w.tier if tier is None else tier, lat, tiles, waves, troof, space=B.KS_MEM_DEVICE)
    torch.cuda.synchronize()
    res = []
    for i in range(len(db)):
        res.append(dict(lat=lat[i].cpu().numpy(), tiles=tiles[i].cpu().numpy() if aux else None,
                        waves=waves[i].cpu().numpy() if aux else None,
                        troof=troof[i].cpu().numpy() if aux else None, lat_dev=lat[i]))
    return res


def compose(ctx: B.Context, w: Workload, lat_dev: list, dbuckets: List[DeviceBucket], device: str = "cuda:0",
            params: Optional[dict] = None):
    """ks_compose_steps on device-resident latencies; returns (step_lat [ns,n_steps], cfg_lat [ns,n_cfg])."""
    torch = _torch()
    ns = len(w.specs)
    n_cfg = int(w.cfg_off.shape[0]) - 1 if w.cfg_off is not None else 0
    cfg = torch.from_numpy(np.ascontiguousarray(w.cfg_off, dtype=np.int32)).to(device) if n_cfg > 0 else None
    step = torch.empty((ns, w.n_steps), dtype=torch.float32, device=device)
    tot = torch.empty((ns, max(n_cfg, 1)), dtype=torch.float32, device=device)
    ctx.compose_steps(lat_dev, [b.step_off for b in dbuckets], [b.n for b in dbuckets], w.n_steps, ns,
                      params or w.step_params, cfg, n_cfg, step, tot, space=B.KS_MEM_DEVICE,
                      mult=[b.mult for b in dbuckets])
    torch.cuda.synchronize()
    return step.cpu().numpy(), tot.cpu().numpy()[:, :n_cfg]
