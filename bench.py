#!/usr/bin/env python
"""bench.py — predictions/s of the KernelSight-LM hot path on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (S1-S7: ks_predict_kernels + ks_compose_steps through the
C ABI) over config 2: 1,000,000 mixed kernel descriptors (GEMM 50% / attention 30% / elementwise
20%), Tier-A heads 12->128->128->1, 3906 serving steps, 16 configurations.  Inputs are resident in
HBM for `value`; `e2e` repeats the metric through ks_run_steps with HOST (pinned) buffers.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-extras]
N > 1: launched under torchrun, one rank per GPU; every rank runs its own seeded 1M-descriptor
shard (weak scaling, no data-path collective).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_28565_b200 import sharding as S  # noqa: E402
import workloads as W  # noqa: E402

METRIC = "kernel_latency_predictions_per_sec"
UNIT = "predictions/s"
FLOPS_PER_PRED = {(12, 128): 2 * (16 * 128 + 128 * 128 + 128), (8, 64): 2 * (8 * 64 + 64 * 64 + 64),
                  (32, 256): 2 * (32 * 256 + 256 * 256 + 256)}
BYTES_PER_ROW = {W.FAM_GEMM: 16, W.FAM_ATTN: 16, W.FAM_ELEMWISE: 12, W.FAM_GROUPED: 44, W.FAM_ALLREDUCE: 12}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=float(d["hbm_gbs"]), bf16=float(d["bf16_tflops"]),
                    bf16_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), source="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, source="fallback")   # B200_PROFILING.md


def load_traffic():
    """Per-launch DRAM bytes of the dominant kernel from the committed ncu capture (profiles/traffic.txt:
    lines of "<key> <bytes>"), or an empty dict."""
    p = os.path.join(ROOT, "profiles", "traffic.txt")
    out = {}
    if os.path.exists(p):
        for line in open(p):
            parts = line.split()
            if len(parts) == 2 and not line.startswith("#"):
                try:
                    out[parts[0]] = int(parts[1])
                except ValueError:
                    pass
    return out


class ClockSampler:
    """Polls SM clock and throttle reasons through NVML while the timed region runs."""
    BAD = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20}
    NOTE = {"sw_power_cap": 0x4, "hw_power_brake": 0x80}

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz, self._stop = [], set(), None, threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False
        self.t = threading.Thread(target=self._run, daemon=True)

    def _poll(self):
        nv = self.nv
        self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
        try:
            r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
        except Exception:
            r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
        for k, bit in {**self.BAD, **self.NOTE}.items():
            if r & bit:
                self.reasons.add(k)

    def _run(self):
        while not self._stop.is_set():
            try:
                self._poll()
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        if self.ok:
            self.t.start()

    def stop(self):
        self._stop.set()
        if self.ok:
            self.t.join(timeout=1.0)
            try:
                self._poll()
            except Exception:
                pass
        return dict(sm_mhz=float(np.median(self.samples)) if self.samples else None, sm_max_mhz=self.max_mhz,
                    reasons=sorted(self.reasons), samples=len(self.samples))


def oracle_models(w):
    """The oracle's copies of the workload's heads and grids (model loading, outside any timed region)."""
    from oracle import oracle as O
    O.build()
    return {f: O.Head(h) for f, h in w.heads.items()}, {f: O.Grid(g) for f, g in w.grids.items()}


def oracle_sample_rate(w, stride: int, models=None):
    """Time the oracle, as it stands, on every `stride`-th row of every bucket (+ Eq. 4 composition)."""
    from oracle import oracle as O
    heads, grids = models if models is not None else oracle_models(w)
    rows = [np.arange(0, b.n, stride) for b in w.buckets]
    t0 = time.perf_counter()
    lats, offs, n = [], [], 0
    for b, r in zip(w.buckets, rows):
        out = O.predict_bucket(b, w.specs, w.tier, head=heads.get(b.slot), grid=grids.get(b.slot), rows=r)
        lats.append(out["lat"][0])
        offs.append(np.searchsorted(r, b.step_off).astype(np.int64))   # sampled rows keep their step
        n += len(r) * len(w.specs)
    O.compose(lats, offs, w.n_steps, w.step_params, w.cfg_off)
    dt = time.perf_counter() - t0
    return n / dt, n, dt


def run_reference(args):
    """--impl reference: the CPU oracle, unmodified, on bounded samples of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = W.config2()
    models = oracle_models(w)
    stride = 100                                 # 10,000 of the 1,000,000 rows per step (~0.15 s)
    for _ in range(args.warmup):
        oracle_sample_rate(w, stride, models)
    t0 = time.perf_counter()
    n_tot = 0
    for _ in range(args.steps):
        _, n, _ = oracle_sample_rate(w, stride, models)
        n_tot += n
    dt = time.perf_counter() - t0
    val = n_tot / dt
    sample = f"every {stride}th row of each cfg2 bucket ({n_tot // max(args.steps, 1)} rows) per step, Tier A + Eq. 4"
    line = dict(metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=1e3 * dt / max(args.steps, 1), higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic", impl="reference",
                config=dict(workload="cfg2_mixed_1M (BASELINE.json configs[1]), bounded sample per step", tier="A"),
                cpu_baseline=dict(value=val, unit=UNIT, cores=1, kind="oracle", sample=sample),
                e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line))


# =============================================================================== our arm
class Harness:
    def __init__(self, device_index: int):
        import torch
        from paper_2606_28565_b200 import binding as B
        from paper_2606_28565_b200 import build as ksbuild
        from paper_2606_28565_b200 import driver as D
        ksbuild.build()
        self.torch, self.B, self.D = torch, B, D
        self.dev = f"cuda:{device_index}"
        torch.cuda.set_device(device_index)
        self.stream = torch.cuda.Stream()
        self.ctx = B.Context(device_index, stream=self.stream.cuda_stream)
        self.flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=self.dev)   # > 126 MB L2

    def flush_l2(self):
        self.flush_buf.zero_()

    def prepare(self, w):
        torch = self.torch
        self.D.load_models(self.ctx, w)
        db = self.D.to_device(w, self.dev)
        ns = len(w.specs)
        lat = [torch.empty((ns, b.n), dtype=torch.float32, device=self.dev) for b in db]
        n_cfg = int(w.cfg_off.shape[0]) - 1
        cfg = torch.from_numpy(np.ascontiguousarray(w.cfg_off, dtype=np.int32)).to(self.dev)
        step = torch.empty((ns, w.n_steps), dtype=torch.float32, device=self.dev)
        tot = torch.empty((ns, max(n_cfg, 1)), dtype=torch.float32, device=self.dev)
        torch.cuda.synchronize()                     # uploads ran on the default stream
        return dict(w=w, db=db, lat=lat, cfg=cfg, n_cfg=n_cfg, step=step, tot=tot, ns=ns)

    def prepare_rows(self, w):
        """prepare() for a workload without step segmentation (per-kernel predictions only)."""
        torch = self.torch
        self.D.load_models(self.ctx, w)
        db = self.D.to_device(w, self.dev)
        lat = [torch.empty((len(w.specs), b.n), dtype=torch.float32, device=self.dev) for b in db]
        torch.cuda.synchronize()
        return dict(w=w, db=db, lat=lat, ns=len(w.specs))

    def predict(self, st, buckets=None, lat=None):
        db = st["db"] if buckets is None else buckets
        self.ctx.predict_kernels(db, st["w"].specs, st["w"].tier, st["lat"] if lat is None else lat,
                                 space=self.B.KS_MEM_DEVICE)

    def compose(self, st):
        w = st["w"]
        self.ctx.compose_steps(st["lat"], [b.step_off for b in st["db"]], [b.n for b in st["db"]], w.n_steps, st["ns"],
                               w.step_params, st["cfg"], st["n_cfg"], st["step"], st["tot"], space=self.B.KS_MEM_DEVICE)

    def timed(self, fns, iters: int, warmup: int):
        """Run the callables in order `iters` times on the ctx stream with an L2 flush before every
        iteration; returns per-callable mean milliseconds (CUDA events around each callable)."""
        torch = self.torch
        n = len(fns)
        with torch.cuda.stream(self.stream):
            for _ in range(warmup):
                self.flush_l2()
                for f in fns:
                    f()
            evs = [[torch.cuda.Event(enable_timing=True) for _ in range(n + 1)] for _ in range(iters)]
            torch.cuda.synchronize()
            for it in range(iters):
                self.flush_l2()
                evs[it][0].record()
                for k, f in enumerate(fns):
                    f()
                    evs[it][k + 1].record()
            torch.cuda.synchronize()
        ms = np.array([[evs[it][k].elapsed_time(evs[it][k + 1]) for k in range(n)] for it in range(iters)])
        return ms


EX_ITERS, EX_WARM = 10, 3
PROFILE = False


def clone_sets(st, n_sets):
    """n_sets independent copies of a prepared workload's device buffers (inputs and outputs), so that
    back-to-back launches never find their data in the 126 MB L2 (rotation: every set is touched once
    per n_sets launches, and n_sets x bytes-per-set is several times the L2)."""
    import copy
    sets = []
    for _ in range(n_sets):
        db = [copy.copy(b) for b in st["db"]]
        for b in db:
            b.cols = [c.clone() for c in b.cols]
        sets.append(dict(db=db, lat=[x.clone() for x in st["lat"]]))
    return sets


def timed_b2b(h, fn, n_sets, iters):
    """Mean microseconds of fn(i) over `iters` back-to-back launches (one CUDA-event pair around all of
    them, on the ctx stream) after n_sets warm-up launches; fn(i) must use buffer set i % n_sets."""
    torch = h.torch
    with torch.cuda.stream(h.stream):
        for i in range(max(n_sets, 3)):
            fn(i)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(iters):
            fn(i)
        e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / iters * 1e3


def stream_roofline(h: Harness, st, peaks, iters=None, sets=None):
    """Per-family streaming-kernel HBM rate (one single-bucket ks_predict_kernels launch each) + compose."""
    out = {}
    w = st["w"]
    for i, b in enumerate(st["db"]):
        fn = (lambda i=i: h.predict(st, buckets=[st["db"][i]], lat=[st["lat"][i]]))
        ms = h.timed([fn], iters or EX_ITERS, EX_WARM)[:, 0]
        byts = BYTES_PER_ROW[b.family] * b.n * st["ns"] if st["ns"] == 1 else (BYTES_PER_ROW[b.family] - 4 + 4 * st["ns"]) * b.n
        gbs = byts / (ms.mean() * 1e-3) / 1e9
        out[W.FAM_NAMES[b.family]] = dict(rows=b.n, ms=float(ms.mean()), ms_min=float(ms.min()), gbs=float(gbs),
                                          frac_hbm=float(gbs / peaks["hbm"]), bytes_per_row=BYTES_PER_ROW[b.family])
        if sets is not None:   # back-to-back over rotating buffer sets: no launch gap, no flush tail
            us = timed_b2b(h, lambda k, i=i: h.predict(st, buckets=[sets[k % len(sets)]["db"][i]],
                                                       lat=[sets[k % len(sets)]["lat"][i]]), len(sets), 4 * len(sets))
            out[W.FAM_NAMES[b.family]].update(us_b2b=float(us), gbs_b2b=float(byts / us / 1e3),
                                              frac_hbm_b2b=float(byts / us / 1e3 / peaks["hbm"]))
    return out


def compose_roofline(h: Harness, st, peaks, iters=None, sets=None):
    w = st["w"]
    h.predict(st)
    ms = h.timed([lambda: h.compose(st)], iters or EX_ITERS, EX_WARM)[:, 0]
    rows = sum(b.n for b in st["db"]) * st["ns"]
    byts = 4 * rows + st["ns"] * w.n_steps * (4 + 4 * len(st["db"]))
    gbs = byts / (ms.mean() * 1e-3) / 1e9
    out = dict(rows=rows, steps=w.n_steps, ms=float(ms.mean()), ms_min=float(ms.min()), gbs=float(gbs),
               frac_hbm=float(gbs / peaks["hbm"]), launches_per_call=2)
    if sets is not None:
        for k in range(len(sets)):
            for a, b_ in zip(sets[k]["lat"], st["lat"]):
                a.copy_(b_)
        h.torch.cuda.synchronize()

        def comp(k):
            lat = sets[k % len(sets)]["lat"]
            h.ctx.compose_steps(lat, [b.step_off for b in st["db"]], [b.n for b in st["db"]], w.n_steps, st["ns"],
                                w.step_params, st["cfg"], st["n_cfg"], st["step"], st["tot"], space=h.B.KS_MEM_DEVICE)
        us = timed_b2b(h, comp, len(sets), 4 * len(sets))
        out.update(us_b2b=float(us), gbs_b2b=float(byts / us / 1e3), frac_hbm_b2b=float(byts / us / 1e3 / peaks["hbm"]))
    return out


def run_extras(h: Harness, peaks):
    """The other BASELINE.json configs at full size: per-kernel roofline context (not the bench line)."""
    ex = {}
    torch = h.torch
    # config 4a: Tier NONE streaming kernels + composition at ~29.9M kernel instances
    st = h.prepare(W.config4())
    sets = None if PROFILE else clone_sets(st, 4)
    ex["cfg4a_tierNONE"] = dict(stream=stream_roofline(h, st, peaks, sets=sets),
                                compose=compose_roofline(h, st, peaks, sets=sets))
    del sets
    ms = h.timed([lambda: h.predict(st), lambda: h.compose(st)], EX_ITERS, EX_WARM)
    ex["cfg4a_tierNONE"]["predictions_per_s"] = float(st["w"].n_rows / (ms.sum(axis=1).mean() * 1e-3))
    del st
    torch.cuda.empty_cache()
    # config 4b: the same 100k steps with Tier-A heads, materialised (29.9M rows) and in the paper's
    # layer-homogeneous form (one layer per step with multiplicity L, ~1.2M rows)
    for key, wl in (("cfg4b_tierA", W.config4(tier=W.TIER_A)), ("cfg4b_layer_homogeneous", W.config4(tier=W.TIER_A, dedupe=True))):
        st = h.prepare(wl)
        mult = [b.mult for b in st["db"]]

        def comp(st=st, wl=wl, mult=mult):
            h.ctx.compose_steps(st["lat"], [b.step_off for b in st["db"]], [b.n for b in st["db"]], wl.n_steps, st["ns"],
                                wl.step_params, st["cfg"], st["n_cfg"], st["step"], st["tot"], space=h.B.KS_MEM_DEVICE,
                                mult=mult)
        ms = h.timed([lambda st=st: h.predict(st), comp], 5 if not PROFILE else 1, 2 if not PROFILE else 1)
        t = float(ms.sum(axis=1).mean())
        ex[key] = dict(rows=wl.n_rows, steps=wl.n_steps, ms=t, predict_ms=float(ms[:, 0].mean()), compose_ms=float(ms[:, 1].mean()),
                       steps_per_s=float(wl.n_steps / (t * 1e-3)), kernel_instances_per_s=float(29898400 / (t * 1e-3)))
        del st
        torch.cuda.empty_cache()
    # NEXT-3: tensor-parallel all-reduce rows (Eq. 3), 6.4M rows = two per layer of cfg4's 100k steps
    st = h.prepare_rows(W.allreduce_rows())
    sets = None if PROFILE else clone_sets(st, 6)
    ex["allreduce_eq3"] = dict(stream=stream_roofline(h, st, peaks, sets=sets))
    del st, sets
    torch.cuda.empty_cache()
    # NEXT-2: bounded analytical head for every family of cfg2 (Tier A without the contraction)
    wb = W.config2()
    rng = np.random.Generator(np.random.PCG64(12))
    wb.bounded = {f: W.make_bounded_head(rng, 12) for f in list(wb.heads)}
    wb.heads = {}
    st = h.prepare(wb)
    ms = h.timed([lambda: h.predict(st)], EX_ITERS, EX_WARM)[:, 0]
    ex["cfg2_bounded_head"] = dict(ms=float(ms.mean()), predictions_per_s=float(wb.n_rows / (ms.mean() * 1e-3)),
                                   launches=3, note="streaming kernel, ~300 instructions per row: issue-bound")
    del st
    torch.cuda.empty_cache()
    # the packed bf16x2 activation mode of the Tier-A kernels (ks_set_gelu_mode(1); not the default: ~4x the
    # activation rounding error, still 10x inside the 1e-2 bar) on the bench workload
    st = h.prepare(W.config2())
    h.ctx.set_gelu_mode(1)
    ms = h.timed([lambda: h.predict(st)], EX_ITERS, EX_WARM)[:, 0]
    h.ctx.set_gelu_mode(0)
    ex["cfg2_gelu_mode1"] = dict(ms=float(ms.mean()), predictions_per_s=float(st["w"].n_rows / (ms.mean() * 1e-3)),
                                 note="Tier-A kernel only; packed bf16x2 GELU arithmetic")
    del st
    torch.cuda.empty_cache()
    # NEXT-2: MLP ensembles (Q17), 4 members of width 32 per family of cfg2, packed into one pass of the Tier-A kernel
    we = W.config2()
    rng = np.random.Generator(np.random.PCG64(13))
    we.ensembles = {f: W.make_ensemble(rng, 12, 32, 4) for f in list(we.heads)}
    we.heads = {}
    st = h.prepare(we)
    ms = h.timed([lambda: h.predict(st)], EX_ITERS, EX_WARM)[:, 0]
    ex["cfg2_ensemble_4x32"] = dict(ms=float(ms.mean()), predictions_per_s=float(we.n_rows / (ms.mean() * 1e-3)),
                                    launches=1, note="same kernel and tile shape as cfg2's single heads (H = 128)")
    del st
    torch.cuda.empty_cache()
    # config 3: Tier B, 4M queries
    st = h.prepare(W.config3())
    sets = None if PROFILE else clone_sets(st, 8)
    ex["cfg3_tierB"] = dict(stream=stream_roofline(h, st, peaks, sets=sets))
    del sets
    ms = h.timed([lambda: h.predict(st)], EX_ITERS, EX_WARM)
    ex["cfg3_tierB"]["predictions_per_s"] = float(st["w"].n_rows / (ms[:, 0].mean() * 1e-3))
    del st
    torch.cuda.empty_cache()
    # NEXT-1: density-routed Tier B on cfg3's 4M queries (grid inside the hull, 12->128->128->1 heads outside)
    st = h.prepare(W.config3(routed=True))
    ms = h.timed([lambda: h.predict(st)], EX_ITERS, EX_WARM)[:, 0]
    ex["cfg3_tierB_routed"] = dict(ms=float(ms.mean()), predictions_per_s=float(st["w"].n_rows / (ms.mean() * 1e-3)),
                                   launches=4, note="2 Tier-B passes that list the out-of-hull rows + 2 Tier-A passes over the lists")
    del st
    torch.cuda.empty_cache()
    # config 1: 4096 GEMM descriptors, launch-latency bound
    st = h.prepare(W.config1())
    ms = h.timed([lambda: h.predict(st)], 2 * EX_ITERS, EX_WARM)
    ex["cfg1_pr1"] = dict(us_per_batch=float(ms[:, 0].mean() * 1e3), predictions_per_s=float(4096 / (ms[:, 0].mean() * 1e-3)))
    del st
    # config 5: what-if sweep, 64 specs x 4,194,304 rows, heads 32->256->256->1
    st = h.prepare(W.config5())
    ms = h.timed([lambda: h.predict(st)], min(3, EX_ITERS), 1)[:, 0]
    n = st["w"].n_rows * st["ns"]
    tf = FLOPS_PER_PRED[(32, 256)] * n / (ms.mean() * 1e-3) / 1e12
    ex["cfg5_whatif"] = dict(predictions=n, ms=float(ms.mean()), predictions_per_s=float(n / (ms.mean() * 1e-3)),
                             tflops=float(tf), frac_tensor_sustained=float(tf / peaks["bf16_sustained"]))
    del st
    torch.cuda.empty_cache()
    # SURVEY.md §8(d) caveat (i): cfg 3's kernels last ~20 us and cfg 4a's attention bucket 16 us (launch ramp,
    # 128 KiB grid staging per CTA); the same kernels at 16x / 8x the row count show the steady rate
    if not PROFILE:
        st = h.prepare(W.config3(n=16 * 4_194_304))
        ex["asymptotic_cfg3_tierB_x16"] = dict(stream=stream_roofline(h, st, peaks, iters=3))
        del st
        torch.cuda.empty_cache()
        w4 = W.config4()
        attn = next(b for b in w4.buckets if b.family == W.FAM_ATTN)
        big = W.Bucket(W.FAM_ATTN, [np.tile(c, 8) for c in attn.cols], dtype_bytes=attn.dtype_bytes, hq=attn.hq,
                       hkv=attn.hkv, head_dim=attn.head_dim)
        w8 = W.Workload("cfg4a_attention_x8", [big], w4.specs, W.TIER_NONE)
        del w4
        st = h.prepare_rows(w8)
        ex["asymptotic_cfg4a_attention_x8"] = dict(stream=stream_roofline(h, st, peaks, iters=3))
        del st
        torch.cuda.empty_cache()
    ex["sim_closed_loop"] = sim_extras(h)
    return ex


def sim_extras(h):
    """NEXT-4: the closed simulation loop (host schedulers + one pass of the GPU path per iteration):
    256 what-if replicas x 200 requests each; wall-clock throughput of ks_sim_run (latency-bound: every
    iteration waits for its step times before the next batches can be formed)."""
    import time
    B = h.B
    out = {}
    n_rep, n_req = (256, 200) if not PROFILE else (8, 10)
    reps = W.sim_replicas(n_replicas=n_rep, n_requests=n_req, seed=6)
    model, spec = W.ServingModel(), W.spec_gb200()
    for name, tier in (("tierNONE", W.TIER_NONE), ("tierA", W.TIER_A)):
        if tier == W.TIER_A:
            rng = np.random.Generator(np.random.PCG64(1))
            for f in (W.FAM_GEMM, W.FAM_ATTN, W.FAM_ELEMWISE):
                h.ctx.load_heads(f, W.make_head(rng, 12, 128))
        best = None
        for _ in range(1 if PROFILE else 3):
            scheds = []
            for r in reps:
                s = B.Scheduler(r.max_num_batched_tokens, r.max_num_seqs, r.block_size, r.num_blocks)
                s.add_requests(r.arrival, r.prompt_len, r.max_new)
                scheds.append(s)
            clock = np.zeros(n_rep, np.float64)
            t0 = time.perf_counter()
            st, _, _ = B.sim_run(h.ctx, scheds, clock, model, spec, tier, W.STEP_PARAMS_CFG4)
            dt = time.perf_counter() - t0
            for s in scheds:
                s.close()
            if best is None or dt < best[0]:
                best = (dt, st, float(clock.max()))
        dt, st, sim_end = best
        it = max(st["iterations"], 1)
        out[name] = dict(replicas=n_rep, requests_per_replica=n_req, iterations=st["iterations"], steps=st["steps"],
                         rows=st["rows"], kernel_instances=st["kernel_instances"], wall_s=dt,
                         steps_per_s=st["steps"] / dt, kernel_instances_per_s=st["kernel_instances"] / dt,
                         us_per_iteration=dt / it * 1e6, simulated_s=sim_end,
                         us_per_iteration_by_phase=dict(schedule_and_pack=st["schedule_s"] / it * 1e6,
                                                        enqueue=st["enqueue_s"] / it * 1e6, wait_gpu=st["wait_s"] / it * 1e6,
                                                        commit=st["commit_s"] / it * 1e6))
    # the oracle's closed loop (Python scheduler + C predictor), one replica, bounded: 30 requests
    from oracle import sched as OS
    r = reps[0]
    o = OS.Scheduler(OS.SchedConfig(r.max_num_batched_tokens, r.max_num_seqs, r.block_size, r.num_blocks),
                     r.arrival[:30], r.prompt_len[:30], r.max_new[:30])
    om = OS.Model(**vars(model))
    t0 = time.perf_counter()
    _, priced, _ = OS.simulate(o, lambda b: float(OS.price_steps([b], om, spec, W.TIER_NONE, W.STEP_PARAMS_CFG4)[0]),
                               max_steps=None if not PROFILE else 20)
    dt = time.perf_counter() - t0
    out["oracle_tierNONE"] = dict(kind="oracle", sample="1 replica x 30 requests", steps=len(priced), wall_s=dt,
                                  steps_per_s=len(priced) / dt)
    return out


def run_ours(args):
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; the product path has no CPU fallback")
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    peaks = load_peaks()
    h = Harness(local)
    w = W.config2(seed=S.shard_seed(1, rank))      # every rank its own shard of the same recipe
    st = h.prepare(w)
    K, Wm = args.steps, max(args.warmup, 3)
    if args.profile:                               # ncu capture mode: few launches, no numbers reported
        global EX_ITERS, EX_WARM, PROFILE
        EX_ITERS, EX_WARM, Wm, PROFILE = 1, 1, args.warmup, True

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # warm-up, then the timed region: K steps, barrier + synchronize on both sides
    h.timed([lambda: h.predict(st), lambda: h.compose(st)], 1, Wm)
    launches0 = h.ctx.launch_count()
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    t_wall0 = time.perf_counter()
    # one CUDA-event pair around each whole step (predict + compose back to back, as a caller issues them:
    # the step kernel is launched programmatically dependent on the prediction kernel, and an event between
    # the two would serialise that), L2 flushed before every step outside the event pair
    step_ms = h.timed([lambda: (h.predict(st), h.compose(st))], K, 0)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    launches = h.ctx.launch_count() - launches0
    total_s = S.max_over_ranks(float(step_ms.sum()) * 1e-3, dist, h.dev)      # device time, max over ranks
    value = world * w.n_rows * K / total_s
    # per-kernel split for the roofline lines (not part of `value`): the same K steps with an event between
    ms = h.timed([lambda: h.predict(st), lambda: h.compose(st)], K, 0)

    # end to end through the C ABI with HOST (pinned) buffers: H2D + kernels + D2H inside the timed region
    hb = h.D.to_pinned(w)
    n_cfg = st["n_cfg"]
    step_h = torch.empty((1, w.n_steps), dtype=torch.float32).pin_memory()
    tot_h = torch.empty((1, n_cfg), dtype=torch.float32).pin_memory()
    cfg_h = torch.from_numpy(np.ascontiguousarray(w.cfg_off, dtype=np.int32)).pin_memory()
    lat_h = [torch.empty((1, b.n), dtype=torch.float32).pin_memory() for b in hb]

    def e2e_step(lat=None):
        h.ctx.run_steps(hb, [b.step_off for b in hb], w.specs, w.tier, w.n_steps, w.step_params, cfg_h, n_cfg,
                        step_h, tot_h, latency=lat, space=h.B.KS_MEM_HOST)

    def e2e_time(lat):
        Ke = 1 if args.profile else K
        # warm-up: the host-driven loop (copies, launches, a sync per step) needs ~0.2 s of activity
        # before clocks and the copy path settle (measured: 630 us/step at first, 330 us steady)
        t_w = time.perf_counter()
        n_w = 0
        while n_w < (1 if args.profile else 3) or (not args.profile and time.perf_counter() - t_w < 0.5):
            e2e_step(lat)
            n_w += 1
        # the host-driven loop is sensitive to what the host and the copy engines did just before (single
        # runs of K steps scatter by +-15 %): three repetitions of K steps, the median is reported
        rates = []
        for _ in range(1 if args.profile else 3):
            barrier()
            t0 = time.perf_counter()
            for _ in range(Ke):
                e2e_step(lat)
            torch.cuda.synchronize()
            rates.append(world * w.n_rows * Ke / S.max_over_ranks(time.perf_counter() - t0, dist, h.dev))
        return float(np.median(rates))

    # e2e: host descriptors in, the step's RESULT out (per-step and per-configuration latencies, S6-S7);
    # the per-kernel latencies are an intermediate and stay in HBM.  The variant that also returns every
    # per-kernel latency to the host (4 MB more D2H per step) is reported beside it.
    h2d = sum(4 * b.n * len(b.cols) + 4 * (w.n_steps + 1) for b in hb) + 4 * (n_cfg + 1)
    d2h = 4 * w.n_steps + 4 * n_cfg
    e2e = dict(value=e2e_time(None), unit=UNIT, h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h),
               returns="step and configuration latencies")
    e2e["with_kernel_latencies"] = dict(value=e2e_time(lat_h), unit=UNIT, h2d_bytes_per_step=int(h2d),
                                        d2h_bytes_per_step=int(d2h + sum(4 * b.n for b in hb)))

    if rank != 0:
        return
    # roofline of the dominant kernel (the fused Tier-A tcgen05 kernel = the single ks_predict_kernels launch)
    head = next(iter(w.heads.values()))
    flops = FLOPS_PER_PRED[(head.n_in, head.h1)] * w.n_rows
    mlp_ms = float(ms[:, 0].mean())
    achieved = flops / (mlp_ms * 1e-3) / 1e12
    traffic = load_traffic().get("ks_mlp_kernel_cfg2_bytes_per_launch")
    roofline = dict(bound="tensor", kernel="ks_mlp_ws_kernel<12,128>", achieved=achieved, peak=peaks["bf16"], unit="TFLOP/s",
                    frac=achieved / peaks["bf16"], traffic=traffic, peak_source=f"bf16 burst, {peaks['source']}",
                    flops_per_prediction=FLOPS_PER_PRED[(head.n_in, head.h1)], kernel_ms=mlp_ms,
                    compose_ms=float(ms[:, 1].mean()), step_ms=float(step_ms.mean()),
                    share_of_step=float(ms[:, 0].mean() / step_ms.mean()))
    # the binding unit of the Tier-A kernel is the MUFU pipe (2H tanh per prediction, 16 lanes/clk/SM):
    # peak = 16 x SMs x max SM clock
    tanh_per_s = 2 * head.h1 * w.n_rows / (mlp_ms * 1e-3)
    mufu_peak = 16 * torch.cuda.get_device_properties(local).multi_processor_count * (clocks.get("sm_max_mhz") or 1965) * 1e6
    roofline_alu = dict(bound="alu", kernel=roofline["kernel"], achieved=tanh_per_s / 1e12, peak=mufu_peak / 1e12,
                        unit="Ttanh/s", frac=tanh_per_s / mufu_peak,
                        note="MUFU.TANH evaluations; peak = 16 lanes/clk/SM x SMs x max SM clock")
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=K, warmup=Wm,
                ms_per_step=1e3 * total_s / K, higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="bf16", data="synthetic",
                config=dict(workload="cfg2_mixed_1M: BASELINE.json configs[1], 1,000,000 descriptors "
                                     "(GEMM 50/attention 30/elementwise 20), heads 12->128->128->1",
                            tier="A", n_steps=w.n_steps, n_cfg=n_cfg, rows_per_gpu=w.n_rows,
                            l2="flushed before every step (256 MiB write, outside the event pairs)",
                            timing="CUDA events on the ctx stream around predict and compose of every step"),
                clocks=clocks, e2e=e2e, gpu_launches=int(launches), roofline=roofline, roofline_alu=roofline_alu,
                wall_s_timed_region=t_wall)
    if world == 1:
        if not args.no_extras:
            line["extras"] = run_extras(h, peaks)
        wc = W.config2()
        rate, n, dt = oracle_sample_rate(wc, 1000 if args.profile else args.cpu_stride, oracle_models(wc))
        line["cpu_baseline"] = dict(value=rate, unit=UNIT, cores=1, kind="oracle",
                                    sample=f"every {args.cpu_stride}th row of each cfg2 bucket ({n} rows, {dt:.1f} s), "
                                           "Tier A + Eq. 4 composition, gcc -O2 single thread")
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--no-extras", action="store_true", help="skip the other configs' per-kernel measurements")
    ap.add_argument("--profile", action="store_true", help="ncu capture mode: one iteration of everything")
    ap.add_argument("--cpu-stride", type=int, default=2, help="oracle baseline samples every n-th row")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
