#!/usr/bin/env python
"""bench.py — predictions/s of the KernelSight-LM hot path on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (S1-S7: ks_predict_kernels + ks_compose_steps through the C ABI)
over the LARGEST single-GPU config of BASELINE.json, config 5: the what-if sweep, 4,194,304 kernel instances
of an 8-expert MoE decoder x 64 hardware-spec vectors = 268,435,456 predictions per step, Tier-A heads
32->256->256->1 on the tcgen05 tensor cores, 10,625 serving steps composed per spec.  Inputs are resident in
HBM for `value`; `e2e` is the same metric through ks_run_steps with HOST (pinned) buffers.  `extras` carries one
block per other config (1-4) — value, roofline of its dominant kernel, e2e, live parity against the oracle —
and the widened rows.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-extras] [--scaling weak|strong]

N > 1: one rank per GPU (the script re-launches itself under torch.distributed.run when WORLD_SIZE is unset).
weak: every rank prices its own seeded config-5 workload; strong: the 64 spec vectors are split over the ranks
(sharding.shard_specs), every rank runs the path on its share and the per-configuration totals meet in one
all-reduce.  No data-path collective either way.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402
from paper_2606_28565_b200 import sharding as S  # noqa: E402

METRIC = "kernel_latency_predictions_per_sec"
UNIT = "predictions/s"
FLOPS_PER_PRED = {(12, 128): 2 * (16 * 128 + 128 * 128 + 128), (8, 64): 2 * (8 * 64 + 64 * 64 + 64),
                  (32, 256): 2 * (32 * 256 + 256 * 256 + 256)}
BYTES_PER_ROW = {W.FAM_GEMM: 16, W.FAM_ATTN: 16, W.FAM_ELEMWISE: 12, W.FAM_GROUPED: 44, W.FAM_ALLREDUCE: 12}
CFG5_NAME = ("cfg5_whatif_moe: BASELINE.json configs[4], 4,194,304 kernel instances of an 8-expert top-2 MoE decoder "
             "x 64 hardware-spec vectors = 268,435,456 predictions, heads 32->256->256->1")
TIER_NAMES = {0: "NONE", 1: "A", 2: "B", 3: "B_ROUTED"}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=float(d["hbm_gbs"]), bf16=float(d["bf16_tflops"]),
                    bf16_sustained=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                    source="measured (MEASURED_PEAKS.json)")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, source="fallback (B200_PROFILING.md)")


def load_traffic():
    """Per-launch DRAM bytes of the dominant kernels from the committed ncu captures (profiles/traffic.txt: lines of
    "<key> <bytes> <capture file>"), or an empty dict.  These are NOT measured in this run (ncu cannot run inside a
    timed benchmark); every entry names the capture it comes from."""
    p = os.path.join(ROOT, "profiles", "traffic.txt")
    out = {}
    if os.path.exists(p):
        for line in open(p):
            parts = line.split()
            if len(parts) >= 2 and not line.startswith("#"):
                try:
                    out[parts[0]] = (int(parts[1]), parts[2] if len(parts) > 2 else "profiles/traffic.txt")
                except ValueError:
                    pass
    return out


def host_info():
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return dict(nproc=os.cpu_count(), cpu_model=model)


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


# =============================================================================== the oracle legs (CPU)
def oracle_models(w):
    """The oracle's copies of the workload's heads and grids (model loading, outside any timed region)."""
    from oracle import oracle as O
    O.build()
    return {f: O.Head(h) for f, h in w.heads.items()}, {f: O.Grid(g) for f, g in w.grids.items()}


def oracle_sample_rate(w, stride: int, models=None):
    """Time the oracle, as it stands, on every `stride`-th row of every bucket x all specs (+ Eq. 4 composition)."""
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


def _oracle_worker(args):
    """One process of the all-cores oracle figure: the oracle, unchanged, over its own disjoint rows."""
    cfg, stride, part, parts = args
    from oracle import oracle as O
    w = W.CONFIGS[cfg]()
    heads, grids = {f: O.Head(h) for f, h in w.heads.items()}, {f: O.Grid(g) for f, g in w.grids.items()}
    t0 = time.perf_counter()
    n = 0
    for b in w.buckets:
        r = np.arange(0, b.n, stride)[part::parts]
        O.predict_bucket(b, w.specs, w.tier, head=heads.get(b.slot), grid=grids.get(b.slot), rows=r)
        n += len(r) * len(w.specs)
    return n, time.perf_counter() - t0


def oracle_all_cores(cfg: str, stride: int):
    """The optional all-cores figure of SURVEY.md §8(d): independent processes over disjoint rows of the same sample, no
    change to the oracle; rate = predictions of all processes / the slowest process's time."""
    import multiprocessing as mp
    procs = os.cpu_count() or 1
    try:
        with mp.get_context("spawn").Pool(procs) as pool:
            res = pool.map(_oracle_worker, [(cfg, stride, p, procs) for p in range(procs)])
        n, dt = sum(r[0] for r in res), max(r[1] for r in res)
        return dict(value=n / dt, unit=UNIT, cores=procs, kind="oracle, one process per core over disjoint rows",
                    sample=f"{n} predictions, slowest process {dt:.1f} s")
    except Exception as e:                                   # a reported extra, never a reason to lose the bench line
        return dict(value=None, error=str(e)[:200])


def run_reference(args):
    """--impl reference: the CPU oracle, unmodified, on bounded samples of the headline workload (config 5)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = W.config5()
    models = oracle_models(w)
    stride = 65536                               # ~64 rows x 64 specs = ~4,100 predictions per step (~0.4 s)
    for _ in range(args.warmup):
        oracle_sample_rate(w, stride, models)
    t0 = time.perf_counter()
    n_tot = 0
    for _ in range(args.steps):
        _, n, _ = oracle_sample_rate(w, stride, models)
        n_tot += n
    dt = time.perf_counter() - t0
    val = n_tot / dt
    sample = (f"every {stride}th row of each cfg5 bucket x 64 specs ({n_tot // max(args.steps, 1)} predictions) per step, "
              "Tier A + Eq. 4, gcc -O2 single thread")
    line = dict(metric=METRIC, value=val, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=1e3 * dt / max(args.steps, 1), higher_is_better=True, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic", impl="reference",
                config=dict(workload=CFG5_NAME + "; bounded sample per step", tier="A"),
                cpu_baseline=dict(value=val, unit=UNIT, cores=1, kind="oracle", sample=sample, host=host_info()),
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
        self.red_dev = "cpu"                         # where the cross-rank reductions run (set by run_ours)
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
                               w.step_params, st["cfg"], st["n_cfg"], st["step"], st["tot"],
                               space=self.B.KS_MEM_DEVICE, mult=[b.mult for b in st["db"]])

    def timed(self, fns, iters: int, warmup: int):
        """Run the callables in order `iters` times on the ctx stream with an L2 flush before every
        iteration; returns per-callable milliseconds (CUDA events around each callable)."""
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


def stream_bytes(b, ns):
    return BYTES_PER_ROW[b.family] * b.n if ns == 1 else (BYTES_PER_ROW[b.family] - 4 + 4 * ns) * b.n


def stream_roofline(h: Harness, st, peaks, iters=None, sets=None):
    """Per-family streaming-kernel HBM rate (one single-bucket ks_predict_kernels launch each)."""
    out = {}
    for i, b in enumerate(st["db"]):
        fn = (lambda i=i: h.predict(st, buckets=[st["db"][i]], lat=[st["lat"][i]]))
        ms = h.timed([fn], iters or EX_ITERS, EX_WARM)[:, 0]
        byts = stream_bytes(b, st["ns"])
        gbs = byts / (ms.mean() * 1e-3) / 1e9
        out[W.FAM_NAMES[b.family]] = dict(rows=b.n, ms=float(ms.mean()), ms_min=float(ms.min()), gbs=float(gbs),
                                          frac_hbm=float(gbs / peaks["hbm"]), bytes_per_row=BYTES_PER_ROW[b.family])
        if sets is not None:   # back-to-back over rotating buffer sets: no launch gap, no flush tail
            us = timed_b2b(h, lambda k, i=i: h.predict(st, buckets=[sets[k % len(sets)]["db"][i]],
                                                       lat=[sets[k % len(sets)]["lat"][i]]), len(sets), 4 * len(sets))
            out[W.FAM_NAMES[b.family]].update(us_b2b=float(us), gbs_b2b=float(byts / us / 1e3),
                                              frac_hbm_b2b=float(byts / us / 1e3 / peaks["hbm"]))
    return out


def predict_all_roofline(h: Harness, st, peaks, iters=None, sets=None):
    """All buckets in ONE ks_predict_kernels call (Tier B: one merged launch)."""
    ms = h.timed([lambda: h.predict(st)], iters or EX_ITERS, EX_WARM)[:, 0]
    byts = sum(stream_bytes(b, st["ns"]) for b in st["db"])
    out = dict(rows=sum(b.n for b in st["db"]), bytes=int(byts), ms=float(ms.mean()), ms_min=float(ms.min()),
               frac_hbm=float(byts / (ms.mean() * 1e-3) / 1e9 / peaks["hbm"]))
    if sets is not None:
        us = timed_b2b(h, lambda k: h.predict(st, buckets=sets[k % len(sets)]["db"], lat=sets[k % len(sets)]["lat"]),
                       len(sets), 4 * len(sets))
        out.update(us_b2b=float(us), frac_hbm_b2b=float(byts / us / 1e3 / peaks["hbm"]))
    return out


def compose_bytes(st):
    w = st["w"]
    return 4 * sum(b.n for b in st["db"]) * st["ns"] + st["ns"] * w.n_steps * (4 + 4 * len(st["db"]))


def compose_roofline(h: Harness, st, peaks, iters=None, sets=None):
    w = st["w"]
    h.predict(st)
    ms = h.timed([lambda: h.compose(st)], iters or EX_ITERS, EX_WARM)[:, 0]
    byts = compose_bytes(st)
    gbs = byts / (ms.mean() * 1e-3) / 1e9
    out = dict(rows=sum(b.n for b in st["db"]) * st["ns"], steps=w.n_steps, ms=float(ms.mean()), ms_min=float(ms.min()),
               gbs=float(gbs), frac_hbm=float(gbs / peaks["hbm"]), launches_per_call=2)
    if sets is not None:
        for k in range(len(sets)):
            for a, b_ in zip(sets[k]["lat"], st["lat"]):
                a.copy_(b_)
        h.torch.cuda.synchronize()

        def comp(k, n_cfg):
            h.ctx.compose_steps(sets[k % len(sets)]["lat"], [b.step_off for b in st["db"]], [b.n for b in st["db"]],
                                w.n_steps, st["ns"], w.step_params, st["cfg"], n_cfg, st["step"], st["tot"],
                                space=h.B.KS_MEM_DEVICE)
        us = timed_b2b(h, lambda k: comp(k, st["n_cfg"]), len(sets), 4 * len(sets))
        us0 = timed_b2b(h, lambda k: comp(k, 0), len(sets), 4 * len(sets))
        out.update(us_b2b=float(us), gbs_b2b=float(byts / us / 1e3), frac_hbm_b2b=float(byts / us / 1e3 / peaks["hbm"]),
                   step_kernel_alone_us_b2b=float(us0),
                   step_kernel_alone_frac_hbm_b2b=float(byts / us0 / 1e3 / peaks["hbm"]))
    return out


def run_steps_roofline(h: Harness, st, peaks, iters=None, sets=None):
    """ks_run_steps in device space (Tier NONE, one spec: the one-kernel path of ks_fused.cu) with and without the
    per-kernel latency output; bytes = descriptor columns (+ 4 per kernel instance when the latencies are written)
    + step offsets and step latencies."""
    w = st["w"]
    cols = sum((BYTES_PER_ROW[b.family] - 4) * b.n for b in st["db"])
    steps = w.n_steps * (4 + 4 * len(st["db"]))
    rows = sum(b.n for b in st["db"])

    def run(db, lat):
        h.ctx.run_steps(db, [b.step_off for b in st["db"]], w.specs, w.tier, w.n_steps, w.step_params, st["cfg"], st["n_cfg"],
                        st["step"], st["tot"], latency=lat, space=h.B.KS_MEM_DEVICE)
    out = {}
    for name, with_lat in (("with_kernel_latencies", True), ("steps_only", False)):
        byts = cols + steps + (4 * rows if with_lat else 0)
        ms = h.timed([lambda: run(st["db"], st["lat"] if with_lat else None)], iters or EX_ITERS, EX_WARM)[:, 0]
        o = dict(bytes=int(byts), ms=float(ms.mean()), ms_min=float(ms.min()), launches_per_call=2,
                 frac_hbm=float(byts / (ms.mean() * 1e-3) / 1e9 / peaks["hbm"]),
                 kernel_instances_per_s=float(rows / (ms.mean() * 1e-3)))
        if sets is not None:
            us = timed_b2b(h, lambda k: run(sets[k % len(sets)]["db"], sets[k % len(sets)]["lat"] if with_lat else None),
                           len(sets), 4 * len(sets))
            o.update(us_b2b=float(us), frac_hbm_b2b=float(byts / us / 1e3 / peaks["hbm"]),
                     kernel_instances_per_s_b2b=float(rows / us * 1e6))
        out[name] = o
    out["note"] = ("one kernel computes the latencies in the step kernel's staging phase (no 2 x 4 B per kernel instance of "
                   "write + re-read); outputs bit-identical to ks_predict_kernels + ks_compose_steps")
    return out


# ------------------------------------------------------------------------------- end to end + parity per config
def e2e_measure(h: Harness, w, K: int, world: int = 1, dist=None, with_kernel_latencies: bool = False):
    """The metric through ks_run_steps with HOST (pinned) buffers: H2D + kernels + D2H inside the timed region.
    Returns the step's RESULT (per-step and per-configuration latencies); per-kernel latencies stay in HBM unless
    with_kernel_latencies."""
    torch = h.torch
    hb = h.D.to_pinned(w)
    ns = len(w.specs)
    n_cfg = int(w.cfg_off.shape[0]) - 1
    step_h = torch.empty((ns, w.n_steps), dtype=torch.float32).pin_memory()
    tot_h = torch.empty((ns, max(n_cfg, 1)), dtype=torch.float32).pin_memory()
    cfg_h = torch.from_numpy(np.ascontiguousarray(w.cfg_off, dtype=np.int32)).pin_memory()
    lat_h = [torch.empty((ns, b.n), dtype=torch.float32).pin_memory() for b in hb] if with_kernel_latencies else None

    def step():
        h.ctx.run_steps(hb, [b.step_off for b in hb], w.specs, w.tier, w.n_steps, w.step_params, cfg_h, n_cfg,
                        step_h, tot_h, latency=lat_h, space=h.B.KS_MEM_HOST)

    # warm-up: the host-driven loop (copies, launches, a sync per step) needs ~0.2 s of activity before clocks and the
    # copy path settle; then three repetitions of K steps, the median is reported (single runs scatter by +-15 %)
    t_w, n_w = time.perf_counter(), 0
    while n_w < (1 if PROFILE else 3) or (not PROFILE and time.perf_counter() - t_w < 0.5):
        step()
        n_w += 1
    rates = []
    n_pred = w.n_rows * ns
    for _ in range(1 if PROFILE else 3):
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(K):
            step()
        torch.cuda.synchronize()
        rates.append(world * n_pred * K / S.max_over_ranks(time.perf_counter() - t0, dist, h.red_dev))
    h2d = sum(4 * b.n * len(b.cols) + 4 * (w.n_steps + 1) + (4 * b.n if b.mult is not None else 0) for b in hb) + 4 * (n_cfg + 1)
    d2h = 4 * ns * w.n_steps + 4 * ns * n_cfg + (sum(4 * b.n * ns for b in hb) if with_kernel_latencies else 0)
    return dict(value=float(np.median(rates)), unit=UNIT, h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h),
                returns="step and configuration latencies" + (" + every per-kernel latency" if with_kernel_latencies else ""),
                steps_per_repetition=K)


def parity_sample(h: Harness, st, stride: int):
    """Live check of this run's outputs against the oracle on every `stride`-th row (+ the first and last 64) of every
    bucket, all specs: max relative error of the latency.  The oracle runs here, outside every timed region."""
    from oracle import oracle as O
    w = st["w"]
    heads, grids = oracle_models(w)
    h.predict(st)
    h.torch.cuda.synchronize()
    worst = 0.0
    for b, lat in zip(w.buckets, st["lat"]):
        if b.n == 0:
            continue
        rows = np.unique(np.concatenate([np.arange(0, b.n, stride), np.arange(min(64, b.n)), np.arange(max(b.n - 64, 0), b.n)]))
        o = O.predict_bucket(b, w.specs, w.tier, head=heads.get(b.slot), grid=grids.get(b.slot), rows=rows)
        g = lat[:, h.torch.from_numpy(rows).to(lat.device)].cpu().numpy().astype(np.float64)
        worst = max(worst, float(np.max(np.abs(g - o["lat"]) / np.maximum(np.abs(o["lat"]), 1e-300))))
    return worst


def config_block(h: Harness, w, peaks, K: int, roofline_fn, parity_stride: int, e2e_steps: int):
    """One `extras` block: whole-path throughput with inputs resident, roofline of the dominant kernel, e2e, parity."""
    st = h.prepare(w)
    ms = h.timed([lambda: h.predict(st), lambda: h.compose(st)], K, 2 if not PROFILE else 1)
    step_ms = float(ms.sum(axis=1).mean())
    n_pred = w.n_rows * st["ns"]
    blk = dict(workload=w.name, predictions=n_pred, tier=TIER_NAMES[w.tier], value=float(n_pred / (step_ms * 1e-3)), unit=UNIT,
               ms_per_step=step_ms, predict_ms=float(ms[:, 0].mean()), compose_ms=float(ms[:, 1].mean()))
    blk["roofline"] = roofline_fn(st, ms)
    blk["max_rel_err_vs_oracle"] = parity_sample(h, st, parity_stride)
    del st
    h.torch.cuda.empty_cache()
    if e2e_steps > 0:
        blk["e2e"] = e2e_measure(h, w, e2e_steps)
    h.torch.cuda.empty_cache()
    return blk


def _traffic(key):
    tr = load_traffic().get(key)
    return dict(traffic=tr[0] if tr else None,
                traffic_source=f"ncu capture {tr[1]} (dram__bytes_read.sum + dram__bytes_write.sum; not measured in this run)" if tr else None)


def tensor_roofline(kernel, n_in, h1, n_pred, kernel_ms, peak, peak_name, traffic_key, extra=None):
    flops = FLOPS_PER_PRED[(n_in, h1)]
    achieved = flops * n_pred / (kernel_ms * 1e-3) / 1e12
    out = dict(bound="tensor", kernel=kernel, achieved=achieved, peak=peak, unit="TFLOP/s", frac=achieved / peak,
               **_traffic(traffic_key), peak_source=peak_name, flops_per_prediction=flops, kernel_ms=kernel_ms)
    if extra:
        out.update(extra)
    return out


def hbm_roofline(kernel, byts, kernel_ms, peaks, traffic_key, extra=None):
    achieved = byts / (kernel_ms * 1e-3) / 1e9
    out = dict(bound="hbm", kernel=kernel, achieved=achieved, peak=peaks["hbm"], unit="GB/s", frac=achieved / peaks["hbm"],
               **_traffic(traffic_key), peak_source=f"copy rate, {peaks['source']}", algorithmic_bytes=int(byts),
               kernel_ms=kernel_ms)
    if extra:
        out.update(extra)
    return out


def run_extras(h: Harness, peaks):
    """Configs 1-4 at full size, one block each, then the widened rows."""
    ex = {}
    torch = h.torch
    K = 1 if PROFILE else 10
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    # ---- config 1: 4,096 GEMM descriptors, head 8->64->64->1 (launch-latency-bound)
    ex["cfg1"] = config_block(h, W.config1(), peaks, 2 * K, lambda st, ms: tensor_roofline(
        "ks_mlp_ws_kernel<8,64>", 8, 64, 4096, float(ms[:, 0].mean()), peaks["bf16"], f"bf16 burst, {peaks['source']}",
        "cfg1_mlp_bytes_per_launch", dict(note="32 tiles of 128 rows on 148 SMs: one launch latency, not a throughput")),
        parity_stride=1, e2e_steps=20 if not PROFILE else 1)

    # ---- config 2: 1M mixed descriptors, heads 12->128->128->1
    def cfg2_roof(st, ms):
        kms = float(ms[:, 0].mean())
        r = tensor_roofline("ks_mlp_ws_kernel<12,128>", 12, 128, st["w"].n_rows, kms, peaks["bf16"],
                            f"bf16 burst, {peaks['source']}", "cfg2_mlp_bytes_per_launch")
        mufu = 16 * n_sm * 1965e6
        r["alu"] = dict(bound="alu", achieved=2 * 128 * st["w"].n_rows / (kms * 1e-3) / 1e12, peak=mufu / 1e12, unit="Ttanh/s",
                        frac=2 * 128 * st["w"].n_rows / (kms * 1e-3) / mufu,
                        note="MUFU.TANH evaluations; peak = 16 lanes/clk/SM x SMs x 1965 MHz (DESIGN.md §5)")
        return r
    ex["cfg2"] = config_block(h, W.config2(), peaks, 2 * K, cfg2_roof, parity_stride=997, e2e_steps=20 if not PROFILE else 1)

    # ---- config 3: Tier B, 4M queries, one merged launch
    w3 = W.config3()
    ex["cfg3"] = config_block(h, w3, peaks, 2 * K, lambda st, ms: hbm_roofline(
        "ks_tierb_kernel (GEMM + attention buckets in one launch)", sum(stream_bytes(b, 1) for b in st["db"]),
        float(ms[:, 0].mean()), peaks, "cfg3_tierb_bytes_per_launch",
        dict(note="16 B per query; bound by the eight random shared-memory gathers per query, see DESIGN.md §5")),
        parity_stride=1009, e2e_steps=10 if not PROFILE else 1)
    st = h.prepare(w3)
    sets = None if PROFILE else clone_sets(st, 8)
    ex["cfg3"]["kernels"] = dict(tierB_all_buckets=predict_all_roofline(h, st, peaks, sets=sets),
                                 per_bucket_launches=stream_roofline(h, st, peaks, sets=sets))
    del st, sets
    torch.cuda.empty_cache()

    # ---- config 4a: Tier NONE streaming kernels + composition at 29.9M kernel instances
    w4 = W.config4()

    def cfg4a_roof(st, ms):
        byts = sum(stream_bytes(b, 1) for b in st["db"]) + compose_bytes(st)
        return hbm_roofline("ks_stream_kernel x 3 + ks_compose_kernel + ks_cfg_total_kernel (the whole step)", byts,
                            float(ms.sum(axis=1).mean()), peaks, "cfg4a_step_bytes",
                            dict(note="5 launches, each timed in `kernels` below"))
    ex["cfg4a"] = config_block(h, w4, peaks, K, cfg4a_roof, parity_stride=4999, e2e_steps=3 if not PROFILE else 1)
    st = h.prepare(w4)
    sets = None if PROFILE else clone_sets(st, 4)
    ex["cfg4a"]["kernels"] = dict(stream=stream_roofline(h, st, peaks, sets=sets),
                                  compose=compose_roofline(h, st, peaks, sets=sets))
    ex["cfg4a"]["run_steps_one_kernel"] = run_steps_roofline(h, st, peaks, sets=sets)
    del st, sets
    torch.cuda.empty_cache()

    # ---- config 4b: the same 100k steps with Tier-A heads, materialised (29.9M rows) and in the paper's
    # layer-homogeneous form (one layer per step with multiplicity L, ~1.2M rows)
    ex["cfg4b"] = config_block(h, W.config4(tier=W.TIER_A), peaks, 3 if not PROFILE else 1, lambda st, ms: tensor_roofline(
        "ks_mlp_ws_kernel<12,128>", 12, 128, st["w"].n_rows, float(ms[:, 0].mean()), peaks["bf16"],
        f"bf16 burst, {peaks['source']}", "cfg4b_mlp_bytes_per_launch"), parity_stride=9973, e2e_steps=2 if not PROFILE else 1)
    wl = W.config4(tier=W.TIER_A, dedupe=True)
    st = h.prepare(wl)
    ms = h.timed([lambda: h.predict(st), lambda: h.compose(st)], 5 if not PROFILE else 1, 2 if not PROFILE else 1)
    t = float(ms.sum(axis=1).mean())
    ex["cfg4b_layer_homogeneous"] = dict(rows=wl.n_rows, steps=wl.n_steps, ms=t, predict_ms=float(ms[:, 0].mean()),
                                         compose_ms=float(ms[:, 1].mean()), steps_per_s=float(wl.n_steps / (t * 1e-3)),
                                         kernel_instances_per_s=float(29898400 / (t * 1e-3)))
    del st
    torch.cuda.empty_cache()

    # ---- the eight model slots of the paper's family list in one call
    st = h.prepare(W.config_families(n=1_000_000))
    ms = h.timed([lambda: h.predict(st)], EX_ITERS, EX_WARM)[:, 0]
    ex["families_8_slots"] = dict(rows=st["w"].n_rows, ms=float(ms.mean()), predictions_per_s=float(st["w"].n_rows / (ms.mean() * 1e-3)),
                                  launches=2, max_rel_err_vs_oracle=parity_sample(h, st, 997),
                                  note="8 buckets, 8 model slots (GEMM, LM head, attention prefill / decode, RMSNorm, SiLU x Mul, "
                                       "RoPE, KV write), heads 12->128->128->1")
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
    # the Tier-A activation and output options on cfg2
    st = h.prepare(W.config2())
    h.ctx.set_gelu_mode(1)
    ms = h.timed([lambda: h.predict(st)], EX_ITERS, EX_WARM)[:, 0]
    h.ctx.set_gelu_mode(0)
    ex["cfg2_gelu_mode1"] = dict(ms=float(ms.mean()), predictions_per_s=float(st["w"].n_rows / (ms.mean() * 1e-3)),
                                 note="Tier-A kernel only; packed bf16x2 GELU arithmetic (not the default: slower, DESIGN.md §5)")
    for f in st["w"].heads:
        h.ctx.set_head_output(f, h.B.KS_HEAD_LOG_ETA)
    ms = h.timed([lambda: h.predict(st)], EX_ITERS, EX_WARM)[:, 0]
    ex["cfg2_log_eta_heads"] = dict(ms=float(ms.mean()), predictions_per_s=float(st["w"].n_rows / (ms.mean() * 1e-3)),
                                    note="heads read as log eta (PAPER.md:199): same kernel")
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
    # NEXT-1: density-routed Tier B on cfg3's 4M queries (grid inside the hull, 12->128->128->1 heads outside)
    st = h.prepare(W.config3(routed=True))
    ms = h.timed([lambda: h.predict(st)], EX_ITERS, EX_WARM)[:, 0]
    ex["cfg3_tierB_routed"] = dict(ms=float(ms.mean()), predictions_per_s=float(st["w"].n_rows / (ms.mean() * 1e-3)),
                                   launches=2, max_rel_err_vs_oracle=parity_sample(h, st, 1009),
                                   note="1 Tier-B pass that lists the out-of-hull rows + 1 Tier-A pass over the lists")
    del st
    torch.cuda.empty_cache()
    # SURVEY.md §8(d) caveat (i): cfg 3's kernel lasts ~25 us and cfg 4a's attention bucket 16 us (launch ramp,
    # 128 KiB grid staging per CTA); the same kernels at 16x / 8x the row count show the steady rate
    if not PROFILE:
        st = h.prepare(W.config3(n=16 * 4_194_304))
        ex["asymptotic_cfg3_tierB_x16"] = predict_all_roofline(h, st, peaks, iters=3)
        del st
        torch.cuda.empty_cache()
        attn = next(b for b in w4.buckets if b.family == W.FAM_ATTN)
        big = W.Bucket(W.FAM_ATTN, [np.tile(c, 8) for c in attn.cols], dtype_bytes=attn.dtype_bytes, hq=attn.hq,
                       hkv=attn.hkv, head_dim=attn.head_dim)
        w8 = W.Workload("cfg4a_attention_x8", [big], w4.specs, W.TIER_NONE)
        st = h.prepare_rows(w8)
        ex["asymptotic_cfg4a_attention_x8"] = dict(stream=stream_roofline(h, st, peaks, iters=3))
        del st
        torch.cuda.empty_cache()
    del w4
    ex["sim_closed_loop"] = sim_extras(h)
    return ex


def sim_extras(h):
    """NEXT-4: the closed simulation loop (host schedulers + one pass of the GPU path per iteration):
    256 what-if replicas x 200 requests each; wall-clock throughput of ks_sim_run (latency-bound: every
    iteration waits for its step times before the next batches can be formed)."""
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
    n_dev = torch.cuda.device_count()
    shared_gpu = world > n_dev                    # more ranks than GPUs: a functional check on one GPU, never a result
    dist = None
    if world > 1:
        import torch.distributed as dist
        if shared_gpu:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev_index = local % n_dev
    peaks = load_peaks()
    h = Harness(dev_index)
    h.red_dev = "cpu" if (dist is None or shared_gpu) else h.dev
    strong = args.scaling == "strong" and world > 1
    w_full = W.config5(seed=4 if strong else S.shard_seed(4, rank))
    w = S.shard_specs(w_full, rank, world) if strong else w_full   # strong: this rank's share of the 64 spec vectors
    st = h.prepare(w)
    K, Wm = args.steps, max(args.warmup, 3)
    if args.profile:                               # ncu capture mode: few launches, no numbers reported
        global EX_ITERS, EX_WARM, PROFILE
        EX_ITERS, EX_WARM, Wm, PROFILE = 1, 1, args.warmup, True
    n_cfg = st["n_cfg"]
    spec0, _ = S.shard_range(len(w_full.specs), rank, world) if strong else (0, 0)
    tot_all = torch.zeros((len(w_full.specs), n_cfg), dtype=torch.float32, device=h.red_dev) if strong else None

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def step():
        h.predict(st)
        h.compose(st)

    def exchange():
        """strong scaling: the path's one exchange step — the per-configuration totals of all shards (kilobytes)."""
        tot_all.zero_()
        tot_all[spec0:spec0 + st["ns"]] = st["tot"][:, :n_cfg].to(h.red_dev)
        S.allreduce_cfg_totals(tot_all, dist)

    # warm-up, then the timed region: K steps, barrier + synchronize on both sides
    h.timed([step], 1, Wm)
    launches0 = h.ctx.launch_count()
    sampler = ClockSampler(dev_index)
    barrier()
    sampler.start()
    t_wall0 = time.perf_counter()
    # one CUDA-event pair around each whole step (predict + compose back to back, as a caller issues them: the step
    # kernel is launched programmatically dependent on the prediction kernel, and an event between the two would
    # serialise that), L2 flushed before every step outside the event pair
    step_ms = h.timed([step], K, 0)
    t_x = 0.0
    if strong:                                     # after the K steps: totals of the last step meet once per step's worth
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        exchange()
        t_x = (time.perf_counter() - t0) * K       # charged K times: a caller exchanges after every step
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    launches = h.ctx.launch_count() - launches0
    total_s = S.max_over_ranks(float(step_ms.sum()) * 1e-3 + t_x, dist, h.red_dev)      # device time, max over ranks
    n_pred_rank = w.n_rows * st["ns"]
    value = (w_full.n_rows * len(w_full.specs) if strong else world * n_pred_rank) * K / total_s
    # per-kernel split for the roofline (not part of `value`): a few steps with an event between the two calls
    ms = h.timed([lambda: h.predict(st), lambda: h.compose(st)], min(K, 10), 0)
    worst = parity_sample(h, st, 4099) if rank == 0 else None
    del st
    torch.cuda.empty_cache()
    # end to end through the C ABI with HOST (pinned) buffers
    e2e = e2e_measure(h, w, max(1, min(K, 10)), world, dist)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    head = next(iter(w.heads.values()))
    kernel_ms = float(ms[:, 0].mean())
    tf = FLOPS_PER_PRED[(head.n_in, head.h1)] * n_pred_rank / (kernel_ms * 1e-3) / 1e12
    roofline = tensor_roofline("ks_mlp_ws256_kernel<32>", head.n_in, head.h1, n_pred_rank, kernel_ms, peaks["bf16_sustained"],
                               f"bf16 sustained (a {kernel_ms:.0f} ms kernel inside a long step), {peaks['source']}",
                               "cfg5_mlp_bytes_per_launch",
                               dict(frac_of_burst_peak=tf / peaks["bf16"], compose_ms=float(ms[:, 1].mean()),
                                    step_ms=float(step_ms.mean()), share_of_step=float(kernel_ms / ms.sum(axis=1).mean())))
    tanh_per_s = 2 * head.h1 * n_pred_rank / (kernel_ms * 1e-3)
    mufu_peak = 16 * torch.cuda.get_device_properties(dev_index).multi_processor_count * (clocks.get("sm_max_mhz") or 1965) * 1e6
    roofline_alu = dict(bound="alu", kernel=roofline["kernel"], achieved=tanh_per_s / 1e12, peak=mufu_peak / 1e12,
                        unit="Ttanh/s", frac=tanh_per_s / mufu_peak,
                        note="MUFU.TANH evaluations; peak = 16 lanes/clk/SM x SMs x max SM clock (the clock under this load is lower)")
    shard_note = "single GPU" if world == 1 else ("64 spec vectors split over the ranks, totals all-reduced" if strong
                                                  else "every rank its own seeded workload")
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=K, warmup=Wm,
                ms_per_step=1e3 * total_s / K, higher_is_better=True, scaling="strong" if strong else "weak", vs_baseline=None,
                dtype="bf16", data="synthetic",
                config=dict(workload=CFG5_NAME, tier="A", n_steps=w.n_steps, n_cfg=int(w.cfg_off.shape[0]) - 1,
                            rows_per_gpu=w.n_rows, specs_per_gpu=len(w.specs), predictions_per_gpu_per_step=n_pred_rank,
                            sharding=shard_note,
                            l2="flushed before every step (256 MiB write, outside the event pairs); a step also writes 1.07 GB of "
                               "latencies, 8x the L2",
                            timing="one CUDA-event pair on the ctx stream around predict + compose of every step"),
                clocks=clocks, e2e=e2e, gpu_launches=int(launches), roofline=roofline, roofline_alu=roofline_alu,
                max_rel_err_vs_oracle=worst, wall_s_timed_region=t_wall)
    if shared_gpu:
        line["shared_gpu"] = f"{world} ranks on {n_dev} GPU(s): functional check only, not a scaling result"
    if world == 1:
        if not args.no_extras:
            line["extras"] = run_extras(h, peaks)
        stride = 65536 if args.profile else args.cpu_stride
        rate, n, dt = oracle_sample_rate(w_full, stride, oracle_models(w_full))
        line["cpu_baseline"] = dict(value=rate, unit=UNIT, cores=1, kind="oracle", host=host_info(),
                                    sample=f"every {stride}th row of each cfg5 bucket x 64 specs ({n} predictions, {dt:.1f} s), "
                                           "Tier A + Eq. 4 composition, gcc -O2 single thread")
        if not args.profile:
            line["cpu_baseline"]["all_cores"] = oracle_all_cores("cfg5", stride)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def relaunch_under_torchrun(args) -> int:
    """`--gpus N` without a launcher: start N ranks of this script on this node (127.0.0.1 rendezvous)."""
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--scaling", choices=["weak", "strong"], default="weak")
    ap.add_argument("--no-extras", action="store_true", help="skip the other configs' blocks")
    ap.add_argument("--profile", action="store_true", help="ncu capture mode: one iteration of everything")
    ap.add_argument("--cpu-stride", type=int, default=1024, help="oracle baseline samples every n-th row (x 64 specs)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(relaunch_under_torchrun(args))
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
