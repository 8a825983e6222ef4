"""paper_2606_28565_b200 — B200-native batched kernel-latency prediction (KernelSight-LM hot path).

csrc/      hand-written sm_100a CUDA kernels + the C ABI (include/ks.h) -> libks.so
binding    ctypes binding with the C entry points' names (argument marshalling only)
driver     thin host driver (device memory via torch, model loading)
workloads  seeded synthetic inputs for the five BASELINE.json configs (no method arithmetic)
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "binding", "driver", "build"]
