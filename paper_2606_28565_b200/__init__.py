"""paper_2606_28565_b200 — B200-native batched kernel-latency prediction (KernelSight-LM hot path).

csrc/      hand-written sm_100a CUDA kernels + the C ABI (include/ks.h) -> libks.so
binding    ctypes binding with the C entry points' names (argument marshalling only)
driver     thin host driver (device memory via torch, model loading)
sharding   step-range / spec split of a workload over ranks and the one reduction that crosses them

The seeded synthetic inputs live OUTSIDE this package, in the top-level ``workloads`` package: it is the one
module the CPU oracle and this package both import, and it holds none of the method's arithmetic.
"""
import os as _os
import sys as _sys

_ROOT = _os.path.dirname(_os.path.dirname(_os.path.abspath(__file__)))
if _ROOT not in _sys.path:          # ``workloads`` sits beside this package at the repository root
    _sys.path.insert(0, _ROOT)

__all__ = ["binding", "driver", "build", "sharding"]
