"""ctypes wrapper around the CPU oracle (oracle/ks_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  Never imported by the
product package ``paper_2606_28565_b200``; imports nothing from its CUDA path
(only the shared, arithmetic-free ``workloads`` dataclasses are accepted as inputs).
Argument marshalling only — all arithmetic is in the C file.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ks_oracle.c")
_HDR = os.path.join(_HERE, "ks_oracle.h")
_LIB = os.path.join(_HERE, "libks_oracle.so")
MAX_COLS = 10


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (as it stands; never tuned)."""
    stale = (not os.path.exists(_LIB)) or any(
        os.path.getmtime(p) > os.path.getmtime(_LIB) for p in (_SRC, _HDR))
    if force or stale:
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


class Spec(C.Structure):
    _fields_ = [("peak_flops", C.c_double), ("peak_bw", C.c_double), ("n_sm", C.c_int64),
                ("ctas_per_sm", C.c_int64), ("tile_m", C.c_int64), ("tile_n", C.c_int64),
                ("ew_elems_per_cta", C.c_int64), ("l2_bytes", C.c_double), ("t0", C.c_double),
                ("ar_alpha0", C.c_double), ("ar_beta_eff", C.c_double)]


class Desc(C.Structure):
    _fields_ = [("family", C.c_int), ("v", C.c_int64 * MAX_COLS), ("s", C.c_int64),
                ("hq", C.c_int64), ("hkv", C.c_int64), ("d", C.c_int64)]


class Roof(C.Structure):
    _fields_ = [("F", C.c_double), ("Y", C.c_double), ("B", C.c_int64), ("W", C.c_int64),
                ("u", C.c_double), ("t_comp", C.c_double), ("t_mem", C.c_double), ("t_roof", C.c_double)]


class HeadC(C.Structure):
    _fields_ = [("n_in", C.c_int), ("h1", C.c_int), ("h2", C.c_int),
                ("W1", C.POINTER(C.c_double)), ("b1", C.POINTER(C.c_double)),
                ("W2", C.POINTER(C.c_double)), ("b2", C.POINTER(C.c_double)),
                ("w3", C.POINTER(C.c_double)), ("b3", C.c_double), ("log_eta", C.c_int)]


class GridC(C.Structure):
    _fields_ = [("dims", C.c_int64 * 3), ("lo", C.c_double * 3), ("hi", C.c_double * 3),
                ("values", C.POINTER(C.c_double))]


class StepParams(C.Structure):
    _fields_ = [("c_disp", C.c_double), ("floor_l", C.c_double), ("c_ovl", C.c_double),
                ("c_tail", C.c_double), ("body_scale", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.kso_bf16.restype = C.c_double
        L.kso_bf16.argtypes = [C.c_double]
        L.kso_gelu.restype = C.c_double
        L.kso_gelu.argtypes = [C.c_double]
        L.kso_sigmoid.restype = C.c_double
        L.kso_sigmoid.argtypes = [C.c_double]
        L.kso_eta_from_log.restype = C.c_double
        L.kso_eta_from_log.argtypes = [C.c_double]
        L.kso_head_e.restype = C.c_double
        L.kso_head_e.argtypes = [C.POINTER(HeadC), C.POINTER(C.c_double)]
        L.kso_bounded_e.restype = C.c_double
        L.kso_bounded_e.argtypes = [C.POINTER(BoundedC), C.POINTER(C.c_double), C.c_int64]
        L.kso_predict_batch_bounded.restype = C.c_int
        L.kso_predict_batch_bounded.argtypes = [C.c_int, C.c_int64, C.POINTER(C.POINTER(C.c_double)), C.c_int,
                                                C.c_int64, C.c_int64, C.c_int64, C.c_int64, C.POINTER(Spec), C.c_int,
                                                C.POINTER(BoundedC), C.POINTER(C.c_double), C.POINTER(C.c_int64),
                                                C.POINTER(C.c_int64), C.POINTER(C.c_double)]
        L.kso_ensemble_e.restype = C.c_double
        L.kso_ensemble_e.argtypes = [C.POINTER(HeadC), C.c_int, C.POINTER(C.c_double)]
        L.kso_predict_batch_ensemble.restype = C.c_int
        L.kso_predict_batch_ensemble.argtypes = [C.c_int, C.c_int64, C.POINTER(C.POINTER(C.c_double)), C.c_int,
                                                 C.c_int64, C.c_int64, C.c_int64, C.c_int64, C.POINTER(Spec), C.c_int,
                                                 C.POINTER(HeadC), C.c_int, C.POINTER(C.c_double),
                                                 C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_double)]
        L.kso_predict_batch_routed.restype = C.c_int
        L.kso_predict_batch_routed.argtypes = [C.c_int, C.c_int64, C.POINTER(C.POINTER(C.c_double)), C.c_int,
                                               C.c_int64, C.c_int64, C.c_int64, C.c_int64, C.POINTER(Spec), C.c_int,
                                               C.POINTER(GridC), C.POINTER(HeadC), C.POINTER(BoundedC),
                                               C.POINTER(C.c_double), C.POINTER(C.c_int64), C.POINTER(C.c_int64),
                                               C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        L.kso_allreduce.restype = C.c_double
        L.kso_allreduce.argtypes = [C.c_int64, C.c_int64, C.POINTER(Spec)]
        L.kso_attn_pairs.restype = C.c_int64
        L.kso_attn_pairs.argtypes = [C.c_int64, C.c_int64]
        L.kso_wave.restype = None
        L.kso_wave.argtypes = [C.c_int64, C.c_int64, C.POINTER(C.c_int64), C.POINTER(C.c_double)]
        L.kso_roofline.restype = None
        L.kso_roofline.argtypes = [C.POINTER(Desc), C.POINTER(Spec), C.POINTER(Roof)]
        L.kso_features.restype = None
        L.kso_features.argtypes = [C.POINTER(Desc), C.POINTER(Spec), C.POINTER(Roof), C.c_int,
                                   C.POINTER(C.c_double)]
        L.kso_mlp_z.restype = C.c_double
        L.kso_mlp_z.argtypes = [C.POINTER(HeadC), C.POINTER(C.c_double)]
        L.kso_trilinear.restype = C.c_double
        L.kso_trilinear.argtypes = [C.POINTER(GridC), C.POINTER(C.c_double)]
        L.kso_predict_one.restype = C.c_double
        L.kso_predict_one.argtypes = [C.POINTER(Desc), C.POINTER(Spec), C.c_int, C.POINTER(HeadC),
                                      C.POINTER(GridC), C.POINTER(Roof), C.POINTER(C.c_double)]
        L.kso_predict_batch.restype = C.c_int
        L.kso_predict_batch.argtypes = [C.c_int, C.c_int64, C.POINTER(C.POINTER(C.c_double)), C.c_int,
                                        C.c_int64, C.c_int64, C.c_int64, C.c_int64, C.POINTER(Spec),
                                        C.c_int, C.c_int, C.POINTER(HeadC), C.POINTER(GridC),
                                        C.POINTER(C.c_double), C.POINTER(C.c_int64),
                                        C.POINTER(C.c_int64), C.POINTER(C.c_double)]
        L.kso_compose.restype = None
        L.kso_compose.argtypes = [C.c_int, C.POINTER(C.POINTER(C.c_double)),
                                  C.POINTER(C.POINTER(C.c_int64)), C.c_int64, C.POINTER(StepParams),
                                  C.POINTER(C.c_int64), C.c_int64, C.POINTER(C.c_double),
                                  C.POINTER(C.c_double)]
        L.kso_compose_weighted.restype = None
        L.kso_compose_weighted.argtypes = [C.c_int, C.POINTER(C.POINTER(C.c_double)), C.POINTER(C.POINTER(C.c_int64)),
                                           C.POINTER(C.POINTER(C.c_int64)), C.c_int64, C.POINTER(StepParams),
                                           C.POINTER(C.c_int64), C.c_int64, C.POINTER(C.c_double),
                                           C.POINTER(C.c_double)]
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_int64))


def make_spec(s: dict) -> Spec:
    return Spec(float(s["peak_flops"]), float(s["peak_bw"]), int(s["n_sm"]), int(s["ctas_per_sm"]),
                int(s["tile_m"]), int(s["tile_n"]), int(s["ew_elems_per_cta"]), float(s["l2_bytes"]),
                float(s["t0"]), float(s.get("ar_alpha0", 0.0)), float(s.get("ar_beta_eff", 1.0)))


def make_desc(family: int, v: Sequence[int], s: int = 2, hq: int = 0, hkv: int = 0, d: int = 0) -> Desc:
    arr = (C.c_int64 * MAX_COLS)(*([int(x) for x in v] + [0] * (MAX_COLS - len(v))))
    return Desc(int(family), arr, int(s), int(hq), int(hkv), int(d))


def bf16(x):
    """Elementwise RNE rounding to bf16 precision (returns float64 array)."""
    L = lib()
    a = np.asarray(x, dtype=np.float64)
    out = np.array([L.kso_bf16(float(v)) for v in a.reshape(-1)], dtype=np.float64)
    return out.reshape(a.shape)


class Head:
    """Holds bf16-rounded double copies of a head's weights (the rounding the library applies at load)."""

    def __init__(self, h, round_weights: bool = True):
        r = bf16 if round_weights else (lambda a: np.asarray(a, np.float64))
        self.W1 = np.ascontiguousarray(r(h.W1))
        self.W2 = np.ascontiguousarray(r(h.W2))
        self.w3 = np.ascontiguousarray(r(h.w3))
        self.b1 = np.ascontiguousarray(h.b1, dtype=np.float64)
        self.b2 = np.ascontiguousarray(h.b2, dtype=np.float64)
        self.c = HeadC(int(h.n_in), int(h.h1), int(h.h2), _dp(self.W1), _dp(self.b1), _dp(self.W2),
                       _dp(self.b2), _dp(self.w3), float(h.b3), int(getattr(h, "out_mode", 0)))


class Ensemble:
    """k MLP members of one shape ("small MLP ensemble"; Q17): e = mean of sigmoid(z_m)."""

    def __init__(self, members, round_weights: bool = True):
        self.heads = [Head(m, round_weights) for m in members]
        self.k = len(self.heads)
        self.c = (HeadC * self.k)(*[h.c for h in self.heads])


class BoundedC(C.Structure):
    _fields_ = [("n_in", C.c_int), ("w_gamma", C.POINTER(C.c_double)), ("w_alpha", C.POINTER(C.c_double)),
                ("b_gamma", C.c_double), ("b_alpha", C.c_double)]


class Bounded:
    """The bounded analytical head's weights as the library receives them (fp32 values, held as double)."""

    def __init__(self, h):
        self.wg = np.ascontiguousarray(np.asarray(h.w_gamma, np.float32), dtype=np.float64)
        self.wa = np.ascontiguousarray(np.asarray(h.w_alpha, np.float32), dtype=np.float64)
        self.c = BoundedC(int(h.n_in), _dp(self.wg), _dp(self.wa), float(np.float32(h.b_gamma)),
                          float(np.float32(h.b_alpha)))


class Grid:
    def __init__(self, g):
        self.values = np.ascontiguousarray(g.values, dtype=np.float64)
        self.c = GridC((C.c_int64 * 3)(*[int(x) for x in g.dims]),
                       (C.c_double * 3)(*[float(x) for x in g.lo_log2]),
                       (C.c_double * 3)(*[float(x) for x in g.hi_log2]), _dp(self.values))


def roofline(desc: Desc, spec: Spec) -> Roof:
    r = Roof()
    lib().kso_roofline(C.byref(desc), C.byref(spec), C.byref(r))
    return r


def wave(B: int, S: int):
    W = C.c_int64()
    u = C.c_double()
    lib().kso_wave(int(B), int(S), C.byref(W), C.byref(u))
    return W.value, u.value


def features(desc: Desc, spec: Spec, n_in: int) -> np.ndarray:
    r = roofline(desc, spec)
    x = np.zeros(n_in, np.float64)
    lib().kso_features(C.byref(desc), C.byref(spec), C.byref(r), int(n_in), _dp(x))
    return x


def eta_from_log(z: float) -> float:
    return float(lib().kso_eta_from_log(float(z)))


def head_e(head: Head, x) -> float:
    x = np.ascontiguousarray(x, dtype=np.float64)
    return float(lib().kso_head_e(C.byref(head.c), _dp(x)))


def mlp_z(head: Head, x) -> float:
    x = np.ascontiguousarray(x, dtype=np.float64)
    return lib().kso_mlp_z(C.byref(head.c), _dp(x))


def trilinear(grid: Grid, v) -> float:
    v = np.ascontiguousarray(v, dtype=np.float64)
    return lib().kso_trilinear(C.byref(grid.c), _dp(v))


def predict_one(desc: Desc, spec: Spec, tier: int, head: Optional[Head] = None,
                grid: Optional[Grid] = None):
    r = Roof()
    e = C.c_double()
    t = lib().kso_predict_one(C.byref(desc), C.byref(spec), int(tier), C.byref(head.c) if head else None,
                              C.byref(grid.c) if grid else None, C.byref(r), C.byref(e))
    return t, r, e.value


def bounded_e(bh: "Bounded", x, W: int) -> float:
    xa = np.ascontiguousarray(x, dtype=np.float64)
    return float(lib().kso_bounded_e(C.byref(bh.c), _dp(xa), int(W)))


def ensemble_e(ens: "Ensemble", x) -> float:
    xa = np.ascontiguousarray(x, dtype=np.float64)
    return float(lib().kso_ensemble_e(ens.c, ens.k, _dp(xa)))


def predict_bucket(bucket, specs: Sequence[dict], tier: int, head: Optional[Head] = None,
                   grid: Optional[Grid] = None, rows: Optional[np.ndarray] = None,
                   bounded: Optional["Bounded"] = None, ensemble: Optional["Ensemble"] = None):
    """Run the oracle over one workloads.Bucket (optionally only ``rows``) for every spec.

    Returns dict(lat [n_specs,n] f64, tiles i64, waves i64, troof f64).
    """
    cols = [np.ascontiguousarray(c if rows is None else c[rows], dtype=np.float64) for c in bucket.cols]
    n = int(cols[0].shape[0]) if cols else 0
    ns = len(specs)
    sp = (Spec * ns)(*[make_spec(s) for s in specs])
    colp = (C.POINTER(C.c_double) * len(cols))(*[_dp(c) for c in cols])
    lat = np.zeros((ns, n), np.float64)
    troof = np.zeros((ns, n), np.float64)
    tiles = np.zeros((ns, n), np.int64)
    waves = np.zeros((ns, n), np.int64)
    if tier == 3:                               # density-routed Tier B: grid inside the hull, head outside
        routed = np.zeros(n, np.int64)
        rc = lib().kso_predict_batch_routed(int(bucket.family), n, colp, len(cols), int(bucket.dtype_bytes),
                                            int(bucket.hq), int(bucket.hkv), int(bucket.head_dim), sp, ns,
                                            C.byref(grid.c) if grid else None, C.byref(head.c) if head else None,
                                            C.byref(bounded.c) if bounded else None, _dp(lat), _ip(tiles),
                                            _ip(waves), _dp(troof), _ip(routed))
        if rc != 0:
            raise ValueError("kso_predict_batch_routed: bad arguments")
        return dict(lat=lat, tiles=tiles, waves=waves, troof=troof, routed=routed)
    if ensemble is not None and tier == 1:     # Tier A with an MLP ensemble for this family
        rc = lib().kso_predict_batch_ensemble(int(bucket.family), n, colp, len(cols), int(bucket.dtype_bytes),
                                              int(bucket.hq), int(bucket.hkv), int(bucket.head_dim), sp, ns,
                                              ensemble.c, ensemble.k, _dp(lat), _ip(tiles), _ip(waves), _dp(troof))
        if rc != 0:
            raise ValueError("kso_predict_batch_ensemble: bad arguments")
        return dict(lat=lat, tiles=tiles, waves=waves, troof=troof)
    if bounded is not None and tier == 1:      # Tier A with the bounded analytical head for this family
        rc = lib().kso_predict_batch_bounded(int(bucket.family), n, colp, len(cols), int(bucket.dtype_bytes),
                                             int(bucket.hq), int(bucket.hkv), int(bucket.head_dim), sp, ns,
                                             C.byref(bounded.c), _dp(lat), _ip(tiles), _ip(waves), _dp(troof))
        if rc != 0:
            raise ValueError("kso_predict_batch_bounded: bad arguments")
        return dict(lat=lat, tiles=tiles, waves=waves, troof=troof)
    rc = lib().kso_predict_batch(int(bucket.family), n, colp, len(cols), int(bucket.dtype_bytes),
                                 int(bucket.hq), int(bucket.hkv), int(bucket.head_dim), sp, ns, int(tier),
                                 C.byref(head.c) if head else None, C.byref(grid.c) if grid else None,
                                 _dp(lat), _ip(tiles), _ip(waves), _dp(troof))
    if rc != 0:
        raise ValueError("kso_predict_batch: bad arguments")
    return dict(lat=lat, tiles=tiles, waves=waves, troof=troof)


def compose(lats: Sequence[np.ndarray], step_offs: Sequence[np.ndarray], n_steps: int, params: dict,
            cfg_off: np.ndarray, mults: Optional[Sequence[Optional[np.ndarray]]] = None):
    """lats[b]: [n_b] float64 for ONE spec; returns (step_lat [n_steps], cfg_lat [n_cfg]).
    mults[b] (optional): per-row multiplicities of the layer-homogeneous form."""
    nb = len(lats)
    la = [np.ascontiguousarray(x, dtype=np.float64) for x in lats]
    so = [np.ascontiguousarray(x, dtype=np.int64) for x in step_offs]
    co = np.ascontiguousarray(cfg_off, dtype=np.int64)
    n_cfg = co.shape[0] - 1
    lp = (C.POINTER(C.c_double) * nb)(*[_dp(x) for x in la])
    sp = (C.POINTER(C.c_int64) * nb)(*[_ip(x) for x in so])
    p = StepParams(float(params["c_disp"]), float(params["floor_l"]), float(params["c_ovl"]),
                   float(params["c_tail"]), float(params["body_scale"]))
    step_lat = np.zeros(n_steps, np.float64)
    cfg_lat = np.zeros(max(n_cfg, 0), np.float64)
    if mults is not None and any(m is not None for m in mults):
        ma = [None if m is None else np.ascontiguousarray(m, dtype=np.int64) for m in mults]
        mp = (C.POINTER(C.c_int64) * nb)(*[_ip(x) if x is not None else C.POINTER(C.c_int64)() for x in ma])
        lib().kso_compose_weighted(nb, lp, mp, sp, int(n_steps), C.byref(p), _ip(co), int(n_cfg), _dp(step_lat),
                                   _dp(cfg_lat))
        return step_lat, cfg_lat
    lib().kso_compose(nb, lp, sp, int(n_steps), C.byref(p), _ip(co), int(n_cfg), _dp(step_lat), _dp(cfg_lat))
    return step_lat, cfg_lat
