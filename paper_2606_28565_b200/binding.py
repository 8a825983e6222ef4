"""Thin ctypes binding over libks (include/ks.h).  Argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; this module converts numpy
arrays / torch tensors into pointers and structs.  PyTorch is used for device memory and streams
only.  There is no CPU fallback: if libks.so is missing or no sm_100 device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libks.so")

KS_OK, KS_EINVAL, KS_ENOMEM, KS_ECUDA, KS_ESTATE, KS_EUNSUPPORTED, KS_ELIMIT = range(7)
KS_STATIC_ROUTE_MAX_ROWS = 1 << 20
KS_FAM_GEMM, KS_FAM_GROUPED_GEMM, KS_FAM_ATTN, KS_FAM_ELEMWISE = range(4)
KS_TIER_NONE, KS_TIER_A, KS_TIER_B = range(3)
KS_SLOT_FAMILY, KS_MAX_MODEL_SLOTS = -1, 16
KS_HEAD_UTILISATION, KS_HEAD_LOG_ETA = 0, 1
KS_COL_I32, KS_COL_F32 = 0, 1
KS_MEM_DEVICE, KS_MEM_HOST = 0, 1
KS_MAX_COLS, KS_MAX_BATCHES = 10, 8
EXPORTS = ["ks_create", "ks_load_heads", "ks_load_head_ensemble", "ks_load_bounded_head", "ks_load_grid", "ks_set_head_output",
           "ks_predict_kernels", "ks_predict_routed_static", "ks_compose_steps",
           "ks_compose_steps_weighted",
           "ks_run_steps", "ks_sched_create", "ks_sched_add_requests", "ks_sched_add_prefixed_requests", "ks_sched_step", "ks_sched_commit",
           "ks_sched_results", "ks_sched_get_stats", "ks_sched_destroy", "ks_sim_run",
           "ks_get_launch_count", "ks_set_gelu_mode", "ks_destroy", "ks_status_string"]


class KsError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {status_string(status)}")


class ks_hw_spec(C.Structure):
    _fields_ = [("peak_flops", C.c_float), ("peak_bw", C.c_float), ("n_sm", C.c_int32),
                ("ctas_per_sm", C.c_int32), ("tile_m", C.c_int32), ("tile_n", C.c_int32),
                ("ew_elems_per_cta", C.c_int32), ("l2_bytes", C.c_float), ("t0", C.c_float),
                ("ar_alpha0", C.c_float), ("ar_beta_eff", C.c_float)]


class ks_desc_batch(C.Structure):
    _fields_ = [("family", C.c_int32), ("n", C.c_int32), ("col_dtype", C.c_int32), ("dtype_bytes", C.c_int32),
                ("n_cols", C.c_int32), ("attn_hq", C.c_int32), ("attn_hkv", C.c_int32),
                ("attn_head_dim", C.c_int32), ("cols", C.c_void_p * KS_MAX_COLS), ("model_slot", C.c_int32),
                ("mult", C.c_void_p)]


class ks_step_params(C.Structure):
    _fields_ = [("c_disp", C.c_float), ("floor_l", C.c_float), ("c_ovl", C.c_float), ("c_tail", C.c_float),
                ("body_scale", C.c_float)]


class ks_sched_config(C.Structure):
    _fields_ = [("max_num_batched_tokens", C.c_int32), ("max_num_seqs", C.c_int32), ("block_size", C.c_int32),
                ("num_blocks", C.c_int32), ("enable_prefix_cache", C.c_int32), ("disk_blocks", C.c_int32)]


class ks_model_desc(C.Structure):
    _fields_ = [(k, C.c_int32) for k in ("n_layers", "hidden", "ffn", "vocab", "hq", "hkv", "head_dim",
                                         "dtype_bytes", "tp", "fine_slots")]


class ks_sched_stats(C.Structure):
    _fields_ = [("n_steps", C.c_int64), ("tokens_scheduled", C.c_int64), ("n_preemptions", C.c_int64),
                ("gpu_hit_blocks", C.c_int64), ("disk_hit_blocks", C.c_int64), ("evictions", C.c_int64),
                ("n_requests", C.c_int32), ("n_finished", C.c_int32), ("n_running", C.c_int32),
                ("n_waiting", C.c_int32), ("free_blocks", C.c_int32), ("pad", C.c_int32)]


class ks_sim_stats(C.Structure):
    _fields_ = [("iterations", C.c_int64), ("steps", C.c_int64), ("rows", C.c_int64), ("kernel_instances", C.c_int64),
                ("schedule_s", C.c_double), ("enqueue_s", C.c_double), ("wait_s", C.c_double), ("commit_s", C.c_double)]


_lib = None


def load() -> C.CDLL:
    """dlopen libks.so (built in-tree by ``python -m paper_2606_28565_b200.build``). Fails loudly."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} not found: build the CUDA library first "
                           "(python -m paper_2606_28565_b200.build). There is no CPU fallback.")
    L = C.CDLL(LIB_PATH)
    vp, i32, fp = C.c_void_p, C.c_int, C.POINTER(C.c_float)
    L.ks_create.argtypes = [C.POINTER(vp), i32, vp]
    L.ks_load_heads.argtypes = [vp, i32, i32, i32, i32, fp, fp, fp, fp, fp, C.c_float]
    L.ks_load_head_ensemble.argtypes = [vp, i32, i32, i32, i32, fp, fp, fp, fp, fp, fp]
    L.ks_load_bounded_head.argtypes = [vp, i32, i32, fp, C.c_float, fp, C.c_float]
    L.ks_load_grid.argtypes = [vp, i32, C.POINTER(C.c_int32), fp, fp, fp]
    L.ks_set_head_output.argtypes = [vp, i32, i32]
    L.ks_predict_kernels.argtypes = [vp, C.POINTER(ks_desc_batch), i32, C.POINTER(ks_hw_spec), i32, i32, i32,
                                     C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
    L.ks_predict_routed_static.argtypes = [vp, C.POINTER(ks_desc_batch), i32, C.POINTER(ks_hw_spec), i32,
                                           C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
    L.ks_compose_steps.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(C.c_int32), i32, i32, i32,
                                   C.POINTER(ks_step_params), vp, i32, i32, vp, vp]
    L.ks_compose_steps_weighted.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(C.c_int32), i32,
                                            i32, i32, C.POINTER(ks_step_params), vp, i32, i32, vp, vp]
    L.ks_run_steps.argtypes = [vp, C.POINTER(ks_desc_batch), C.POINTER(vp), i32, C.POINTER(ks_hw_spec), i32, i32,
                               i32, C.POINTER(ks_step_params), vp, i32, i32, C.POINTER(vp), vp, vp]
    dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int32)
    L.ks_sched_create.argtypes = [C.POINTER(vp), C.POINTER(ks_sched_config)]
    L.ks_sched_add_requests.argtypes = [vp, i32, dp, ip, ip]
    L.ks_sched_add_prefixed_requests.argtypes = [vp, i32, dp, ip, ip, ip, ip]
    L.ks_sched_step.argtypes = [vp, C.c_double, C.c_int32, ip, ip, ip, ip, dp]
    L.ks_sched_commit.argtypes = [vp, C.c_double]
    L.ks_sched_results.argtypes = [vp, dp, dp, ip, ip]
    L.ks_sched_get_stats.argtypes = [vp, C.POINTER(ks_sched_stats)]
    L.ks_sched_destroy.argtypes = [vp]
    L.ks_sim_run.argtypes = [vp, C.POINTER(vp), dp, i32, C.POINTER(ks_model_desc), C.POINTER(ks_hw_spec), i32,
                             C.POINTER(ks_step_params), C.c_int64, ip, fp, C.c_int64, C.POINTER(C.c_int64),
                             C.POINTER(ks_sim_stats)]
    L.ks_get_launch_count.argtypes = [vp, C.POINTER(C.c_int64)]
    L.ks_set_gelu_mode.argtypes = [vp, i32]
    L.ks_destroy.argtypes = [vp]
    L.ks_status_string.argtypes = [i32]
    L.ks_status_string.restype = C.c_char_p
    for name in EXPORTS[:-1]:
        getattr(L, name).restype = C.c_int
    _lib = L
    return L


def status_string(s: int) -> str:
    return load().ks_status_string(int(s)).decode()


def _check(st: int, where: str):
    if st != KS_OK:
        raise KsError(st, where)


def _ptr(a) -> Optional[int]:
    """Address of a numpy array or torch tensor (None -> NULL)."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return int(a.data_ptr())


def _is_host(a) -> bool:
    return isinstance(a, np.ndarray) or (hasattr(a, "is_cuda") and not a.is_cuda)


def _ptr_array(items: Sequence) -> "C.Array":
    arr = (C.c_void_p * max(len(items), 1))()
    for i, it in enumerate(items):
        arr[i] = _ptr(it)
    return arr


def make_spec(s: dict) -> ks_hw_spec:
    return ks_hw_spec(float(s["peak_flops"]), float(s["peak_bw"]), int(s["n_sm"]), int(s["ctas_per_sm"]),
                      int(s["tile_m"]), int(s["tile_n"]), int(s["ew_elems_per_cta"]), float(s["l2_bytes"]),
                      float(s["t0"]), float(s.get("ar_alpha0", 0.0)), float(s.get("ar_beta_eff", 1.0)))


def make_batch(bucket) -> ks_desc_batch:
    """bucket: any object with family, cols (numpy arrays or torch tensors), dtype_bytes, hq, hkv, head_dim."""
    cols = list(bucket.cols)
    n = int(cols[0].shape[0]) if cols else 0
    dt = str(cols[0].dtype) if cols else "int32"
    if "float32" in dt:
        cd = KS_COL_F32
    elif "int32" in dt:
        cd = KS_COL_I32
    else:
        raise TypeError(f"descriptor columns must be int32 or float32, got {dt}")
    arr = (C.c_void_p * KS_MAX_COLS)()
    for i, c in enumerate(cols):
        if hasattr(c, "is_contiguous") and not c.is_contiguous():
            raise ValueError("descriptor columns must be contiguous")
        arr[i] = _ptr(c)
    mult = getattr(bucket, "mult", None)             # optional per-row multiplicities (int32)
    if mult is not None and "int32" not in str(mult.dtype):
        raise TypeError("multiplicities must be int32")
    slot = getattr(bucket, "model_slot", None)      # None = the slot numbered like the family
    return ks_desc_batch(int(bucket.family), n, cd, int(bucket.dtype_bytes), len(cols), int(bucket.hq),
                         int(bucket.hkv), int(bucket.head_dim), arr, KS_SLOT_FAMILY if slot is None else int(slot),
                         _ptr(mult) if mult is not None else None)


def make_step_params(p: dict) -> ks_step_params:
    return ks_step_params(float(p["c_disp"]), float(p["floor_l"]), float(p["c_ovl"]), float(p["c_tail"]),
                          float(p["body_scale"]))


class Context:
    """Owns one ks_ctx.  Method names mirror the C entry points."""

    def __init__(self, device: int = 0, stream: Optional[int] = None):
        self._h = C.c_void_p()
        self._lib = load()
        _check(self._lib.ks_create(C.byref(self._h), int(device), C.c_void_p(stream or 0)), "ks_create")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.ks_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- loading (the first argument of every loader is a model SLOT; slot = family for one model per family)
    def load_heads(self, family: int, head) -> None:
        f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
        W1, b1, W2, b2, w3 = f32(head.W1), f32(head.b1), f32(head.W2), f32(head.b2), f32(head.w3)
        fp = lambda a: a.ctypes.data_as(C.POINTER(C.c_float))
        _check(self._lib.ks_load_heads(self._h, int(family), int(head.n_in), int(head.h1), int(head.h2), fp(W1),
                                       fp(b1), fp(W2), fp(b2), fp(w3), float(head.b3)), "ks_load_heads")
        if int(getattr(head, "out_mode", KS_HEAD_UTILISATION)) != KS_HEAD_UTILISATION:
            self.set_head_output(family, int(head.out_mode))

    def set_head_output(self, slot: int, mode: int) -> None:
        _check(self._lib.ks_set_head_output(self._h, int(slot), int(mode)), "ks_set_head_output")

    def load_head_ensemble(self, family: int, members) -> None:
        """members: workloads.Head objects of one shape (n_in -> h -> h -> 1)."""
        m0 = members[0]
        if any((m.n_in, m.h1, m.h2) != (m0.n_in, m0.h1, m0.h1) for m in members):
            raise ValueError("ensemble members must share one shape n_in -> h -> h -> 1")
        st = lambda name: np.ascontiguousarray(np.stack([np.asarray(getattr(m, name), np.float32) for m in members]))
        W1, b1, W2, b2, w3 = st("W1"), st("b1"), st("W2"), st("b2"), st("w3")
        b3 = np.array([m.b3 for m in members], np.float32)
        fp = lambda a: a.ctypes.data_as(C.POINTER(C.c_float))
        _check(self._lib.ks_load_head_ensemble(self._h, int(family), int(m0.n_in), int(m0.h1), len(members), fp(W1),
                                               fp(b1), fp(W2), fp(b2), fp(w3), fp(b3)), "ks_load_head_ensemble")

    def load_bounded_head(self, family: int, head) -> None:
        wg = np.ascontiguousarray(head.w_gamma, dtype=np.float32)
        wa = np.ascontiguousarray(head.w_alpha, dtype=np.float32)
        fp = lambda a: a.ctypes.data_as(C.POINTER(C.c_float))
        _check(self._lib.ks_load_bounded_head(self._h, int(family), int(head.n_in), fp(wg), float(head.b_gamma),
                                              fp(wa), float(head.b_alpha)), "ks_load_bounded_head")

    def load_grid(self, family: int, grid) -> None:
        dims = np.ascontiguousarray(grid.dims, dtype=np.int32)
        lo = np.ascontiguousarray(grid.lo_log2, dtype=np.float32)
        hi = np.ascontiguousarray(grid.hi_log2, dtype=np.float32)
        vals = np.ascontiguousarray(grid.values, dtype=np.float32)
        fp = lambda a: a.ctypes.data_as(C.POINTER(C.c_float))
        _check(self._lib.ks_load_grid(self._h, int(family), dims.ctypes.data_as(C.POINTER(C.c_int32)), fp(lo),
                                      fp(hi), fp(vals)), "ks_load_grid")

    def set_gelu_mode(self, mode: int) -> None:
        _check(self._lib.ks_set_gelu_mode(self._h, int(mode)), "ks_set_gelu_mode")

    def launch_count(self) -> int:
        out = C.c_int64()
        _check(self._lib.ks_get_launch_count(self._h, C.byref(out)), "ks_get_launch_count")
        return out.value

    # ---- compute
    def predict_kernels(self, buckets: Sequence, specs: Sequence[dict], tier: int, latency: Sequence,
                        tiles: Optional[Sequence] = None, waves: Optional[Sequence] = None,
                        t_roof: Optional[Sequence] = None, space: Optional[int] = None) -> None:
        nb = len(buckets)
        batches = (ks_desc_batch * max(nb, 1))(*[make_batch(b) for b in buckets])
        sp = (ks_hw_spec * max(len(specs), 1))(*[make_spec(s) for s in specs])
        if space is None:
            space = KS_MEM_HOST if (nb and _is_host(latency[0])) else KS_MEM_DEVICE
        opt = lambda x: _ptr_array(x) if x is not None else None
        _check(self._lib.ks_predict_kernels(self._h, batches, nb, sp, len(specs), int(tier), int(space),
                                            _ptr_array(latency), opt(tiles), opt(waves), opt(t_roof)),
               "ks_predict_kernels")

    def predict_routed_static(self, buckets: Sequence, specs: Sequence[dict], latency: Sequence,
                              tiles: Optional[Sequence] = None, waves: Optional[Sequence] = None,
                              t_roof: Optional[Sequence] = None) -> None:
        """Density-routed prediction on device buffers with the row lists in the library's fixed device array:
        no allocation; at most KS_STATIC_ROUTE_MAX_ROWS routed rows per call (KS_ELIMIT beyond)."""
        nb = len(buckets)
        batches = (ks_desc_batch * max(nb, 1))(*[make_batch(b) for b in buckets])
        sp = (ks_hw_spec * max(len(specs), 1))(*[make_spec(s) for s in specs])
        opt = lambda x: _ptr_array(x) if x is not None else None
        _check(self._lib.ks_predict_routed_static(self._h, batches, nb, sp, len(specs), _ptr_array(latency),
                                                  opt(tiles), opt(waves), opt(t_roof)), "ks_predict_routed_static")

    def compose_steps(self, latency: Sequence, step_off: Sequence, batch_n: Sequence[int], n_steps: int,
                      n_specs: int, params: dict, cfg_off, n_cfg: int, step_latency, cfg_latency,
                      space: Optional[int] = None, mult: Optional[Sequence] = None) -> None:
        nb = len(latency)
        bn = (C.c_int32 * max(nb, 1))(*[int(x) for x in batch_n])
        p = make_step_params(params)
        if space is None:
            space = KS_MEM_HOST if _is_host(step_latency) else KS_MEM_DEVICE
        if mult is not None and any(m is not None for m in mult):
            _check(self._lib.ks_compose_steps_weighted(self._h, _ptr_array(latency), _ptr_array(mult),
                                                       _ptr_array(step_off), bn, nb, int(n_steps), int(n_specs),
                                                       C.byref(p), _ptr(cfg_off), int(n_cfg), int(space),
                                                       _ptr(step_latency), _ptr(cfg_latency)),
                   "ks_compose_steps_weighted")
            return
        _check(self._lib.ks_compose_steps(self._h, _ptr_array(latency), _ptr_array(step_off), bn, nb, int(n_steps),
                                          int(n_specs), C.byref(p), _ptr(cfg_off), int(n_cfg), int(space),
                                          _ptr(step_latency), _ptr(cfg_latency)), "ks_compose_steps")

    def run_steps(self, buckets: Sequence, step_off: Sequence, specs: Sequence[dict], tier: int, n_steps: int,
                  params: dict, cfg_off, n_cfg: int, step_latency, cfg_latency, latency: Optional[Sequence] = None,
                  space: Optional[int] = None) -> None:
        nb = len(buckets)
        batches = (ks_desc_batch * max(nb, 1))(*[make_batch(b) for b in buckets])
        sp = (ks_hw_spec * max(len(specs), 1))(*[make_spec(s) for s in specs])
        p = make_step_params(params)
        if space is None:
            space = KS_MEM_HOST if _is_host(step_latency) else KS_MEM_DEVICE
        _check(self._lib.ks_run_steps(self._h, batches, _ptr_array(step_off), nb, sp, len(specs), int(tier),
                                      int(n_steps), C.byref(p), _ptr(cfg_off), int(n_cfg), int(space),
                                      _ptr_array(latency) if latency is not None else None, _ptr(step_latency),
                                      _ptr(cfg_latency)), "ks_run_steps")


class Scheduler:
    """One replica's serving scheduler (ks_sched_*): host logic, needs no GPU.  Marshalling only."""

    def __init__(self, max_num_batched_tokens: int, max_num_seqs: int, block_size: int, num_blocks: int,
                 enable_prefix_cache: bool = False, disk_blocks: int = 0):
        self._lib = load()
        self._h = C.c_void_p()
        cfg = ks_sched_config(int(max_num_batched_tokens), int(max_num_seqs), int(block_size), int(num_blocks),
                              int(bool(enable_prefix_cache)), int(disk_blocks))
        _check(self._lib.ks_sched_create(C.byref(self._h), C.byref(cfg)), "ks_sched_create")
        self.cap = int(max_num_seqs)
        self.n_requests = 0
        self._req = np.zeros(self.cap, np.int32)
        self._new = np.zeros(self.cap, np.int32)
        self._hist = np.zeros(self.cap, np.int32)

    def add_requests(self, arrival, prompt_len, max_new, prefix_id=None, prefix_len=None) -> None:
        a = np.ascontiguousarray(arrival, dtype=np.float64)
        p = np.ascontiguousarray(prompt_len, dtype=np.int32)
        o = np.ascontiguousarray(max_new, dtype=np.int32)
        if not (a.shape == p.shape == o.shape and a.ndim == 1):
            raise ValueError("arrival, prompt_len, max_new: 1-D arrays of one length")
        ip = C.POINTER(C.c_int32)
        if prefix_id is None and prefix_len is None:
            _check(self._lib.ks_sched_add_requests(self._h, a.shape[0], a.ctypes.data_as(C.POINTER(C.c_double)),
                                                   p.ctypes.data_as(ip), o.ctypes.data_as(ip)), "ks_sched_add_requests")
        else:
            pi = np.ascontiguousarray(prefix_id, dtype=np.int32)
            pl = np.ascontiguousarray(prefix_len, dtype=np.int32)
            if not (pi.shape == pl.shape == a.shape):
                raise ValueError("prefix_id, prefix_len: one entry per request")
            _check(self._lib.ks_sched_add_prefixed_requests(self._h, a.shape[0], a.ctypes.data_as(C.POINTER(C.c_double)),
                                                            p.ctypes.data_as(ip), o.ctypes.data_as(ip), pi.ctypes.data_as(ip),
                                                            pl.ctypes.data_as(ip)), "ks_sched_add_prefixed_requests")
        self.n_requests += int(a.shape[0])

    def step(self, now: float):
        """-> (list of (request, n_new, hist), next_arrival)"""
        n = C.c_int32()
        nxt = C.c_double()
        ip = C.POINTER(C.c_int32)
        _check(self._lib.ks_sched_step(self._h, float(now), self.cap, C.byref(n), self._req.ctypes.data_as(ip),
                                       self._new.ctypes.data_as(ip), self._hist.ctypes.data_as(ip), C.byref(nxt)),
               "ks_sched_step")
        k = n.value
        return list(zip(self._req[:k].tolist(), self._new[:k].tolist(), self._hist[:k].tolist())), nxt.value

    def commit(self, t_end: float) -> None:
        _check(self._lib.ks_sched_commit(self._h, float(t_end)), "ks_sched_commit")

    def results(self):
        ft = np.zeros(self.n_requests, np.float64)
        fin = np.zeros(self.n_requests, np.float64)
        npre = np.zeros(self.n_requests, np.int32)
        cached = np.zeros(self.n_requests, np.int32)
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int32)
        _check(self._lib.ks_sched_results(self._h, ft.ctypes.data_as(dp), fin.ctypes.data_as(dp),
                                          npre.ctypes.data_as(ip), cached.ctypes.data_as(ip)), "ks_sched_results")
        return dict(first_token=ft, finish=fin, n_preempt=npre, cached_tokens=cached)

    def stats(self) -> dict:
        st = ks_sched_stats()
        _check(self._lib.ks_sched_get_stats(self._h, C.byref(st)), "ks_sched_get_stats")
        return {k: getattr(st, k) for k, _ in ks_sched_stats._fields_ if k != "pad"}

    def close(self) -> None:
        if self._h:
            self._lib.ks_sched_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def make_model_desc(m) -> ks_model_desc:
    """m: any object with n_layers, hidden, ffn, vocab, hq, hkv, head_dim, dtype_bytes, tp."""
    return ks_model_desc(*[int(getattr(m, k, 0)) for k, _ in ks_model_desc._fields_])


def sim_run(ctx: "Context", scheds: Sequence[Scheduler], clock: np.ndarray, model, spec: dict, tier: int, params: dict,
            max_iters: int = 0, log_cap: int = 0):
    """ks_sim_run: clock is a float64 array [n_replicas], updated in place.  Returns (stats dict, step_replica, step_time)."""
    n = len(scheds)
    if not (isinstance(clock, np.ndarray) and clock.dtype == np.float64 and clock.shape == (n,) and clock.flags.c_contiguous):
        raise ValueError("clock: contiguous float64 array [n_replicas]")
    hs = (C.c_void_p * max(n, 1))(*[s._h.value for s in scheds])
    md, sp, pp = make_model_desc(model), make_spec(spec), make_step_params(params)
    rep = np.zeros(max(log_cap, 1), np.int32)
    tim = np.zeros(max(log_cap, 1), np.float32)
    nlog = C.c_int64()
    st = ks_sim_stats()
    _check(ctx._lib.ks_sim_run(ctx._h, hs, clock.ctypes.data_as(C.POINTER(C.c_double)), n, C.byref(md), C.byref(sp),
                               int(tier), C.byref(pp), int(max_iters), rep.ctypes.data_as(C.POINTER(C.c_int32)),
                               tim.ctypes.data_as(C.POINTER(C.c_float)), int(log_cap), C.byref(nlog), C.byref(st)),
           "ks_sim_run")
    k = nlog.value
    return {f: getattr(st, f) for f, _ in ks_sim_stats._fields_}, rep[:k].copy(), tim[:k].copy()
