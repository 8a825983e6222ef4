"""Seeded synthetic workload generators for the five BASELINE.json configs.

This package is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2606_28565_b200/``); it belongs to neither and imports neither.  It holds none of the method's arithmetic
(no FLOP/byte formulas, no roofline, no features, no MLP, no interpolation, no
sums): it only draws kernel-instance descriptors, hardware-spec vectors, head
weights, efficiency grids and step/config segmentations with
``numpy.random.Generator(PCG64(seed))`` following the recipe in DESIGN.md §4
(SURVEY.md §8(d)).  The descriptor-emission rule of a serving step (which
kernels a mixed prefill/decode step launches, §5.8) lives here
because it is the thin host driver's job, not the predictor's.

The paper's own workloads (production trace PAPER.md:253, microbenchmark
database PAPER.md:151) are not available; these inputs stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional

import numpy as np

# kernel families (values match include/ks.h and oracle/ks_oracle.h, each of
# which declares its own copy)
FAM_GEMM, FAM_GROUPED, FAM_ATTN, FAM_ELEMWISE, FAM_ALLREDUCE = 0, 1, 2, 3, 4
FAM_NAMES = {0: "gemm", 1: "grouped_gemm", 2: "attention", 3: "elementwise", 4: "allreduce"}
TIER_NONE, TIER_A, TIER_B, TIER_B_ROUTED = 0, 1, 2, 3
# efficiency-model slots beyond the per-decode-family ones (slot = family for 0..4), after the families of the
# paper's Tables 2 and 4; the library and the oracle wrapper treat a slot as an index
SLOT_LM_HEAD, SLOT_ATTN_PREFILL, SLOT_ATTN_DECODE, SLOT_RMSNORM, SLOT_SILU_MUL, SLOT_ROPE, SLOT_KV_WRITE = 5, 6, 7, 8, 9, 10, 11
SLOT_EMBEDDING, SLOT_RESIDUAL_ADD = 12, 13
HEAD_UTILISATION, HEAD_LOG_ETA = 0, 1      # what an MLP head's output means
# elementwise sub-operations (reading Q1)
SUB_RMSNORM, SUB_SILU_MUL, SUB_ROPE, SUB_KV_WRITE, SUB_EMBED, SUB_RESADD = 0, 1, 2, 3, 4, 5
N_EXPERTS = 8


@dataclass
class Bucket:
    """One family bucket: SoA columns, all the same length and dtype."""
    family: int
    cols: List[np.ndarray]
    dtype_bytes: int = 2
    hq: int = 0
    hkv: int = 0
    head_dim: int = 0
    step_off: Optional[np.ndarray] = None  # CSR [n_steps+1] int32 into this bucket
    mult: Optional[np.ndarray] = None      # per-row multiplicity (layer-homogeneous form); None = ones
    model_slot: Optional[int] = None       # efficiency-model slot that prices the bucket (eta is learned
                                           # per kernel family, finer than the decode family); None = the family's slot

    @property
    def slot(self) -> int:
        return self.family if self.model_slot is None else int(self.model_slot)

    @property
    def n(self) -> int:
        return int(self.cols[0].shape[0]) if self.cols else 0


@dataclass
class Head:
    n_in: int
    h1: int
    h2: int
    W1: np.ndarray  # [n_in][h1] fp32
    b1: np.ndarray  # [h1]
    W2: np.ndarray  # [h1][h2]
    b2: np.ndarray  # [h2]
    w3: np.ndarray  # [h2]
    b3: float
    out_mode: int = 0   # HEAD_UTILISATION (sigmoid out) or HEAD_LOG_ETA (z = log eta)


@dataclass
class BoundedHead:
    """Bounded analytical head: gamma(x) = sigmoid(w_gamma.x + b_gamma),
    alpha(x) = max(0, w_alpha.x + b_alpha); utilisation e = gamma - alpha / W."""
    n_in: int
    w_gamma: np.ndarray  # [n_in] fp32
    b_gamma: float
    w_alpha: np.ndarray  # [n_in] fp32
    b_alpha: float


@dataclass
class Grid:
    dims: np.ndarray      # int32[3]
    lo_log2: np.ndarray   # float32[3]
    hi_log2: np.ndarray   # float32[3]
    values: np.ndarray    # fp32 [d0][d1][d2], last axis fastest


@dataclass
class Workload:
    name: str
    buckets: List[Bucket]
    specs: List[dict]
    tier: int
    heads: Dict[int, Head] = field(default_factory=dict)
    grids: Dict[int, Grid] = field(default_factory=dict)
    bounded: Dict[int, BoundedHead] = field(default_factory=dict)   # families whose Tier-A head is the bounded form
    ensembles: Dict[int, List[Head]] = field(default_factory=dict)  # families whose Tier-A head is an MLP ensemble
    n_steps: int = 0
    cfg_off: Optional[np.ndarray] = None  # CSR [n_cfg+1] int32 over steps
    step_params: Optional[dict] = None
    seed: int = 0

    @property
    def n_rows(self) -> int:
        return sum(b.n for b in self.buckets)


def spec_gb200(**over) -> dict:
    """Config 1's spec vector (Table 5 GB200 peaks; SM/tile fields [BJ])."""
    s = dict(peak_flops=2.25e15, peak_bw=8.0e12, n_sm=148, ctas_per_sm=1, tile_m=128,
             tile_n=128, ew_elems_per_cta=4096, l2_bytes=126e6, t0=2e-6,
             ar_alpha0=10e-6, ar_beta_eff=900e9)   # interconnect (Eq. 3): NVLink 5 datasheet bandwidth, 10 us startup
    s.update(over)
    return s


STEP_PARAMS_ZERO = dict(c_disp=0.0, floor_l=0.0, c_ovl=0.0, c_tail=0.0, body_scale=1.0)
STEP_PARAMS_CFG4 = dict(c_disp=4e-6, floor_l=0.0, c_ovl=0.0, c_tail=0.0, body_scale=1.0)
STEP_PARAMS_HOSTBOUND = dict(c_disp=4e-6, floor_l=5e-3, c_ovl=8e-3, c_tail=5e-4, body_scale=1.0)


# ----------------------------------------------------------------------------- helpers
def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def _log_uniform_int(rng, lo: int, hi: int, n: int) -> np.ndarray:
    x = rng.uniform(np.log2(lo), np.log2(hi), size=n)
    return np.clip(np.rint(np.exp2(x)), lo, hi).astype(np.int64)


def make_head(rng, n_in: int, h: int, bias_std: float = 0.1, w_std: float = 0.1) -> Head:
    W1 = rng.normal(0.0, w_std, size=(n_in, h)).astype(np.float32)
    W2 = rng.normal(0.0, w_std, size=(h, h)).astype(np.float32)
    w3 = rng.normal(0.0, w_std, size=(h,)).astype(np.float32)
    if bias_std > 0:
        b1 = rng.normal(0.0, bias_std, size=(h,)).astype(np.float32)
        b2 = rng.normal(0.0, bias_std, size=(h,)).astype(np.float32)
        b3 = float(np.float32(rng.normal(0.0, bias_std)))
    else:
        b1 = np.zeros(h, np.float32)
        b2 = np.zeros(h, np.float32)
        b3 = 0.0
    return Head(n_in, h, h, W1, b1, W2, b2, w3, b3)


def make_ensemble(rng, n_in: int, h_member: int, k: int, bias_std: float = 0.1, w_std: float = 0.1) -> List[Head]:
    """k independently drawn MLP members of one shape ("small MLP ensemble"; Q17)."""
    return [make_head(rng, n_in, h_member, bias_std, w_std) for _ in range(k)]


def make_bounded_head(rng, n_in: int) -> BoundedHead:
    """Random bounded head: peak utilisation gamma around sigmoid(1) = 0.73, partial-wave overhead alpha ~ 0.2."""
    return BoundedHead(n_in, rng.normal(0.0, 0.3, n_in).astype(np.float32), float(np.float32(rng.normal(1.0, 0.3))),
                       rng.normal(0.0, 0.15, n_in).astype(np.float32), float(np.float32(rng.uniform(0.05, 0.4))))


def _box3(v: np.ndarray) -> np.ndarray:
    """Separable 3-tap box filter (1/3,1/3,1/3) along each axis, edge replication."""
    v = v.astype(np.float64)
    for ax in range(3):
        p = np.concatenate([np.take(v, [0], axis=ax), v, np.take(v, [-1], axis=ax)], axis=ax)
        n = v.shape[ax]
        v = (np.take(p, range(0, n), axis=ax) + np.take(p, range(1, n + 1), axis=ax)
             + np.take(p, range(2, n + 2), axis=ax)) / 3.0
    return v.astype(np.float32)


def make_grid(rng, lo, hi, dims=(32, 32, 32)) -> Grid:
    vals = rng.uniform(0.2, 0.95, size=dims)
    return Grid(np.asarray(dims, np.int32), np.asarray(lo, np.float32),
                np.asarray(hi, np.float32), np.ascontiguousarray(_box3(vals)))


GEMM_NK = np.array([4096, 5120, 8192, 11008, 14336], dtype=np.int64)


def _gemm_rows(rng, n: int):
    M = np.left_shift(1, rng.integers(0, 14, size=n)).astype(np.int64)
    N = GEMM_NK[rng.integers(0, 5, size=n)]
    K = GEMM_NK[rng.integers(0, 5, size=n)]
    return M, N, K


def _attn_rows(rng, n: int):
    B_ = _log_uniform_int(rng, 1, 256, n)
    decode = rng.random(n) < 0.5
    q = np.where(decode, 1, _log_uniform_int(rng, 128, 8192, n))
    x = rng.uniform(0.0, 1.0, size=n) * np.log2(32768 - q + 1)
    hist = np.clip(np.rint(np.exp2(x)).astype(np.int64) - 1, 0, 32768 - q)
    return B_, q, q + hist


def _elem_rows(rng, n: int):
    ne = _log_uniform_int(rng, 4096, 32 * 2 ** 20, n)
    sub = rng.integers(0, 6, size=n).astype(np.int64)
    return ne, sub


def _i32(*cols):
    return [np.ascontiguousarray(c, dtype=np.int32) for c in cols]


def uniform_step_offsets(rng, n_rows: int, n_steps: int) -> np.ndarray:
    """CSR offsets splitting n_rows into n_steps multinomial-sized (possibly empty) segments."""
    if n_steps <= 0:
        return np.zeros(1, np.int32)
    cnt = rng.multinomial(n_rows, np.full(n_steps, 1.0 / n_steps))
    return np.concatenate([[0], np.cumsum(cnt)]).astype(np.int32)


def cfg_offsets(rng, n_steps: int, n_cfg: int) -> np.ndarray:
    cnt = rng.multinomial(n_steps, np.full(n_cfg, 1.0 / n_cfg))
    return np.concatenate([[0], np.cumsum(cnt)]).astype(np.int32)


# ----------------------------------------------------------------------------- config 1
def config1(n: int = 4096, seed: int = 0) -> Workload:
    """PR1 ref: GEMM descriptors as fp32 SoA holding exact ints; head 8->64->64->1, biases 0."""
    rng = _rng(seed)
    M, N, K = _gemm_rows(rng, n)
    cols = [np.ascontiguousarray(c, dtype=np.float32) for c in (M, N, K)]
    head = make_head(rng, 8, 64, bias_std=0.0)
    b = Bucket(FAM_GEMM, cols, dtype_bytes=2)
    n_steps = max(1, n // 128)
    b.step_off = uniform_step_offsets(rng, n, n_steps)
    return Workload("cfg1_pr1_gemm", [b], [spec_gb200()], TIER_A, heads={FAM_GEMM: head},
                    n_steps=n_steps, cfg_off=cfg_offsets(rng, n_steps, min(4, n_steps)),
                    step_params=dict(STEP_PARAMS_ZERO), seed=seed)


# ----------------------------------------------------------------------------- config 2
def config2(n: int = 1_000_000, seed: int = 1, n_in: int = 12, h: int = 128,
            n_steps: Optional[int] = None, n_cfg: int = 16) -> Workload:
    """1M mixed descriptors: GEMM 50% / attention 30% / elementwise-norm 20%; three heads.

    The config names no step structure; for the step-composition rows (S6/S7)
    each bucket is split into ``n_steps`` multinomial segments (default n/256).
    """
    rng = _rng(seed)
    ng, na = int(round(0.5 * n)), int(round(0.3 * n))
    ne = n - ng - na
    M, N, K = _gemm_rows(rng, ng)
    B_, q, kv = _attn_rows(rng, na)
    nel, sub = _elem_rows(rng, ne)
    heads = {f: make_head(rng, n_in, h) for f in (FAM_GEMM, FAM_ATTN, FAM_ELEMWISE)}
    if n_steps is None:
        n_steps = max(1, n // 256)
    buckets = [Bucket(FAM_GEMM, _i32(M, N, K)),
               Bucket(FAM_ATTN, _i32(B_, q, kv), hq=32, hkv=8, head_dim=128),
               Bucket(FAM_ELEMWISE, _i32(nel, sub))]
    for b in buckets:
        b.step_off = uniform_step_offsets(rng, b.n, n_steps)
    return Workload("cfg2_mixed_1M", buckets, [spec_gb200()], TIER_A, heads=heads,
                    n_steps=n_steps, cfg_off=cfg_offsets(rng, n_steps, min(n_cfg, n_steps)),
                    step_params=dict(STEP_PARAMS_CFG4), seed=seed)


# ----------------------------------------------------------------------------- config 3
GEMM_SPAN = ((0.0, 10.0, 10.0), (13.0, 14.0, 14.0))
ATTN_SPAN = ((0.0, 0.0, 0.0), (8.0, 13.0, 15.0))


def _grid_queries(rng, n: int, lo, hi):
    lo = np.asarray(lo, np.float64)
    hi = np.asarray(hi, np.float64)
    x = rng.uniform(lo[None, :], hi[None, :], size=(n, 3))
    oob = rng.random(n) < 0.10
    axis = rng.integers(0, 3, size=n)
    below = rng.random(n) < 0.5
    push = rng.uniform(0.0, 2.0, size=n)
    rows = np.nonzero(oob)[0]
    ax = axis[rows]
    x[rows, ax] = np.where(below[rows], lo[ax] - push[rows], hi[ax] + push[rows])
    return np.maximum(np.rint(np.exp2(x)), 1.0).astype(np.int64)


def config3(n: int = 4_194_304, seed: int = 2, routed: bool = False, n_in: int = 12, h: int = 128) -> Workload:
    """Tier B: GEMM/attention queries against 32^3 measured-efficiency grids, 10% OOB (clamped).
    routed=True (not a BASELINE.json config): the 10 % out-of-hull queries fall
    back to per-family Tier-A heads (cfg-2-sized, seed 1) instead of being clamped."""
    rng = _rng(seed)
    ng = n // 2
    na = n - ng
    grids = {FAM_GEMM: make_grid(rng, *GEMM_SPAN), FAM_ATTN: make_grid(rng, *ATTN_SPAN)}
    g = _grid_queries(rng, ng, *GEMM_SPAN)
    a = _grid_queries(rng, na, *ATTN_SPAN)
    a[:, 2] = np.maximum(a[:, 2], a[:, 1])  # keep kv >= q by raising kv
    buckets = [Bucket(FAM_GEMM, _i32(g[:, 0], g[:, 1], g[:, 2])),
               Bucket(FAM_ATTN, _i32(a[:, 0], a[:, 1], a[:, 2]), hq=32, hkv=8, head_dim=128)]
    n_steps = max(1, n // 256)
    for b in buckets:
        b.step_off = uniform_step_offsets(rng, b.n, n_steps)
    heads = {}
    if routed:
        hr = _rng(1)
        heads = {f: make_head(hr, n_in, h) for f in (FAM_GEMM, FAM_ATTN)}
    return Workload("cfg3_tierB_routed" if routed else "cfg3_tierB_4M", buckets, [spec_gb200()],
                    TIER_B_ROUTED if routed else TIER_B, grids=grids, heads=heads,
                    n_steps=n_steps, cfg_off=cfg_offsets(rng, n_steps, min(16, n_steps)),
                    step_params=dict(STEP_PARAMS_ZERO), seed=seed)


# ----------------------------------------------------------------------------- the paper's model families
ELEM_SPAN = ((12.0, 0.0, 0.0), (25.0, 0.0, 0.0))   # grids of one elementwise sub-op: log2 n on axis 0, two flat axes


def config_families(n: int = 64_000, seed: int = 7, tier: int = TIER_A, n_in: int = 12, h: int = 128,
                    log_eta: bool = False) -> Workload:
    """Eight buckets, one per kernel family the paper learns eta for (Tables 2 and 4, PAPER.md:269-283,
    :321-336): GEMM, LM head, attention prefill, attention decode, RMSNorm, SiLU x Mul, RoPE, KV-cache write — each
    with its OWN head and grid (model slots; two buckets of one decode family carry different models).  Not a
    BASELINE.json config: the parity case for slot dispatch.  log_eta: the heads' outputs are log eta."""
    rng = _rng(seed)
    k = max(n // 8, 1)
    M, N, K = _gemm_rows(rng, k)
    Ml = _log_uniform_int(rng, 1, 512, k)                                   # LM head: M = sequences in the step
    Nl = np.full(k, VOCAB, np.int64)
    Kl = GEMM_NK[rng.integers(0, 5, size=k)]
    B_, q, kv = _attn_rows(rng, 4 * k)
    pre = np.nonzero(q > 1)[0][:k]
    dec = np.nonzero(q == 1)[0][:k]
    ne = [_log_uniform_int(rng, 4096, 32 * 2 ** 20, k) for _ in range(4)]
    at = dict(hq=32, hkv=8, head_dim=128)
    buckets = [Bucket(FAM_GEMM, _i32(M, N, K)),
               Bucket(FAM_GEMM, _i32(Ml, Nl, Kl), model_slot=SLOT_LM_HEAD),
               Bucket(FAM_ATTN, _i32(B_[pre], q[pre], kv[pre]), model_slot=SLOT_ATTN_PREFILL, **at),
               Bucket(FAM_ATTN, _i32(B_[dec], q[dec], kv[dec]), model_slot=SLOT_ATTN_DECODE, **at)]
    for sub, slot, nel in zip((SUB_RMSNORM, SUB_SILU_MUL, SUB_ROPE, SUB_KV_WRITE),
                              (SLOT_RMSNORM, SLOT_SILU_MUL, SLOT_ROPE, SLOT_KV_WRITE), ne):
        buckets.append(Bucket(FAM_ELEMWISE, _i32(nel, np.full(k, sub)), model_slot=slot))
    heads, grids = {}, {}
    for b in buckets:
        heads[b.slot] = make_head(rng, n_in, h)
        heads[b.slot].out_mode = HEAD_LOG_ETA if log_eta else HEAD_UTILISATION
        span = GEMM_SPAN if b.family == FAM_GEMM else ATTN_SPAN if b.family == FAM_ATTN else ELEM_SPAN
        if b.slot == SLOT_LM_HEAD:
            span = ((0.0, 16.0, 10.0), (9.0, 18.0, 14.0))                   # the vocabulary axis is its own span
        grids[b.slot] = make_grid(rng, *span, dims=(32, 32, 32) if b.family != FAM_ELEMWISE else (32, 1, 1))
    n_steps = max(1, k // 16)
    for b in buckets:
        b.step_off = uniform_step_offsets(rng, b.n, n_steps)
    return Workload("families_8_slots", buckets, [spec_gb200()], tier, heads=heads, grids=grids, n_steps=n_steps,
                    cfg_off=cfg_offsets(rng, n_steps, min(8, n_steps)), step_params=dict(STEP_PARAMS_CFG4), seed=seed)


# ----------------------------------------------------------------------------- serving-step emission
HIDDEN, FFN, HQ, HKV, HEAD_DIM, VOCAB, N_LAYERS = 4096, 14336, 32, 8, 128, 131072, 32
QKV_N = (HQ + 2 * HKV) * HEAD_DIM  # 6144


def _tp_shard(x: int, tp: int) -> int:
    """Per-GPU share of a model dimension split tp ways (ceil; Q20)."""
    return -(-int(x) // max(int(tp), 1))


def _draw_steps(rng, n_steps: int):
    """Continuous-batching step mix: Poisson(64) decodes + chunked prefill (512-token chunks)."""
    n_dec = np.clip(rng.poisson(64.0, size=n_steps), 1, 256).astype(np.int64)
    chunk = (rng.random(n_steps) < 0.25).astype(np.int64)
    j = rng.integers(0, 16, size=n_steps).astype(np.int64)
    kv_dec = rng.integers(128, 8193, size=n_steps).astype(np.int64)
    T = n_dec + 512 * chunk
    return n_dec, chunk, 512 * j, kv_dec, T


def _csr(counts: np.ndarray) -> np.ndarray:
    return np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)


def _attn_bucket(n_dec, chunk, hist, kv_dec, n_layers):
    """Per layer: one decode-attention row; +1 prefill row (cached history + own chunk) if chunked."""
    n_steps = n_dec.shape[0]
    per_layer = 1 + chunk                      # rows per layer for each step
    cnt = per_layer * n_layers
    off = _csr(cnt)
    total = int(off[-1])
    step_of = np.repeat(np.arange(n_steps), cnt)
    pos = np.arange(total) - off[:-1][step_of]
    is_prefill = (pos % per_layer[step_of]) == 1
    B_ = np.where(is_prefill, 1, n_dec[step_of])
    q = np.where(is_prefill, 512, 1)
    kv = np.where(is_prefill, hist[step_of] + 512, kv_dec[step_of])
    return B_, q, kv, off


def config4(n_steps: int = 100_000, seed: int = 3, tier: int = TIER_NONE, n_cfg: int = 64,
            step_params: Optional[dict] = None, n_layers: int = N_LAYERS, tp: int = 1,
            dedupe: bool = False) -> Workload:
    """Serving-step composition: 32-layer dense decoder, 9 kernels/layer (+1 prefill attention).
    tp > 1 (not a BASELINE.json config) adds the two tensor-parallel
    all-reduces per layer of PAPER.md:221 as a fourth bucket: S = T x hidden x 2 bytes over P = tp.
    dedupe=True emits the SAME steps in the paper's layer-homogeneous form (PAPER.md:231,
    t_gpu = L t_layer + t_lm_head + t_embed): one layer's kernels per step, each with multiplicity L."""
    rng = _rng(seed)
    n_dec, chunk, hist, kv_dec, T = _draw_steps(rng, n_steps)
    L = n_layers
    if dedupe:
        return _config4_dedupe(rng, n_dec, chunk, hist, kv_dec, T, L, n_steps, tier, n_cfg, step_params, tp, seed)
    # per-GPU shapes under tensor parallelism (Q20): heads, FFN columns and vocabulary split tp ways
    hq, hkv, ffn, vocab = _tp_shard(HQ, tp), _tp_shard(HKV, tp), _tp_shard(FFN, tp), _tp_shard(VOCAB, tp)
    # GEMM bucket: per layer QKV, O, Gate-Up, Down at M=T; then the LM head once per step
    gN = np.array([(hq + 2 * hkv) * HEAD_DIM, HIDDEN, 2 * ffn, HIDDEN] * L + [vocab], np.int64)
    gK = np.array([HIDDEN, hq * HEAD_DIM, HIDDEN, ffn] * L + [HIDDEN], np.int64)
    per = gN.shape[0]
    gM = np.repeat(T, per).reshape(n_steps, per)
    gM[:, -1] = n_dec + chunk
    gemm = Bucket(FAM_GEMM, _i32(gM.reshape(-1), np.tile(gN, n_steps), np.tile(gK, n_steps)))
    gemm.step_off = _csr(np.full(n_steps, per))
    # elementwise bucket: embedding; per layer RMSNorm, RoPE, KV-write, SiLU*Mul; final norm
    mult = np.array([HIDDEN] + [HIDDEN, (hq + hkv) * HEAD_DIM, 2 * hkv * HEAD_DIM, ffn] * L + [HIDDEN], np.int64)
    sub = np.array([SUB_EMBED] + [SUB_RMSNORM, SUB_ROPE, SUB_KV_WRITE, SUB_SILU_MUL] * L + [SUB_RMSNORM], np.int64)
    pe = mult.shape[0]
    ne = (T[:, None] * mult[None, :]).reshape(-1)
    elem = Bucket(FAM_ELEMWISE, _i32(ne, np.tile(sub, n_steps)))
    elem.step_off = _csr(np.full(n_steps, pe))
    B_, q, kv, aoff = _attn_bucket(n_dec, chunk, hist, kv_dec, L)
    attn = Bucket(FAM_ATTN, _i32(B_, q, kv), hq=hq, hkv=hkv, head_dim=HEAD_DIM, step_off=aoff)
    heads = {}
    if tier == TIER_A:
        hr = _rng(1)  # cfg-2-sized heads, seed 1 (SURVEY.md §8(d) cfg 4b)
        heads = {f: make_head(hr, 12, 128) for f in (FAM_GEMM, FAM_ATTN, FAM_ELEMWISE)}
    name = "cfg4a_steps_tierNONE" if tier == TIER_NONE else "cfg4b_steps_tierA"
    buckets = [gemm, attn, elem]
    if tp > 1:
        S = np.repeat(T * HIDDEN * 2, 2 * L)
        buckets.append(Bucket(FAM_ALLREDUCE, _i32(S, np.full(S.shape[0], tp)), step_off=_csr(np.full(n_steps, 2 * L))))
        name += f"_tp{tp}"
    return Workload(name, buckets, [spec_gb200()], tier, heads=heads, n_steps=n_steps,
                    cfg_off=cfg_offsets(rng, n_steps, min(n_cfg, n_steps)),
                    step_params=dict(step_params or STEP_PARAMS_CFG4), seed=seed)


def allreduce_rows(n: int = 6_400_000, seed: int = 5, tp: int = 4) -> Workload:
    """n tensor-parallel all-reduce rows: the two per-layer all-reduces of
    100,000 steps of config 4's decoder (T tokens x hidden x 2 bytes over P = tp), as one bucket."""
    rng = _rng(seed)
    T = np.clip(rng.poisson(64, size=n), 1, 256) + 512 * (rng.random(n) < 0.25)
    return Workload(f"allreduce_tp{tp}", [Bucket(FAM_ALLREDUCE, _i32(T * HIDDEN * 2, np.full(n, tp)))],
                    [spec_gb200()], TIER_NONE, seed=seed)


def _config4_dedupe(rng, n_dec, chunk, hist, kv_dec, T, L, n_steps, tier, n_cfg, step_params, tp, seed):
    i32 = lambda a: np.ascontiguousarray(a, dtype=np.int32)
    hq, hkv, ffn, vocab = _tp_shard(HQ, tp), _tp_shard(HKV, tp), _tp_shard(FFN, tp), _tp_shard(VOCAB, tp)
    gN = np.array([(hq + 2 * hkv) * HEAD_DIM, HIDDEN, 2 * ffn, HIDDEN, vocab], np.int64)
    gK = np.array([HIDDEN, hq * HEAD_DIM, HIDDEN, ffn, HIDDEN], np.int64)
    gM = np.repeat(T, 5).reshape(n_steps, 5)
    gM[:, -1] = n_dec + chunk
    gemm = Bucket(FAM_GEMM, _i32(gM.reshape(-1), np.tile(gN, n_steps), np.tile(gK, n_steps)),
                  step_off=_csr(np.full(n_steps, 5)), mult=i32(np.tile([L, L, L, L, 1], n_steps)))
    mult_e = np.array([HIDDEN, HIDDEN, (hq + hkv) * HEAD_DIM, 2 * hkv * HEAD_DIM, ffn, HIDDEN], np.int64)
    sub = np.array([SUB_EMBED, SUB_RMSNORM, SUB_ROPE, SUB_KV_WRITE, SUB_SILU_MUL, SUB_RMSNORM], np.int64)
    elem = Bucket(FAM_ELEMWISE, _i32((T[:, None] * mult_e[None, :]).reshape(-1), np.tile(sub, n_steps)),
                  step_off=_csr(np.full(n_steps, 6)), mult=i32(np.tile([1, L, L, L, L, 1], n_steps)))
    B_, q, kv, aoff = _attn_bucket(n_dec, chunk, hist, kv_dec, 1)
    attn = Bucket(FAM_ATTN, _i32(B_, q, kv), hq=hq, hkv=hkv, head_dim=HEAD_DIM, step_off=aoff,
                  mult=i32(np.full(B_.shape[0], L)))
    buckets = [gemm, attn, elem]
    if tp > 1:
        buckets.append(Bucket(FAM_ALLREDUCE, _i32(T * HIDDEN * 2, np.full(n_steps, tp)), step_off=_csr(np.full(n_steps, 1)),
                              mult=i32(np.full(n_steps, 2 * L))))
    heads = {}
    if tier == TIER_A:
        hr = _rng(1)
        heads = {f: make_head(hr, 12, 128) for f in (FAM_GEMM, FAM_ATTN, FAM_ELEMWISE)}
    return Workload("cfg4_steps_layer_homogeneous", buckets, [spec_gb200()], tier, heads=heads, n_steps=n_steps,
                    cfg_off=cfg_offsets(rng, n_steps, min(n_cfg, n_steps)),
                    step_params=dict(step_params or STEP_PARAMS_CFG4), seed=seed)


# ----------------------------------------------------------------------------- config 5
def sweep_specs(rng, n_specs: int) -> List[dict]:
    """What-if hardware specs spanning Table 5's ladder, log-uniform."""
    out = []
    for _ in range(n_specs):
        n_sm = int(_log_uniform_int(rng, 80, 160, 1)[0])
        peak = float(np.exp(rng.uniform(np.log(0.3e15), np.log(2.5e15))))
        bw = float(np.exp(rng.uniform(np.log(2e12), np.log(8e12))))
        l2 = float(np.exp(rng.uniform(np.log(32.0), np.log(128.0)))) * 2 ** 20
        out.append(spec_gb200(n_sm=n_sm, peak_flops=float(np.float32(peak)),
                              peak_bw=float(np.float32(bw)), l2_bytes=float(np.float32(l2))))
    return out


def config5(n_rows: int = 2 ** 22, n_specs: int = 64, seed: int = 4, n_in: int = 32, h: int = 256,
            n_layers: int = N_LAYERS) -> Workload:
    """What-if sweep: 8-expert top-2 MoE decoder rows x hardware-spec vectors, four heads.

    Rows are generated step by step; the last step is cut (in bucket order elementwise, GEMM,
    grouped GEMM, attention) so that the buckets hold exactly ``n_rows`` rows in total.
    """
    rng = _rng(seed)
    L, E = n_layers, N_EXPERTS
    pe, pg, pgr = 6 * L + 2, 3 * L + 1, 2 * L
    est = n_rows // (pe + pg + pgr + L) + 2
    n_dec, chunk, hist, kv_dec, T = _draw_steps(rng, est)
    cnt = np.stack([np.full(est, pe), np.full(est, pg), np.full(est, pgr), (1 + chunk) * L], axis=1)
    cum = np.cumsum(cnt.sum(axis=1))
    n_full = int(np.searchsorted(cum, n_rows, side="right"))
    rem = n_rows - (int(cum[n_full - 1]) if n_full > 0 else 0)
    n_steps = n_full + (1 if rem > 0 else 0)
    cnt = cnt[:n_steps].copy()
    if rem > 0:
        for b in range(4):
            take = min(rem, int(cnt[-1, b]))
            cnt[-1, b] = take
            rem -= take
    n_dec, chunk, hist, kv_dec, T = (a[:n_steps] for a in (n_dec, chunk, hist, kv_dec, T))

    def cut(arrs, per, b):
        """Keep the first cnt[s,b] of the `per` rows each step emitted."""
        keep = (np.arange(per)[None, :] < cnt[:, b][:, None]).reshape(-1)
        return [a[keep] for a in arrs]

    # elementwise: embedding; per layer RMSNorm, RoPE, KV-write, RMSNorm, routing, SiLU*Mul; final norm
    mult = np.array([HIDDEN] + [HIDDEN, (HQ + HKV) * HEAD_DIM, 2 * HKV * HEAD_DIM, HIDDEN, E, 2 * FFN] * L
                    + [HIDDEN], np.int64)
    sub = np.array([SUB_EMBED] + [SUB_RMSNORM, SUB_ROPE, SUB_KV_WRITE, SUB_RMSNORM, SUB_RESADD, SUB_SILU_MUL] * L
                   + [SUB_RMSNORM], np.int64)
    ne = (T[:, None] * mult[None, :]).reshape(-1)
    elem = Bucket(FAM_ELEMWISE, _i32(*cut([ne, np.tile(sub, n_steps)], pe, 0)), step_off=_csr(cnt[:, 0]))
    # plain GEMMs: per layer QKV, O, router; LM head
    gN = np.array([QKV_N, HIDDEN, E] * L + [VOCAB], np.int64)
    gK = np.array([HIDDEN, HIDDEN, HIDDEN] * L + [HIDDEN], np.int64)
    gM = np.repeat(T, pg).reshape(n_steps, pg)
    gM[:, -1] = n_dec + chunk
    gemm = Bucket(FAM_GEMM, _i32(*cut([gM.reshape(-1), np.tile(gN, n_steps), np.tile(gK, n_steps)], pg, 1)),
                  step_off=_csr(cnt[:, 1]))
    # grouped GEMMs: per layer Gate-Up and Down share one routing draw m ~ Multinomial(2T, 1/8)
    m = rng.multinomial(np.repeat(2 * T, L), np.full(E, 1.0 / E)).astype(np.int64)   # [n_steps*L][E]
    m2 = np.repeat(m, 2, axis=0)                                                      # gate-up, down
    rN = np.tile(np.array([2 * FFN, HIDDEN], np.int64), n_steps * L)
    rK = np.tile(np.array([HIDDEN, FFN], np.int64), n_steps * L)
    grp = Bucket(FAM_GROUPED, _i32(*cut([rN, rK] + [m2[:, e] for e in range(E)], pgr, 2)),
                 step_off=_csr(cnt[:, 2]))
    B_, q, kv, aoff = _attn_bucket(n_dec, chunk, hist, kv_dec, L)
    full_cnt = (1 + chunk) * L
    keep = np.concatenate([np.arange(c) < k for c, k in zip(full_cnt, cnt[:, 3])]) if n_steps else np.zeros(0, bool)
    attn = Bucket(FAM_ATTN, _i32(B_[keep], q[keep], kv[keep]), hq=HQ, hkv=HKV, head_dim=HEAD_DIM,
                  step_off=_csr(cnt[:, 3]))
    heads = {f: make_head(rng, n_in, h) for f in (FAM_GEMM, FAM_GROUPED, FAM_ATTN, FAM_ELEMWISE)}
    specs = sweep_specs(rng, n_specs)
    return Workload("cfg5_whatif_moe", [elem, gemm, grp, attn], specs, TIER_A, heads=heads,
                    n_steps=n_steps, cfg_off=np.array([0, n_steps], np.int32),
                    step_params=dict(STEP_PARAMS_CFG4), seed=seed)


CONFIGS = {"cfg1": config1, "cfg2": config2, "cfg3": config3, "cfg4": config4, "cfg5": config5}


# ----------------------------------------------------------------------------- serving traces (NEXT-4)
@dataclass
class ServingModel:
    """Dense decoder the simulated steps are priced for (defaults: config 4's model)."""
    n_layers: int = N_LAYERS
    hidden: int = HIDDEN
    ffn: int = FFN
    vocab: int = VOCAB
    hq: int = HQ
    hkv: int = HKV
    head_dim: int = HEAD_DIM
    dtype_bytes: int = 2
    tp: int = 1
    fine_slots: int = 0    # 1: LM head, prefill and decode attention are priced by their own model slots


@dataclass
class Replica:
    """One simulated serving replica: scheduler limits + its request trace."""
    max_num_batched_tokens: int
    max_num_seqs: int
    block_size: int
    num_blocks: int
    arrival: np.ndarray      # float64 [n] seconds
    prompt_len: np.ndarray   # int32 [n]
    max_new: np.ndarray      # int32 [n]
    enable_prefix_cache: bool = False
    disk_blocks: int = 0
    prefix_id: Optional[np.ndarray] = None    # int32 [n], -1 = no shared prefix
    prefix_len: Optional[np.ndarray] = None   # int32 [n]


def serving_trace(rng, n: int, rate: float, prompt_mean: float = 512.0, out_mean: float = 128.0):
    """Poisson arrivals at `rate` requests/s; log-normal prompt and output lengths (sigma 1.0 / 0.8)
    clipped to [8, 8192] / [1, 1024] — the shape of chat-style serving traces (synthetic stand-in for the
    paper's request traces)."""
    arrival = np.cumsum(rng.exponential(1.0 / rate, size=n))
    p = np.clip(np.round(rng.lognormal(np.log(prompt_mean) - 0.5, 1.0, size=n)), 8, 8192).astype(np.int32)
    o = np.clip(np.round(rng.lognormal(np.log(out_mean) - 0.32, 0.8, size=n)), 1, 1024).astype(np.int32)
    return arrival.astype(np.float64), p, o


def add_shared_prefixes(rng, rep: Replica, n_prefixes: int = 8, share: float = 0.7, disk_blocks: int = 0) -> Replica:
    """Give `share` of the requests one of n_prefixes shared system prompts (log-uniform 64..2048 tokens, Zipf-like
    popularity) in front of their own prompt, and switch the replica's prefix cache on."""
    n = rep.arrival.shape[0]
    plen_of = _log_uniform_int(rng, 64, 2048, n_prefixes)
    pop = 1.0 / np.arange(1, n_prefixes + 1)
    pid = np.where(rng.random(n) < share, rng.choice(n_prefixes, size=n, p=pop / pop.sum()), -1).astype(np.int32)
    plen = np.where(pid >= 0, plen_of[np.maximum(pid, 0)], 0).astype(np.int32)
    rep.prefix_id, rep.prefix_len = pid, plen
    rep.prompt_len = np.minimum(rep.prompt_len + plen, 8192).astype(np.int32)
    rep.prefix_len = np.minimum(rep.prefix_len, rep.prompt_len).astype(np.int32)
    rep.enable_prefix_cache, rep.disk_blocks = True, int(disk_blocks)
    return rep


def sim_replicas(n_replicas: int = 64, n_requests: int = 200, seed: int = 6, pressure: bool = False) -> List[Replica]:
    """A what-if sweep over scheduler limits and load: token budget in {1024, 2048, 4096, 8192}, max_num_seqs in
    {32, 64, 128, 256}, arrival rate log-uniform in [4, 64] requests/s.  pressure=True shrinks the KV cache so
    that preemption/recompute happens."""
    rng = _rng(seed)
    out = []
    for _ in range(n_replicas):
        T = int(rng.choice([1024, 2048, 4096, 8192]))
        S = int(rng.choice([32, 64, 128, 256]))
        rate = float(np.exp(rng.uniform(np.log(4.0), np.log(64.0))))
        a, p, o = serving_trace(rng, n_requests, rate)
        nb = 1024 if pressure else 65536      # blocks of 16 tokens: 16k tokens (tight) or 1M tokens (ample)
        out.append(Replica(T, S, 16, nb, a, p, o))
    return out
