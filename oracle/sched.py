"""CPU oracle of the serving scheduler and the closed simulation loop.

TEST INFRASTRUCTURE ONLY (same rules as oracle.py): imported by tests/ and bench.py's oracle legs, never
by the product package; shares no code with the C++ scheduler in ``csrc/ks_sched.cu``.

What it follows, in the paper's order:

* PAPER.md:241  "At each step, the scheduler emits a batch descriptor (decode tokens, prefill-chunk
  lengths, per-request KV lengths) that is exactly the predictor's input".
* PAPER.md:243  "a single token-budget loop advances every request's computed-token count toward its
  target, which unifies continuous batching, chunked prefill, and prefix-cache-aware admission in one
  algorithm, with FCFS queuing and preemption/recompute under KV pressure".
* PAPER.md:249  mixed steps are priced kernel by kernel from the step's token composition: dense GEMMs,
  norms and activations at the total token count; attention per request, a decode over its cached
  context, a prefill chunk over its cached history plus its own causal triangle.
* PAPER.md:231  t_gpu = L t_layer + t_lm_head + t_embed  (one layer's kernels with multiplicity L).
* PAPER.md:159  the completion event of a step is scheduled at now + t_step.

* PAPER.md:247  content-hashed KV cache in two tiers (volatile GPU tier, persistent disk tier): a prefix
  hit reuses cached blocks so only the uncached suffix is recomputed.

The paper gives the loop in one sentence and the cache in two; the precise rules below are DESIGN.md
readings Q18 (scheduler) and Q19 (prefix cache).  Plain Python loops, one request at a time.
"""
from __future__ import annotations

import math
from collections import OrderedDict, deque
from dataclasses import dataclass
from typing import Callable, List, Optional, Sequence, Tuple

import numpy as np


@dataclass
class SchedConfig:
    max_num_batched_tokens: int   # T: token budget of one step
    max_num_seqs: int             # S: most requests running at once
    block_size: int               # tokens per KV-cache block
    num_blocks: int               # KV-cache blocks on the GPU
    enable_prefix_cache: bool = False   # content-hashed prefix cache, GPU tier (Q19)
    disk_blocks: int = 0          # capacity of the persistent disk tier in blocks (0 = no disk tier)


class Scheduler:
    """One replica's scheduler.  step(now) forms the batch of the step that starts at `now`;
    commit(t_end) applies it at the step's completion time."""

    def __init__(self, cfg: SchedConfig, arrival: Sequence[float], prompt_len: Sequence[int], max_new: Sequence[int],
                 prefix_id: Optional[Sequence[int]] = None, prefix_len: Optional[Sequence[int]] = None):
        self.cfg = cfg
        n = len(arrival)
        self.arrival = [float(a) for a in arrival]
        self.P = [int(p) for p in prompt_len]
        self.O = [int(o) for o in max_new]
        for i in range(n):
            if self.P[i] < 1 or self.O[i] < 1:
                raise ValueError("prompt_len and max_new must be >= 1")
            if self._blocks_for(self.P[i] + self.O[i]) > cfg.num_blocks:
                raise ValueError("a request alone must fit the KV cache")
        # FCFS: arrival order, ties by index
        self.order = sorted(range(n), key=lambda i: (self.arrival[i], i))
        self.next_arrival_pos = 0
        self.n_tok = list(self.P)          # tokens known so far = prompt + generated
        self.c = [0] * n                   # computed tokens (KV present)
        self.g = [0] * n                   # generated tokens
        self.blocks = [0] * n              # KV blocks held
        self.free_blocks = cfg.num_blocks
        self.waiting: deque = deque()
        self.running: List[int] = []
        self.batch: List[Tuple[int, int, int]] = []   # (request, n_new, hist) of the step being executed
        self.first_token = [math.nan] * n
        self.finish = [math.nan] * n
        self.n_preempt = [0] * n
        self.n_finished = 0
        self.n_steps = 0
        self.tokens_scheduled = 0
        # prefix cache.  The first prefix_len[i] prompt tokens of request i are the content
        # named prefix_id[i]; full block j of that content has the hash key (prefix_id, j).
        self.pid = [-1] * n if prefix_id is None else [int(v) for v in prefix_id]
        self.plen = [0] * n if prefix_len is None else [int(v) for v in prefix_len]
        for i in range(n):
            if self.pid[i] < 0:
                self.plen[i] = 0
            if not 0 <= self.plen[i] <= self.P[i]:
                raise ValueError("0 <= prefix_len <= prompt_len")
        self.held: List[List[Tuple[int, int]]] = [[] for _ in range(n)]   # cache keys a request holds a reference on
        self.registered = [0] * n          # prefix blocks of the request already looked up / offered to the cache
        self.gpu_ref: dict = {}            # key -> reference count (GPU tier)
        self.lru: OrderedDict = OrderedDict()     # keys with reference count 0, least recently released first
        self.disk: OrderedDict = OrderedDict()    # disk tier, least recently used first
        self.cached_tokens = [0] * n       # prompt tokens served from the cache over all (re)admissions
        self.gpu_hit_blocks = 0
        self.disk_hit_blocks = 0
        self.evictions = 0

    def _blocks_for(self, tokens: int) -> int:
        return -(-tokens // self.cfg.block_size)

    def avail(self) -> int:
        """Blocks an allocation may use: free ones plus cached ones nobody references (evicted on demand)."""
        return self.free_blocks + len(self.lru)

    def _alloc(self, k: int) -> None:
        """Take k blocks: free ones first, then evict unreferenced cached blocks, least recently released first
        (a block evicted from the GPU tier stays in the disk tier if it is there)."""
        assert k <= self.avail()
        while k > 0:
            if self.free_blocks > 0:
                self.free_blocks -= 1
            else:
                key, _ = self.lru.popitem(last=False)
                del self.gpu_ref[key]
                self.evictions += 1
            k -= 1

    def _release(self, r: int) -> None:
        """Request r gives up its blocks: private ones become free, shared ones lose a reference."""
        self.free_blocks += self.blocks[r] - len(self.held[r])
        for key in self.held[r]:
            self.gpu_ref[key] -= 1
            if self.gpu_ref[key] == 0:
                self.lru[key] = True
        self.held[r] = []
        self.blocks[r] = 0
        self.registered[r] = 0

    def _disk_put(self, key) -> None:
        if self.cfg.disk_blocks <= 0:
            return
        if key in self.disk:
            self.disk.move_to_end(key)
            return
        self.disk[key] = True
        if len(self.disk) > self.cfg.disk_blocks:
            self.disk.popitem(last=False)

    def _lookup(self, r: int):
        """Longest leading run of request r's prefix blocks present in the GPU tier or, failing that, the disk
        tier; at least one token of the request is always left to compute.  -> (keys, where) lists."""
        if not self.cfg.enable_prefix_cache or self.pid[r] < 0:
            return [], []
        bs = self.cfg.block_size
        limit = min(self.plen[r] // bs, (self.n_tok[r] - 1) // bs)
        keys, where = [], []
        for j in range(limit):
            key = (self.pid[r], j)
            if key in self.gpu_ref:
                where.append("gpu")
            elif key in self.disk:
                where.append("disk")
            else:
                break
            keys.append(key)
        return keys, where

    def done(self) -> bool:
        return self.n_finished == len(self.P)

    def next_arrival(self) -> float:
        if self.next_arrival_pos < len(self.order):
            return self.arrival[self.order[self.next_arrival_pos]]
        return math.inf

    def step(self, now: float) -> List[Tuple[int, int, int]]:
        """The token-budget loop.  Returns [(request, n_new, hist)], possibly empty (idle)."""
        assert not self.batch, "commit the previous step first"
        cfg = self.cfg
        while self.next_arrival_pos < len(self.order) and self.arrival[self.order[self.next_arrival_pos]] <= now:
            self.waiting.append(self.order[self.next_arrival_pos])
            self.next_arrival_pos += 1
        budget = cfg.max_num_batched_tokens
        batch: List[Tuple[int, int, int]] = []
        preempted = False
        # 1. running requests first, in queue order: each advances towards its target
        i = 0
        while i < len(self.running) and budget > 0:
            r = self.running[i]
            n_new = min(self.n_tok[r] - self.c[r], budget)
            need = self._blocks_for(self.c[r] + n_new) - self.blocks[r]
            alive = True
            while need > self.avail():
                # KV pressure: preempt the request at the back of the running queue; it will be recomputed
                v = self.running.pop()
                self._release(v)
                self.c[v] = 0
                self.n_preempt[v] += 1
                self.waiting.appendleft(v)
                preempted = True
                if v == r:
                    alive = False
                    break
            if not alive:
                break
            self._alloc(need)
            self.blocks[r] += need
            batch.append((r, n_new, self.c[r]))
            budget -= n_new
            i += 1
        # 2. admission from the waiting queue, FCFS, unless this step had to preempt
        if not preempted:
            while self.waiting and budget > 0 and len(self.running) < cfg.max_num_seqs:
                r = self.waiting[0]
                # prefix-cache-aware admission: cached leading blocks are not recomputed
                keys, where = self._lookup(r) if self.c[r] == 0 else ([], [])
                hit = len(keys) * cfg.block_size
                n_new = min(self.n_tok[r] - (self.c[r] + hit), budget)
                need = self._blocks_for(self.c[r] + hit + n_new) - self.blocks[r] - len(keys)
                # blocks leaving the allocatable pool: unreferenced GPU hits, one new block per disk hit, the rest
                taken = sum(1 for k, w in zip(keys, where) if w == "gpu" and self.gpu_ref[k] == 0)
                taken += sum(1 for w in where if w == "disk") + need
                if taken > self.avail():
                    break
                for k, w in zip(keys, where):          # reference the GPU hits first so they cannot be evicted
                    if w == "gpu":
                        if self.gpu_ref[k] == 0:
                            del self.lru[k]
                        self.gpu_ref[k] += 1
                        self.gpu_hit_blocks += 1
                for k, w in zip(keys, where):          # disk hits are loaded into newly allocated GPU blocks
                    if w == "disk":
                        self._alloc(1)
                        self.gpu_ref[k] = 1
                        self._disk_put(k)
                        self.disk_hit_blocks += 1
                self._alloc(need)
                self.held[r] = list(keys)
                self.registered[r] = len(keys)
                self.blocks[r] += need + len(keys)
                self.c[r] += hit
                self.cached_tokens[r] += hit
                self.waiting.popleft()
                self.running.append(r)
                batch.append((r, n_new, self.c[r]))
                budget -= n_new
        self.batch = batch
        return list(batch)

    def commit(self, t_end: float) -> None:
        """The step completes at t_end: computed counts advance; a request whose known
        tokens are all computed emits one token; a request with max_new tokens leaves and frees its blocks."""
        for r, n_new, _ in self.batch:
            self.c[r] += n_new
            self.tokens_scheduled += n_new
            if self.cfg.enable_prefix_cache and self.pid[r] >= 0:
                # full prefix blocks whose KV now exists are offered to the cache (and written through to disk);
                # if the key is already there (another request got there first) the block stays private
                full = min(self.c[r], self.plen[r]) // self.cfg.block_size
                for j in range(self.registered[r], full):
                    key = (self.pid[r], j)
                    if key not in self.gpu_ref:
                        self.gpu_ref[key] = 1
                        self.held[r].append(key)
                    self._disk_put(key)
                self.registered[r] = max(self.registered[r], full)
            if self.c[r] == self.n_tok[r]:
                self.g[r] += 1
                if self.g[r] == 1:
                    self.first_token[r] = t_end
                if self.g[r] == self.O[r]:
                    self.finish[r] = t_end
                    self._release(r)
                    self.running.remove(r)
                    self.n_finished += 1
                else:
                    self.n_tok[r] += 1
        if self.batch:
            self.n_steps += 1
        self.batch = []


@dataclass
class Model:
    """Dense decoder the steps are priced for (defaults = config 4's model)."""
    n_layers: int = 32
    hidden: int = 4096
    ffn: int = 14336
    vocab: int = 131072
    hq: int = 32
    hkv: int = 8
    head_dim: int = 128
    dtype_bytes: int = 2
    tp: int = 1
    fine_slots: int = 0    # 1: the paper's finer model families, see step_rows


# bucket key -> decode family.  Keys 0-4 are the decode families themselves; 5, 6, 7 are the model slots of the LM
# head (decoded as a GEMM) and of prefill / decode attention (Q22; numbering of include/ks.h, restated)
KEY_FAMILY = {0: 0, 2: 2, 3: 3, 4: 4, 5: 0, 6: 2, 7: 2}


def shard(x: int, tp: int) -> int:
    """Per-GPU share of a dimension split tp ways (ceil; a dimension smaller than tp is replicated)."""
    return -(-int(x) // max(int(tp), 1))


def step_rows(batch: Sequence[Tuple[int, int, int]], m: Model):
    """Batch descriptor -> kernel rows of the step, layer-homogeneous form.

    Returns dict family -> (columns [list of int lists], multiplicities).  Families: 0 GEMM (M, N, K),
    2 attention (B, q, kv), 3 elementwise (n, subop), 4 all-reduce (S bytes, P) when tp > 1.
    Sub-operation codes as in DESIGN.md Q1: 0 RMSNorm, 1 SiLU*Mul, 2 RoPE, 3 KV write, 4 embedding.
    With m.fine_slots the keys are MODEL SLOTS (eta is learned separately for "GEMM, the LM head,
    attention prefill and decode, and the elementwise and memory kernels"): 0 the four layer GEMMs, 5 the LM-head row,
    6 the prefill chunks (n_new > 1), 7 the decode requests (n_new = 1), 3 elementwise, 4 all-reduce.
    """
    T = sum(n for _, n, _ in batch)          # dense kernels run over the concatenated tokens
    n_seq = len(batch)                       # one logits row per scheduled request
    L = m.n_layers
    # Tensor parallelism ("partial activations across the P shards"; Q20): every GPU holds
    # ceil(1/P) of the attention heads, of the FFN columns and of the vocabulary.  QKV and Gate-Up are split
    # along N, O and Down along K; norms and the embedding run on the full hidden size on every GPU.
    hq_p, hkv_p = shard(m.hq, m.tp), shard(m.hkv, m.tp)
    ffn_p, vocab_p = shard(m.ffn, m.tp), shard(m.vocab, m.tp)
    qkv_n = (hq_p + 2 * hkv_p) * m.head_dim
    gemm = ([[T, qkv_n, m.hidden], [T, m.hidden, hq_p * m.head_dim], [T, 2 * ffn_p, m.hidden], [T, m.hidden, ffn_p],
             [n_seq, vocab_p, m.hidden]], [L, L, L, L, 1])
    elem = ([[T * m.hidden, 4], [T * m.hidden, 0], [T * (hq_p + hkv_p) * m.head_dim, 2],
             [T * 2 * hkv_p * m.head_dim, 3], [T * ffn_p, 1], [T * m.hidden, 0]], [1, L, L, L, L, 1])
    # attention per request: a decode (q = 1) over its cached context, a prefill chunk over its cached
    # history plus its own causal triangle (the family's pair count handles q x hist + triangle)
    attn = ([[1, n_new, hist + n_new] for _, n_new, hist in batch], [L] * n_seq)
    out = {0: gemm, 2: attn, 3: elem}
    if m.fine_slots:
        pre = [i for i, (_, n_new, _) in enumerate(batch) if n_new > 1]
        dec = [i for i, (_, n_new, _) in enumerate(batch) if n_new == 1]
        out = {0: (gemm[0][:4], gemm[1][:4]), 5: (gemm[0][4:], gemm[1][4:]),
               6: ([attn[0][i] for i in pre], [L] * len(pre)), 7: ([attn[0][i] for i in dec], [L] * len(dec)), 3: elem}
    if m.tp > 1:
        out[4] = ([[T * m.hidden * m.dtype_bytes, m.tp]], [2 * L])
    return out


def simulate(sched: Scheduler, step_time: Callable[[List[Tuple[int, int, int]]], float], t0: float = 0.0,
             max_steps: Optional[int] = None, forced: Optional[Sequence[float]] = None):
    """The closed loop of one replica: form a batch, price it, advance the clock.

    step_time(batch) -> seconds.  `forced`: per-step durations to advance the clock with instead (the
    priced value is still recorded) — used to replay another implementation's clock.  Returns
    (end time, [priced step times], [batches])."""
    now = float(t0)
    priced: List[float] = []
    batches: List[List[Tuple[int, int, int]]] = []
    while not sched.done() and (max_steps is None or len(priced) < max_steps):
        batch = sched.step(now)
        if not batch:
            nxt = sched.next_arrival()
            if not math.isfinite(nxt):
                break
            now = max(now, nxt)               # idle until the next request arrives
            continue
        t = float(step_time(batch))
        priced.append(t)
        batches.append(batch)
        now = now + (float(forced[len(priced) - 1]) if forced is not None else t)
        sched.commit(now)
    return now, priced, batches


def price_steps(batches: Sequence[Sequence[Tuple[int, int, int]]], m: Model, spec: dict, tier: int, params: dict,
                heads=None, grids=None) -> np.ndarray:
    """Step wall times (Eq. 4) of the given batches, priced by the oracle predictor: rows of step_rows ->
    per-kernel latency (oracle.predict_bucket) -> weighted step sums + Eq. 4 (oracle.compose)."""
    from . import oracle as O
    import workloads as W   # dataclasses only (no arithmetic)

    # bucket keys in the order the buckets are summed (with fine slots: keys are model slots, KEY_FAMILY decodes them)
    fams = ([0, 6, 3] if m.fine_slots else [0, 2, 3]) + ([4] if m.tp > 1 else []) + ([5, 7] if m.fine_slots else [])
    cols = {f: [] for f in fams}
    mult = {f: [] for f in fams}
    off = {f: [0] for f in fams}
    for b in batches:
        rows = step_rows(b, m)
        for f in fams:
            cols[f].extend(rows[f][0])
            mult[f].extend(rows[f][1])
            off[f].append(len(cols[f]))
    lats, offs, mults = [], [], []
    for f in fams:
        fam = KEY_FAMILY[f]
        a = np.asarray(cols[f], np.int64).reshape(len(cols[f]), 2 if fam in (3, 4) else 3)
        bk = W.Bucket(fam, [np.ascontiguousarray(a[:, j]) for j in range(a.shape[1])], dtype_bytes=m.dtype_bytes,
                      hq=shard(m.hq, m.tp) if fam == 2 else 0, hkv=shard(m.hkv, m.tp) if fam == 2 else 0,
                      head_dim=m.head_dim if fam == 2 else 0)
        head = O.Head(heads[f]) if (heads and f in heads) else None
        grid = O.Grid(grids[f]) if (grids and f in grids) else None
        lats.append(O.predict_bucket(bk, [spec], tier, head=head, grid=grid)["lat"][0])
        offs.append(np.asarray(off[f], np.int64))
        mults.append(np.asarray(mult[f], np.int64))
    n = len(batches)
    step_lat, _ = O.compose(lats, offs, n, params, np.array([0, n], np.int64), mults=mults)
    return step_lat
