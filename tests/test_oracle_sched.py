"""Pins for the oracle scheduler (oracle/sched.py; Q18): hand-worked schedules,
closed forms for the uncontended regime, conservation laws and per-step invariants under KV pressure."""
import math

import numpy as np
import pytest

from oracle import sched as S

BIG = S.SchedConfig(max_num_batched_tokens=8192, max_num_seqs=256, block_size=16, num_blocks=1 << 20)


def run(cfg, arrival, P, O, dt=1.0):
    s = S.Scheduler(cfg, arrival, P, O)
    end, priced, batches = S.simulate(s, lambda b: dt)
    return s, end, batches


def test_single_request_prefill_then_decodes():
    # P = 10, 3 output tokens: the prefill step emits token 1, two decode steps emit tokens 2 and 3
    s, end, batches = run(BIG, [0.0], [10], [3])
    assert batches == [[(0, 10, 0)], [(0, 1, 10)], [(0, 1, 11)]]
    assert s.first_token == [1.0] and s.finish == [3.0] and end == 3.0


def test_chunked_prefill_splits_a_prompt_over_the_token_budget():
    cfg = S.SchedConfig(256, 8, 16, 4096)
    s, end, batches = run(cfg, [0.0], [1000], [2])
    assert [b[0][1:] for b in batches] == [(256, 0), (256, 256), (256, 512), (232, 768), (1, 1000)]
    assert s.first_token == [4.0] and s.finish == [5.0]


def test_running_requests_come_first_and_prefill_takes_the_leftover_budget():
    # three decoding requests + a 1000-token prompt arriving later, budget 256: chunk = 256 - 3 = 253
    cfg = S.SchedConfig(256, 8, 16, 4096)
    s = S.Scheduler(cfg, [0.0, 0.0, 0.0, 1.5], [4, 5, 6, 1000], [50, 50, 50, 1])
    assert s.step(0.0) == [(0, 4, 0), (1, 5, 0), (2, 6, 0)]
    s.commit(1.0)
    assert s.step(1.0) == [(0, 1, 4), (1, 1, 5), (2, 1, 6)]      # request 3 has not arrived yet
    s.commit(2.0)
    assert s.step(2.0) == [(0, 1, 5), (1, 1, 6), (2, 1, 7), (3, 253, 0)]
    s.commit(3.0)
    assert s.step(3.0)[-1] == (3, 253, 253)


def test_fcfs_by_arrival_then_index_and_max_num_seqs():
    cfg = S.SchedConfig(8192, 2, 16, 4096)
    s = S.Scheduler(cfg, [0.3, 0.1, 0.1, 0.2], [8, 8, 8, 8], [2, 2, 2, 2])
    assert [r for r, _, _ in s.step(0.5)] == [1, 2]                # earliest arrivals, tie by index; cap S = 2
    s.commit(1.0)
    assert [r for r, _, _ in s.step(1.0)] == [1, 2]
    s.commit(2.0)                                                  # both finish
    assert [r for r, _, _ in s.step(2.0)] == [3, 0]


def test_uncontended_closed_form():
    # all requests at t = 0, budget and cache ample: every prompt is prefilled in step 1 and request i
    # finishes at step O_i; with a constant step time dt: first token at dt, finish at O_i dt
    rng = np.random.Generator(np.random.PCG64(3))
    P = rng.integers(1, 60, 40).tolist()
    O = rng.integers(1, 30, 40).tolist()
    s, end, batches = run(BIG, [0.0] * 40, P, O, dt=0.5)
    assert s.first_token == [0.5] * 40
    assert s.finish == [0.5 * o for o in O]
    assert end == 0.5 * max(O) and s.n_steps == max(O)
    assert [len(b) for b in batches] == [sum(1 for o in O if o > k) for k in range(max(O))]


def test_idle_gaps_jump_to_the_next_arrival():
    s, end, _ = run(BIG, [0.0, 10.0], [5, 5], [2, 2], dt=1.0)
    assert s.finish == [2.0, 12.0] and s.first_token == [1.0, 11.0]


def test_preemption_recomputes_the_newest_request():
    # 6 blocks of 4 tokens.  Two requests of 8 prompt tokens: 2 blocks each.  Decoding grows both until the
    # cache is full; the request at the back of the running queue (1) is preempted and recomputed later.
    cfg = S.SchedConfig(64, 4, 4, 6)
    s = S.Scheduler(cfg, [0.0, 0.0], [8, 8], [8, 6])
    log = []
    now = 0.0
    while not s.done():
        b = s.step(now)
        log.append(b)
        now += 1.0
        s.commit(now)
        assert s.free_blocks >= 0 and sum(s.blocks) + s.free_blocks == 6
    # step 1: both prefill (2 + 2 blocks).  steps 2-5: decode at hist 8..11, a third block each at step 2
    # (tokens 9..12 fit in 3 blocks).  step 6: hist 12 needs a 4th block for request 0 (free = 0):
    # request 1 is preempted (its 5 generated tokens are kept, to be recomputed), request 0 runs alone.
    assert log[0] == [(0, 8, 0), (1, 8, 0)]
    assert log[1] == [(0, 1, 8), (1, 1, 9 - 1)]
    assert log[5] == [(0, 1, 12)]
    assert s.n_preempt == [0, 1]
    # request 0 needs 8 + 8 - 1 = 15 computed tokens -> 4 blocks until it finishes (step 8); request 1
    # cannot be re-admitted while a preemption happened in the step, then needs ceil(13/4) = 4 blocks
    # with only 2 free, so it waits for request 0 to finish, then recomputes 8 + 5 = 13 tokens in one
    # step (emitting token 6 = its last)
    assert s.finish[0] == 8.0
    assert log[8] == [(1, 13, 0)] and s.finish[1] == 9.0
    assert s.tokens_scheduled == (8 + 7) + (8 + 4) + 13        # request 0; request 1 before and after its preemption
    assert s.tokens_scheduled == sum(n for b in log for _, n, _ in b)


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_invariants_and_conservation_under_pressure(seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    n = 60
    cfg = S.SchedConfig(int(rng.integers(64, 512)), int(rng.integers(4, 32)), 16, int(rng.integers(40, 120)))
    arrival = np.sort(rng.uniform(0, 30, n)).tolist()
    P = rng.integers(1, 400, n).tolist()
    O = rng.integers(1, 80, n).tolist()
    s = S.Scheduler(cfg, arrival, P, O)
    now, steps = 0.0, 0
    emitted = [0] * n
    while not s.done():
        b = s.step(now)
        if not b:
            assert not s.running and not s.waiting                # idle only when nothing is queued
            now = max(now, s.next_arrival())
            continue
        assert 0 < sum(x[1] for x in b) <= cfg.max_num_batched_tokens          # token budget
        assert len(s.running) <= cfg.max_num_seqs and len({x[0] for x in b}) == len(b)
        assert [x[0] for x in b] == s.running[:len(b)]            # the batch is a prefix of the running queue
        assert sum(s.blocks) + s.free_blocks == cfg.num_blocks and s.free_blocks >= 0
        for r, n_new, hist in b:
            assert arrival[r] <= now and hist == s.c[r] and n_new >= 1
            assert s.blocks[r] * cfg.block_size >= hist + n_new   # KV blocks cover every scheduled token
            if hist + n_new == s.n_tok[r]:
                emitted[r] += 1
        now += 0.01 + 1e-5 * sum(x[1] for x in b)
        s.commit(now)
        steps += 1
        assert steps < 100000
    assert emitted == O                                           # every request emits exactly max_new tokens
    assert all(math.isfinite(f) and f >= ft > a for f, ft, a in zip(s.finish, s.first_token, arrival))
    assert s.free_blocks == cfg.num_blocks and not s.running and not s.waiting
    # conservation: tokens computed = prompt + generated - 1 per request, plus what preemptions threw away
    assert s.tokens_scheduled >= sum(p + o - 1 for p, o in zip(P, O))
    assert (s.tokens_scheduled == sum(p + o - 1 for p, o in zip(P, O))) == (sum(s.n_preempt) == 0)


def test_rejects_a_request_that_can_never_fit():
    with pytest.raises(ValueError):
        S.Scheduler(S.SchedConfig(64, 4, 16, 4), [0.0], [60], [10])


def test_step_rows_follow_the_mixed_step_pricing_rule():
    # two decodes (cached context 100 and 7) + one 32-token prefill chunk with 64 tokens of history
    m = S.Model(n_layers=4, hidden=64, ffn=128, vocab=1000, hq=4, hkv=2, head_dim=16, tp=2)
    rows = S.step_rows([(5, 1, 100), (9, 1, 7), (2, 32, 64)], m)
    T = 34
    # tp = 2 (Q20): each GPU holds 2 of the 4 query heads, 1 of the 2 KV heads, 64 of the 128
    # FFN columns and 500 of the 1000 vocabulary rows: QKV N = (2 + 2x1) x 16 = 64, O K = 2 x 16 = 32, Gate-Up
    # N = 2 x 64, Down K = 64, LM head N = 500; RoPE over (2 + 1) x 16 = 48 and KV write over 2 x 1 x 16 = 32 values
    # per token; SiLU x Mul over 64; norms and the embedding over the full hidden size
    assert rows[0] == ([[T, 64, 64], [T, 64, 32], [T, 128, 64], [T, 64, 64], [3, 500, 64]], [4, 4, 4, 4, 1])
    assert rows[2] == ([[1, 1, 101], [1, 1, 8], [1, 32, 96]], [4, 4, 4])      # per request: (B, q, kv = hist + q)
    assert rows[3] == ([[T * 64, 4], [T * 64, 0], [T * 48, 2], [T * 32, 3], [T * 64, 1], [T * 64, 0]], [1, 4, 4, 4, 4, 1])
    assert rows[4] == ([[T * 64 * 2, 2]], [8])                                # two all-reduces per layer
    # tp = 1 keeps the unsharded shapes; a dimension smaller than tp is replicated (ceil)
    m1 = S.Model(n_layers=4, hidden=64, ffn=128, vocab=1000, hq=4, hkv=2, head_dim=16, tp=1)
    assert S.step_rows([(5, 1, 100)], m1)[0][0][:2] == [[1, 128, 64], [1, 64, 64]] and 4 not in S.step_rows([(5, 1, 100)], m1)
    m4 = S.Model(n_layers=4, hidden=64, ffn=128, vocab=1000, hq=4, hkv=2, head_dim=16, tp=4)
    assert S.step_rows([(5, 1, 100)], m4)[0][0][0] == [1, (1 + 2 * 1) * 16, 64]   # 1 query head, the KV head replicated
    # kernel launches of the step: n = L (4 GEMM + 3 attention + 4 elementwise + 2 all-reduce) + lm_head + embed + final norm
    assert sum(sum(mm) for _, mm in rows.values()) == 4 * (4 + 3 + 4 + 2) + 3


def test_price_steps_equals_hand_composition():
    from oracle import oracle as O
    import workloads as W
    m = S.Model()
    spec = W.spec_gb200()
    batch = [(0, 1, 500), (1, 1, 2000), (2, 512, 1024)]
    t = S.price_steps([batch], m, spec, 0, W.STEP_PARAMS_CFG4)[0]
    # by hand: L x (4 GEMMs + attention rows + 4 elementwise) + lm_head + embed + final norm, Eq. 4 GPU-bound
    def one(f, v, **kw):
        return O.predict_one(O.make_desc(f, v, **kw), O.make_spec(spec), 0)[0]
    T = 514
    layer = (one(0, [T, 6144, 4096]) + one(0, [T, 4096, 4096]) + one(0, [T, 28672, 4096]) + one(0, [T, 4096, 14336])
             + sum(one(2, [1, q, h + q], hq=32, hkv=8, d=128) for _, q, h in batch)
             + one(3, [T * 4096, 0]) + one(3, [T * 40 * 128, 2]) + one(3, [T * 16 * 128, 3]) + one(3, [T * 14336, 1]))
    body = 32 * layer + one(0, [3, 131072, 4096]) + one(3, [T * 4096, 4]) + one(3, [T * 4096, 0])
    n = 32 * (4 + 3 + 4) + 3
    assert abs(t - (body + n * 4e-6)) < 1e-12


def test_price_steps_tp2_equals_hand_composition():
    # tensor parallel degree 2 (Q20): the per-GPU shapes written out by hand for config 4's
    # decoder (16 query heads, 4 KV heads, 7168 FFN columns, 65536 vocabulary rows per GPU) plus two ring all-reduces
    # per layer of S = T x hidden x 2 bytes (Eq. 3), every term priced one descriptor at a time
    from oracle import oracle as O
    import workloads as W
    m = S.Model(tp=2)
    spec = W.spec_gb200()
    batch = [(0, 1, 500), (1, 1, 2000), (2, 512, 1024)]
    t = S.price_steps([batch], m, spec, 0, W.STEP_PARAMS_CFG4)[0]

    def one(f, v, **kw):
        return O.predict_one(O.make_desc(f, v, **kw), O.make_spec(spec), 0)[0]
    T = 514
    layer = (one(0, [T, 3072, 4096]) + one(0, [T, 4096, 2048]) + one(0, [T, 14336, 4096]) + one(0, [T, 4096, 7168])
             + sum(one(2, [1, q, h + q], hq=16, hkv=4, d=128) for _, q, h in batch)
             + one(3, [T * 4096, 0]) + one(3, [T * 20 * 128, 2]) + one(3, [T * 8 * 128, 3]) + one(3, [T * 7168, 1]))
    ar = 10e-6 + 2.0 * (2 - 1) / 2 * (T * 4096 * 2) / 900e9          # Eq. 3 with the spec's alpha0, beta_eff
    body = 32 * (layer + 2 * ar) + one(0, [3, 65536, 4096]) + one(3, [T * 4096, 4]) + one(3, [T * 4096, 0])
    n = 32 * (4 + 3 + 4 + 2) + 3
    assert abs(t - (body + n * 4e-6)) < 1e-12
    # and the point of sharding: the per-GPU compute of a TP = 2 step is smaller than the TP = 1 step's
    t1 = S.price_steps([batch], S.Model(tp=1), spec, 0, W.STEP_PARAMS_CFG4)[0]
    assert body - 32 * 2 * ar < t1 - (32 * 11 + 3) * 4e-6


# ------------------------------------------------------------------ prefix cache (Q19)
def pc_cfg(T=4096, S=16, bs=16, nb=4096, disk=0):
    return S_cfg(T, S, bs, nb, True, disk)


def S_cfg(T, S_, bs, nb, on, disk):
    return S.SchedConfig(T, S_, bs, nb, enable_prefix_cache=on, disk_blocks=disk)


def drive(s, dt=1.0, until=None):
    now, log = 0.0, []
    while not s.done():
        b = s.step(now)
        if not b:
            now = max(now, s.next_arrival())
            continue
        log.append(b)
        now += dt
        s.commit(now)
        held = sum(1 for k, v in s.gpu_ref.items() if v > 0)
        assert s.free_blocks + len(s.lru) + sum(s.blocks[r] - len(s.held[r]) for r in range(len(s.P))) + held == s.cfg.num_blocks
        assert s.free_blocks >= 0 and set(s.lru) == {k for k, v in s.gpu_ref.items() if v == 0}
    return log


def test_prefix_hit_recomputes_only_the_uncached_suffix():
    # "A prefix hit reuses cached blocks so only the uncached suffix is recomputed"
    s = S.Scheduler(pc_cfg(), [0.0, 1.5], [100, 100], [2, 2], prefix_id=[7, 7], prefix_len=[64, 64])
    log = drive(s)
    assert log[0] == [(0, 100, 0)]
    assert log[2] == [(1, 36, 64)]                      # 4 cached blocks of 16 tokens: history 64, 36 new tokens
    assert s.cached_tokens == [0, 64] and s.gpu_hit_blocks == 4
    # without the cache the second request recomputes everything
    s0 = S.Scheduler(S_cfg(4096, 16, 16, 4096, False, 0), [0.0, 1.5], [100, 100], [2, 2], prefix_id=[7, 7], prefix_len=[64, 64])
    assert drive(s0)[2] == [(1, 100, 0)]
    # a different prefix id, or no prefix, never hits
    s2 = S.Scheduler(pc_cfg(), [0.0, 1.5, 1.5], [100, 100, 100], [2, 2, 2], prefix_id=[7, 8, -1], prefix_len=[64, 64, 64])
    assert drive(s2)[2] == [(1, 100, 0), (2, 100, 0)]


def test_only_full_blocks_are_shared_and_one_token_is_always_computed():
    # prefix of 70 tokens = 4 full blocks (64 tokens) + 6 tokens that are not cacheable
    s = S.Scheduler(pc_cfg(), [0.0, 1.5], [90, 90], [1, 1], prefix_id=[1, 1], prefix_len=[70, 70])
    assert drive(s)[1] == [(1, 26, 64)]
    # the whole prompt is cached (64 = 4 blocks): the last block is recomputed so that a token can be sampled
    s = S.Scheduler(pc_cfg(), [0.0, 1.5], [64, 64], [1, 1], prefix_id=[1, 1], prefix_len=[64, 64])
    assert drive(s)[1] == [(1, 16, 48)]
    # requests of the same content but different prefix lengths share the common leading blocks
    s = S.Scheduler(pc_cfg(), [0.0, 1.5], [200, 200], [1, 1], prefix_id=[1, 1], prefix_len=[128, 40])
    assert drive(s)[1] == [(1, 168, 32)]


def test_shared_blocks_are_counted_once_so_more_requests_run_concurrently():
    # "... and more concurrent requests from freed KV capacity": a 512-token shared prefix
    # (32 blocks) + 16 own tokens; 80 blocks hold two such requests without the cache, many with it
    n = 8
    args = ([0.0] + [1.5] * (n - 1), [528] * n, [8] * n)
    on = S.Scheduler(pc_cfg(nb=80), *args, prefix_id=[3] * n, prefix_len=[512] * n)
    off = S.Scheduler(S_cfg(4096, 16, 16, 80, False, 0), *args, prefix_id=[3] * n, prefix_len=[512] * n)
    lon, loff = drive(on), drive(off)
    assert max(len(b) for b in lon) == 8 and max(len(b) for b in loff) == 2
    assert lon[2] == [(0, 1, 529)] + [(r, 16, 512) for r in range(1, 8)]
    assert max(on.finish) < max(off.finish) and len(lon) < len(loff)
    assert sum(on.n_preempt) == 0


def test_lru_eviction_and_the_disk_tier():
    # cache of 12 blocks.  A (prefix 1, 8 blocks) runs and leaves; B (no prefix, 10 blocks) needs the space:
    # A's unreferenced blocks are evicted.  C (prefix 1) then misses on the GPU tier ...
    def run(disk):
        s = S.Scheduler(pc_cfg(bs=16, nb=12, disk=disk), [0.0, 5.0, 10.0], [129, 150, 129], [1, 1, 1],
                        prefix_id=[1, -1, 1], prefix_len=[128, 0, 128])
        return s, drive(s)
    s, log = run(0)
    assert log == [[(0, 129, 0)], [(1, 150, 0)], [(2, 129, 0)]] and s.evictions == 6 and s.disk_hit_blocks == 0   # 4 free + 6 evicted = B's 10 blocks
    # ... unless the persistent disk tier still has them: they are loaded instead of recomputed
    s, log = run(64)
    assert log[2] == [(2, 1, 128)] and s.disk_hit_blocks == 6 and s.gpu_hit_blocks == 2
    # a disk tier of 4 blocks keeps only the 4 most recently written blocks (4..7): block 0 is gone, so no leading run
    s, log = run(4)
    assert log[2] == [(2, 129, 0)]


def test_eviction_takes_the_least_recently_released_blocks_first():
    # A (prefix 1, 4 blocks) finishes at t = 1, B (prefix 2, 4 blocks) at t = 2; cache of 10 blocks.
    # D (no prefix, 6 blocks + nothing shared) needs 4 evictions: all of A's go, B's stay.
    s = S.Scheduler(pc_cfg(bs=16, nb=10), [0.0, 1.0, 2.0, 3.0, 3.0], [65, 65, 90, 65, 65], [1, 1, 1, 1, 1],
                    prefix_id=[1, 2, -1, 1, 2], prefix_len=[64, 64, 0, 64, 64])
    log = drive(s)
    assert log[2] == [(2, 90, 0)] and s.evictions >= 2
    assert log[3][0] == (3, 65, 0)                      # prefix 1 was evicted (released first) ...
    assert log[3][1] == (4, 1, 64)                      # ... prefix 2 survived


def test_cache_without_prefixes_is_the_plain_scheduler():
    rng = np.random.Generator(np.random.PCG64(5))
    n = 50
    arrival = np.sort(rng.uniform(0, 5, n)).tolist()
    P, O = rng.integers(1, 300, n).tolist(), rng.integers(1, 40, n).tolist()
    a = S.Scheduler(S_cfg(256, 8, 16, 60, True, 100), arrival, P, O)
    b = S.Scheduler(S_cfg(256, 8, 16, 60, False, 0), arrival, P, O)
    assert drive(a, dt=0.05) == drive(b, dt=0.05) and a.finish == b.finish


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_prefix_cache_invariants_on_random_traces(seed):
    rng = np.random.Generator(np.random.PCG64(40 + seed))
    n = 70
    arrival = np.sort(rng.uniform(0, 10, n)).tolist()
    pid = rng.integers(-1, 5, n).tolist()
    plen_of = {p: int(rng.integers(20, 400)) for p in range(5)}
    own = rng.integers(1, 120, n)
    plen = [plen_of[p] if p >= 0 else 0 for p in pid]
    P = [pl + int(o) for pl, o in zip(plen, own)]
    O = rng.integers(1, 50, n).tolist()
    nb = int(max(-(-(p + o) // 16) for p, o in zip(P, O)) + rng.integers(5, 60))
    s = S.Scheduler(S_cfg(int(rng.integers(64, 600)), int(rng.integers(2, 16)), 16, nb, True, int(rng.integers(0, 80))),
                    arrival, P, O, prefix_id=pid, prefix_len=plen)
    log = drive(s, dt=0.03)                              # drive() checks the block accounting after every step
    assert all(math.isfinite(f) for f in s.finish) and s.free_blocks + len(s.lru) == nb
    assert all(h % 16 == 0 and h <= pl for h, pl in zip(s.cached_tokens, [x * (1 + k) for x, k in zip(plen, s.n_preempt)]))
    assert sum(s.cached_tokens) > 0
    if sum(s.n_preempt) == 0:                            # every token is either computed once or served from the cache
        assert s.tokens_scheduled + sum(s.cached_tokens) == sum(p + o - 1 for p, o in zip(P, O))


def test_fine_slots_regroup_the_same_rows():
    """eta per family incl. "the LM head, attention prefill and decode".  With fine_slots the step's rows
    are the same rows, grouped by model slot: 0 the four layer GEMMs, 5 the LM head, 6 prefill chunks, 7 decodes."""
    import workloads as W
    from oracle import oracle as O
    m0, m1 = S.Model(n_layers=3), S.Model(n_layers=3, fine_slots=1)
    batch = [(0, 1, 700), (1, 300, 0), (2, 1, 45), (3, 212, 512)]        # two decodes, two prefill chunks
    r0, r1 = S.step_rows(batch, m0), S.step_rows(batch, m1)
    assert sorted(r1) == [0, 3, 5, 6, 7]
    assert r1[0][0] == r0[0][0][:4] and r1[5][0] == [r0[0][0][4]] == [[4, m0.vocab, m0.hidden]] and r1[5][1] == [1]
    assert r1[6][0] == [[1, 300, 300], [1, 212, 724]] and r1[7][0] == [[1, 1, 701], [1, 1, 46]]
    assert r1[6][1] == [3, 3] and r1[7][1] == [3, 3] and r1[3] == r0[3]
    # priced with ONE head for GEMM + LM head and ONE for both attention slots, the regrouping changes nothing ...
    rng = np.random.Generator(np.random.PCG64(3))
    hg, ha, he, hl = (W.make_head(rng, 12, 64) for _ in range(4))
    spec, par = W.spec_gb200(), W.STEP_PARAMS_CFG4
    batches = [batch, [(0, 1, 9)], [(5, 64, 0)]]                          # a decode-only and a prefill-only step too
    coarse = S.price_steps(batches, m0, spec, W.TIER_A, par, heads={0: hg, 2: ha, 3: he})
    same = S.price_steps(batches, m1, spec, W.TIER_A, par, heads={0: hg, 5: hg, 6: ha, 7: ha, 3: he})
    assert np.allclose(same, coarse, rtol=1e-12, atol=0)
    # ... and a different LM head moves every step by exactly the LM-head kernel's change (multiplicity 1)
    fine = S.price_steps(batches, m1, spec, W.TIER_A, par, heads={0: hg, 5: hl, 6: ha, 7: ha, 3: he})
    for i, b in enumerate(batches):
        row = W.Bucket(W.FAM_GEMM, W._i32([len(b)], [m0.vocab], [m0.hidden]))
        d = (O.predict_bucket(row, [spec], W.TIER_A, head=O.Head(hl))["lat"][0, 0]
             - O.predict_bucket(row, [spec], W.TIER_A, head=O.Head(hg))["lat"][0, 0])
        assert abs((fine[i] - coarse[i]) - d) <= 1e-12 * coarse[i]
