"""-m "not gpu": the product's host scheduler (ks_sched_*, csrc/ks_sched.cu) against the oracle scheduler
(oracle/sched.py), bit for bit: every batch (request, new tokens, history), every queue decision, the
per-request results and the counters, on seeded traces with and without KV pressure.  The scheduler is
host logic and needs no GPU; step times here come from a fixed function of the batch so both sides see
identical clocks."""
import math

import numpy as np
import pytest

from oracle import sched as S
from paper_2606_28565_b200 import binding as B
from paper_2606_28565_b200 import build as ksbuild
import workloads as W


@pytest.fixture(scope="module", autouse=True)
def lib():
    ksbuild.build()
    return B.load()


def step_time(batch):
    return 2e-3 + 1e-5 * sum(n for _, n, _ in batch) + 3e-6 * len(batch)


def run_both(rep: W.Replica, max_steps=200000):
    o = S.Scheduler(S.SchedConfig(rep.max_num_batched_tokens, rep.max_num_seqs, rep.block_size, rep.num_blocks,
                                  rep.enable_prefix_cache, rep.disk_blocks),
                    rep.arrival, rep.prompt_len, rep.max_new, rep.prefix_id, rep.prefix_len)
    p = B.Scheduler(rep.max_num_batched_tokens, rep.max_num_seqs, rep.block_size, rep.num_blocks,
                    rep.enable_prefix_cache, rep.disk_blocks)
    p.add_requests(rep.arrival, rep.prompt_len, rep.max_new, rep.prefix_id, rep.prefix_len)
    now, steps = 0.0, 0
    while not o.done():
        bo = o.step(now)
        bp, nxt = p.step(now)
        assert bp == bo, f"step {steps}: batches differ"
        assert nxt == o.next_arrival()
        if not bo:
            assert math.isfinite(nxt)
            now = max(now, nxt)
            continue
        now += step_time(bo)
        o.commit(now)
        p.commit(now)
        steps += 1
        assert steps < max_steps
    bp, nxt = p.step(now)
    assert bp == [] and nxt == math.inf                       # finished: idle with no arrival left
    res = p.results()
    assert np.array_equal(res["first_token"], np.array(o.first_token))
    assert np.array_equal(res["finish"], np.array(o.finish))
    assert res["n_preempt"].tolist() == o.n_preempt
    assert res["cached_tokens"].tolist() == o.cached_tokens
    st = p.stats()
    assert (st["gpu_hit_blocks"], st["disk_hit_blocks"], st["evictions"]) == (o.gpu_hit_blocks, o.disk_hit_blocks, o.evictions)
    assert (st["n_steps"], st["tokens_scheduled"], st["n_preemptions"]) == (o.n_steps, o.tokens_scheduled, sum(o.n_preempt))
    assert (st["n_requests"], st["n_finished"], st["n_running"], st["n_waiting"]) == (len(o.P), len(o.P), 0, 0)
    assert st["free_blocks"] == rep.num_blocks
    p.close()
    return o


def test_matches_oracle_on_sweep_replicas():
    for rep in W.sim_replicas(n_replicas=6, n_requests=120, seed=60):
        o = run_both(rep)
        assert sum(o.n_preempt) == 0


def test_matches_oracle_under_kv_pressure():
    pre = 0
    for rep in W.sim_replicas(n_replicas=6, n_requests=150, seed=61, pressure=True):
        pre += sum(run_both(rep).n_preempt)
    assert pre > 0                                            # the tight cache did force recomputation


@pytest.mark.parametrize("seed", range(8))
def test_matches_oracle_on_small_adversarial_configs(seed):
    rng = np.random.Generator(np.random.PCG64(700 + seed))
    n = 80
    bs = int(rng.choice([1, 4, 16]))
    P = rng.integers(1, 300, n).astype(np.int32)
    O = rng.integers(1, 60, n).astype(np.int32)
    nb = int(-(-int((P + O).max()) // bs) + rng.integers(0, 40))    # barely enough for the largest request
    arrival = np.round(np.sort(rng.uniform(0, 2.0, n)), 2)          # many equal arrival times: ties by index
    rep = W.Replica(int(rng.integers(8, 400)), int(rng.integers(1, 20)), bs, nb, arrival, P, O)
    run_both(rep)


@pytest.mark.parametrize("seed,disk", [(0, 0), (1, 0), (2, 300), (3, 2000), (4, 40), (5, 0)])
def test_prefix_cache_matches_oracle(seed, disk):
    rng = np.random.Generator(np.random.PCG64(800 + seed))
    hits = ev = dh = 0
    for rep in W.sim_replicas(n_replicas=3, n_requests=120, seed=80 + seed):
        rep = W.add_shared_prefixes(rng, rep, disk_blocks=disk)
        rep.arrival = rep.arrival * 0.05                       # a burst: many requests in flight at once
        rep.num_blocks = int(-(-int((rep.prompt_len + rep.max_new).max()) // 16) + rng.integers(50, 400))
        o = run_both(rep)
        hits, ev, dh = hits + o.gpu_hit_blocks, ev + o.evictions, dh + o.disk_hit_blocks
    assert hits > 0 and ev > 0
    if disk >= 300:
        assert dh > 0                                          # evicted blocks came back from the disk tier


def test_prefix_cache_hand_worked():
    # tests/test_oracle_sched.py::test_lru_eviction_and_the_disk_tier, product side
    p = B.Scheduler(4096, 16, 16, 12, True, 64)
    p.add_requests([0.0, 5.0, 10.0], [129, 150, 129], [1, 1, 1], [1, -1, 1], [128, 0, 128])
    now, log = 0.0, []
    while True:
        b, nxt = p.step(now)
        if not b:
            if not math.isfinite(nxt):
                break
            now = max(now, nxt)
            continue
        log.append(b)
        now += 1.0
        p.commit(now)
    assert log == [[(0, 129, 0)], [(1, 150, 0)], [(2, 1, 128)]]
    st = p.stats()
    assert (st["gpu_hit_blocks"], st["disk_hit_blocks"], st["evictions"]) == (2, 6, 6)
    assert p.results()["cached_tokens"].tolist() == [0, 0, 128]
    p.close()


def test_hand_worked_schedule():
    # tests/test_oracle_sched.py::test_running_requests_come_first...: same numbers, product side
    p = B.Scheduler(256, 8, 16, 4096)
    p.add_requests([0.0, 0.0, 0.0, 1.5], [4, 5, 6, 1000], [50, 50, 50, 1])
    assert p.step(0.0) == ([(0, 4, 0), (1, 5, 0), (2, 6, 0)], 1.5)
    p.commit(1.0)
    assert p.step(1.0)[0] == [(0, 1, 4), (1, 1, 5), (2, 1, 6)]
    p.commit(2.0)
    assert p.step(2.0) == ([(0, 1, 5), (1, 1, 6), (2, 1, 7), (3, 253, 0)], math.inf)
    p.commit(3.0)
    assert p.step(3.0)[0][-1] == (3, 253, 253)
    p.close()


def test_status_codes():
    L = B.load()
    with pytest.raises(B.KsError) as e:
        B.Scheduler(0, 4, 16, 64)
    assert e.value.status == B.KS_EINVAL
    p = B.Scheduler(64, 4, 16, 4)
    with pytest.raises(B.KsError) as e:
        p.add_requests([0.0], [60], [10])                     # 70 tokens never fit 4 blocks of 16
    assert e.value.status == B.KS_EINVAL
    with pytest.raises(B.KsError):
        p.add_requests([float("nan")], [8], [1])
    with pytest.raises(B.KsError):
        p.add_requests([0.0], [0], [1])
    p.add_requests([0.0], [8], [2])
    with pytest.raises(B.KsError) as e:
        p.commit(1.0)                                         # nothing to commit
    assert e.value.status == B.KS_ESTATE
    assert p.step(0.0)[0] == [(0, 8, 0)]
    with pytest.raises(B.KsError) as e:
        p.step(0.5)                                           # previous batch not committed
    assert e.value.status == B.KS_ESTATE
    with pytest.raises(B.KsError) as e:
        p.add_requests([1.0], [8], [2])                       # the trace is fixed once the first step is formed
    assert e.value.status == B.KS_ESTATE
    p.commit(1.0)
    p.close()
    assert L.ks_sched_destroy(None) == B.KS_OK
    assert L.ks_sim_run(None, None, None, 0, None, None, 0, None, 0, None, None, 0, None, None) == B.KS_EINVAL
