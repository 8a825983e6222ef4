"""-m gpu: the closed simulation loop (ks_sim_run: host schedulers + one pass of the GPU path per iteration)
against the oracle (oracle/sched.py), SURVEY.md §8(f) NEXT-4.

The clock of a replica is a running sum of predicted step times, and the scheduler compares arrival times
with it, so an fp32-vs-fp64 difference in a step time could flip an admission.  The comparison therefore
replays the oracle scheduler on the CUDA path's logged step times (identical clocks => identical integer
decisions, checked bit for bit through the per-request results and counters) and checks every logged step
time against the oracle's own price of the same batch within the predictor's tolerance."""
import math

import numpy as np
import pytest

from oracle import sched as S
import workloads as W

pytestmark = pytest.mark.gpu
TOL = {W.TIER_NONE: 1e-5, W.TIER_A: 1e-2}


@pytest.fixture(scope="module")
def ks():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    from paper_2606_28565_b200 import binding as B
    from paper_2606_28565_b200 import build as ksbuild
    ksbuild.build()
    return B


def make_scheds(B, reps):
    out = []
    for r in reps:
        s = B.Scheduler(r.max_num_batched_tokens, r.max_num_seqs, r.block_size, r.num_blocks, r.enable_prefix_cache,
                        r.disk_blocks)
        s.add_requests(r.arrival, r.prompt_len, r.max_new, r.prefix_id, r.prefix_len)
        out.append(s)
    return out


def replay_and_check(B, reps, model, spec, tier, params, heads, scheds, clock, stats, rep_log, time_log):
    assert stats["steps"] == len(rep_log) == len(time_log)
    total_rows = total_inst = 0
    worst = 0.0
    for i, r in enumerate(reps):
        forced = time_log[rep_log == i].astype(np.float64)
        o = S.Scheduler(S.SchedConfig(r.max_num_batched_tokens, r.max_num_seqs, r.block_size, r.num_blocks,
                                      r.enable_prefix_cache, r.disk_blocks),
                        r.arrival, r.prompt_len, r.max_new, r.prefix_id, r.prefix_len)
        end, _, batches = S.simulate(o, lambda b: 0.0, forced=forced, max_steps=len(forced))
        assert len(batches) == len(forced)
        res = scheds[i].results()
        st = scheds[i].stats()
        # identical clocks => identical decisions: per-request times and counters are bit-equal
        assert np.array_equal(res["first_token"], np.array(o.first_token), equal_nan=True)
        assert np.array_equal(res["finish"], np.array(o.finish), equal_nan=True)
        assert res["n_preempt"].tolist() == o.n_preempt and res["cached_tokens"].tolist() == o.cached_tokens
        assert (st["gpu_hit_blocks"], st["disk_hit_blocks"], st["evictions"]) == (o.gpu_hit_blocks, o.disk_hit_blocks, o.evictions)
        assert (st["n_steps"], st["tokens_scheduled"], st["n_finished"]) == (o.n_steps, o.tokens_scheduled, o.n_finished)
        assert clock[i] == end
        # every step time the CUDA path produced vs the oracle's price of the same batch
        want = S.price_steps(batches, S.Model(**vars(model)), spec, tier, params, heads=heads)
        err = np.abs(forced - want) / want
        assert err.max() <= TOL[tier], f"replica {i}: step time rel err {err.max()}"
        worst = max(worst, float(err.max()))
        total_rows += sum(11 + len(b) + (1 if model.tp > 1 else 0) for b in batches)
        total_inst += sum(model.n_layers * (8 + len(b) + (2 if model.tp > 1 else 0)) + 3 for b in batches)
    assert stats["rows"] == total_rows and stats["kernel_instances"] == total_inst
    return worst


@pytest.mark.parametrize("tier,pressure,tp,prefix,fine",
                         [(W.TIER_NONE, False, 1, False, 0), (W.TIER_NONE, True, 4, False, 0), (W.TIER_A, False, 1, False, 0),
                          (W.TIER_NONE, True, 1, True, 0), (W.TIER_A, False, 1, False, 1), (W.TIER_A, True, 2, False, 1)])
def test_closed_loop_matches_oracle_replay(ks, tier, pressure, tp, prefix, fine):
    B = ks
    reps = W.sim_replicas(n_replicas=5, n_requests=40, seed=70 + tp, pressure=pressure)
    if prefix:          # shared system prompts + a two-tier prefix cache
        rng = np.random.Generator(np.random.PCG64(77))
        reps = [W.add_shared_prefixes(rng, r, disk_blocks=256) for r in reps]
    if pressure:        # a burst of requests into a cache of 1024 tokens: decoding outgrows it and forces recomputation
        for r in reps:
            r.prompt_len = np.minimum(r.prompt_len, 600).astype(np.int32)
            r.max_new = np.minimum(r.max_new, 200).astype(np.int32)
            r.arrival = r.arrival * 0.01
            r.num_blocks = 64
            if prefix:
                r.prefix_len = np.minimum(r.prefix_len, r.prompt_len).astype(np.int32)
    model = W.ServingModel(tp=tp, fine_slots=fine)
    spec = W.spec_gb200()
    params = W.STEP_PARAMS_CFG4
    heads = {}
    ctx = B.Context(0)
    try:
        if tier == W.TIER_A:
            rng = np.random.Generator(np.random.PCG64(1))
            # fine: the paper's finer families — LM head, prefill and decode attention priced by their
            # own slots, each with a different head; the plain attention slot stays empty on purpose
            slots = ((W.FAM_GEMM, W.SLOT_ATTN_PREFILL, W.FAM_ELEMWISE, W.SLOT_LM_HEAD, W.SLOT_ATTN_DECODE) if fine
                     else (W.FAM_GEMM, W.FAM_ATTN, W.FAM_ELEMWISE))
            heads = {f: W.make_head(rng, 12, 128) for f in slots}
            for f, h in heads.items():
                ctx.load_heads(f, h)
        scheds = make_scheds(B, reps)
        clock = np.zeros(len(reps), np.float64)
        stats, rep_log, time_log = B.sim_run(ctx, scheds, clock, model, spec, tier, params, log_cap=1 << 20)
        assert all(s.stats()["n_finished"] == s.n_requests for s in scheds)
        worst = replay_and_check(B, reps, model, spec, tier, params, heads, scheds, clock, stats, rep_log, time_log)
        print(f"sim tier {tier} pressure {pressure} tp {tp}: {stats}, max step-time rel err {worst:.2e}, "
              f"preemptions {sum(s.stats()['n_preemptions'] for s in scheds)}")
        if pressure:
            assert sum(s.stats()["n_preemptions"] for s in scheds) > 0
        if prefix:
            assert sum(s.stats()["gpu_hit_blocks"] for s in scheds) > 0
    finally:
        ctx.close()


def test_max_iters_resume_and_determinism(ks):
    B = ks
    reps = W.sim_replicas(n_replicas=4, n_requests=25, seed=75)
    model, spec, params = W.ServingModel(n_layers=8), W.spec_gb200(), W.STEP_PARAMS_HOSTBOUND
    ctx = B.Context(0)
    try:
        a = make_scheds(B, reps)
        ca = np.zeros(4)
        sa, ra, ta = B.sim_run(ctx, a, ca, model, spec, W.TIER_NONE, params, log_cap=1 << 18)
        # the same run cut into slices of 7 iterations: same log, same clocks
        b = make_scheds(B, reps)
        cb = np.zeros(4)
        rb, tb, iters = [], [], 0
        while True:
            s, r, t = B.sim_run(ctx, b, cb, model, spec, W.TIER_NONE, params, max_iters=7, log_cap=1 << 18)
            if s["iterations"] == 0:
                break
            assert s["iterations"] <= 7
            iters += s["iterations"]
            rb.append(r); tb.append(t)
        assert iters == sa["iterations"]
        assert np.array_equal(np.concatenate(rb), ra) and np.array_equal(np.concatenate(tb), ta)
        assert np.array_equal(ca, cb)
        for x, y in zip(a, b):
            assert np.array_equal(x.results()["finish"], y.results()["finish"])
        # host-bound Eq. 4 regime: every step costs at least floor_l + c_tail
        assert ta.min() >= np.float32(5e-3 + 5e-4) * (1 - 1e-6)
    finally:
        ctx.close()


def test_sim_argument_errors_and_empty(ks):
    B = ks
    ctx = B.Context(0)
    try:
        s = B.Scheduler(256, 4, 16, 64)
        clock = np.zeros(1)
        st, r, t = B.sim_run(ctx, [s], clock, W.ServingModel(), W.spec_gb200(), W.TIER_NONE, W.STEP_PARAMS_ZERO)
        assert st["steps"] == 0 and st["iterations"] == 0          # no requests: nothing to do
        with pytest.raises(B.KsError) as e:
            B.sim_run(ctx, [s], clock, W.ServingModel(n_layers=0), W.spec_gb200(), W.TIER_NONE, W.STEP_PARAMS_ZERO)
        assert e.value.status == B.KS_EINVAL
        with pytest.raises(B.KsError) as e:                        # Tier A without heads
            s2 = B.Scheduler(256, 4, 16, 64)
            s2.add_requests([0.0], [8], [2])
            B.sim_run(ctx, [s2], clock, W.ServingModel(), W.spec_gb200(), W.TIER_A, W.STEP_PARAMS_ZERO)
        assert e.value.status == B.KS_ESTATE
    finally:
        ctx.close()
