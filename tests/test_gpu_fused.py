"""-m gpu: the one-kernel Tier-NONE path of ks_run_steps (ks_fused.cu: decode + roofline + floor + step sums + Eq. 4
for one spec vector in device space) against the two-call path (ks_predict_kernels + ks_compose_steps) and against
the CPU oracle.  PAPER.md:191 Eq. 2, :231, :233 Eq. 4.  Tolerance: 1e-5 relative (fp32 sums), and where both paths
stage a chunk the same way the outputs are bit-identical.
"""
import numpy as np
import pytest

from oracle import oracle as O
import workloads as W

pytestmark = pytest.mark.gpu

TOL_F32 = 1e-5


@pytest.fixture(scope="module")
def ks():
    import torch
    from paper_2606_28565_b200 import binding as B
    from paper_2606_28565_b200 import build as ksbuild
    from paper_2606_28565_b200 import driver as D
    ksbuild.build()
    assert torch.cuda.is_available()
    return B, D


def rel_err(got, want):
    want = np.asarray(want, np.float64)
    return np.abs(np.asarray(got, np.float64) - want) / np.maximum(np.abs(want), 1e-300)


def oracle_steps(w):
    lats = [O.predict_bucket(b, w.specs, W.TIER_NONE)["lat"][0] for b in w.buckets]
    so, to = O.compose(lats, [b.step_off for b in w.buckets], w.n_steps, w.step_params, w.cfg_off)
    return lats, so, to


def run_fused(B, D, ctx, w, db, with_lat):
    import torch
    n_cfg = len(w.cfg_off) - 1
    cfg = torch.from_numpy(np.ascontiguousarray(w.cfg_off, dtype=np.int32)).cuda()
    step = torch.full((1, w.n_steps), -1.0, dtype=torch.float32, device="cuda")
    tot = torch.full((1, max(n_cfg, 1)), -1.0, dtype=torch.float32, device="cuda")
    lat = [torch.full((1, b.n), -1.0, dtype=torch.float32, device="cuda") for b in db] if with_lat else None
    n0 = ctx.launch_count()
    ctx.run_steps(db, [b.step_off for b in db], w.specs, W.TIER_NONE, w.n_steps, w.step_params, cfg, n_cfg, step, tot,
                  latency=lat, space=B.KS_MEM_DEVICE)
    torch.cuda.synchronize()
    launches = ctx.launch_count() - n0
    return (step.cpu().numpy(), tot.cpu().numpy()[:, :n_cfg], [x.cpu().numpy() for x in lat] if with_lat else None,
            launches)


@pytest.mark.parametrize("n_steps,tp", [(771, 1), (64, 1), (1000, 2), (33, 4)])
def test_fused_run_steps_equals_two_calls_and_oracle(ks, n_steps, tp):
    B, D = ks
    w = W.config4(n_steps=n_steps, n_layers=5, tp=tp)
    ctx = B.Context(0)
    try:
        db = D.to_device(w)
        g = D.predict(ctx, w, dbuckets=db)
        step2, tot2 = D.compose(ctx, w, [x["lat_dev"] for x in g], db)
        step1, tot1, lat1, launches = run_fused(B, D, ctx, w, db, True)
        assert launches == 2                                  # the fused kernel and the totals kernel
        step0, tot0, _, _ = run_fused(B, D, ctx, w, db, False)  # step-only: no per-kernel latency is written
    finally:
        ctx.close()
    lats, so, to = oracle_steps(w)
    for a, b_, o in zip(lat1, g, lats):
        assert np.array_equal(a, b_["lat"])                   # the same device functions: the same bits
        assert rel_err(a[0], o).max(initial=0) <= TOL_F32
    assert rel_err(step1[0], so).max() <= TOL_F32 and rel_err(tot1[0], to).max() <= TOL_F32
    assert rel_err(step1[0], step2[0]).max() <= 2e-6 and rel_err(tot1[0], tot2[0]).max() <= 2e-6
    assert np.array_equal(step0, step1) and np.array_equal(tot0, tot1)


def test_fused_is_bit_identical_where_both_paths_stage(ks):
    """Row counts that are multiples of 4 (no array-end special case in the two-call path) and more than 16,384 steps
    (32-step chunks on both sides): the step latencies are bit-identical."""
    B, D = ks
    w = W.config4(n_steps=20_000, n_layers=4)
    assert all(b.n % 4 == 0 for b in w.buckets)
    ctx = B.Context(0)
    try:
        db = D.to_device(w)
        g = D.predict(ctx, w, dbuckets=db)
        step2, tot2 = D.compose(ctx, w, [x["lat_dev"] for x in g], db)
        step1, tot1, lat1, _ = run_fused(B, D, ctx, w, db, True)
        again = run_fused(B, D, ctx, w, db, True)
    finally:
        ctx.close()
    assert np.array_equal(step1, step2) and np.array_equal(tot1, tot2)
    assert all(np.array_equal(a, b_["lat"]) for a, b_ in zip(lat1, g))
    assert np.array_equal(again[0], step1) and np.array_equal(again[1], tot1)   # run-to-run


def test_fused_ragged_steps_empty_steps_and_a_chunk_that_does_not_fit(ks):
    """Hand-made step offsets over cfg2's three buckets: empty steps, single-row steps, one step of 30,000 rows (its
    chunk exceeds the staging buffer and is summed from the columns), offsets that are not multiples of 4, rows
    left over behind the last step, and a step count that is not a multiple of the chunk."""
    B, D = ks
    rng = np.random.Generator(np.random.PCG64(77))
    w = W.config2(n=240_011)
    n_steps = 1203
    w.tier = W.TIER_NONE
    for i, b in enumerate(w.buckets):
        cnt = rng.integers(0, max(2, (b.n - 31_000) // n_steps), n_steps)
        cnt[rng.random(n_steps) < 0.2] = 0
        cnt[rng.random(n_steps) < 0.1] = 1
        if i == 0:
            cnt[700] = 30_000
        cnt[-1] = 3
        assert 0 < cnt.sum() <= b.n - 5
        b.step_off = np.concatenate([[0], np.cumsum(cnt)]).astype(np.int32)
    w.n_steps = n_steps
    w.cfg_off = np.array([0, 1, 1, 500, 1203], np.int32)
    w.step_params = dict(c_disp=4e-6, floor_l=3e-4, c_ovl=2e-4, c_tail=1e-5, body_scale=1.25)
    ctx = B.Context(0)
    try:
        db = D.to_device(w)
        g = D.predict(ctx, w, dbuckets=db)
        step2, tot2 = D.compose(ctx, w, [x["lat_dev"] for x in g], db)
        step1, tot1, lat1, _ = run_fused(B, D, ctx, w, db, True)
    finally:
        ctx.close()
    lats, so, to = oracle_steps(w)
    assert rel_err(step1[0], so).max() <= TOL_F32 and rel_err(tot1[0], to).max() <= TOL_F32
    assert rel_err(step1[0], step2[0]).max() <= 2e-6
    for a, b_, bk in zip(lat1, g, w.buckets):
        used = int(bk.step_off[-1])
        assert np.array_equal(a[0, :used], b_["lat"][0, :used])
        assert np.all(a[0, used:] == -1.0)                     # rows behind the last step belong to no step: untouched


@pytest.mark.parametrize("tp", [1, 2])
def test_fused_weighted_rows_match_two_calls_and_oracle(ks, tp):
    """Layer-homogeneous rows (a row stands for m_k identical kernels): the one-kernel path stages
    m_k t_k and the multiplicities; per-kernel latencies stay unweighted and bit-identical, step latencies agree with
    ks_predict_kernels + ks_compose_steps_weighted to fp32 rounding (a product and a sum instead of one FMA) and with
    the oracle to 1e-5; Eq. 4's launch count is the sum of the multiplicities (c_disp = 4 us makes it visible)."""
    B, D = ks
    w = W.config4(n_steps=1203, n_layers=6, dedupe=True, tp=tp)
    assert any(b.mult is not None for b in w.buckets)
    ctx = B.Context(0)
    try:
        db = D.to_device(w)
        g = D.predict(ctx, w, dbuckets=db)
        step2, tot2 = D.compose(ctx, w, [x["lat_dev"] for x in g], db)
        step1, tot1, lat1, launches = run_fused(B, D, ctx, w, db, True)
        assert launches == 2
        step0, tot0, _, _ = run_fused(B, D, ctx, w, db, False)
    finally:
        ctx.close()
    lats = [O.predict_bucket(b, w.specs, W.TIER_NONE)["lat"][0] for b in w.buckets]
    so, to = O.compose(lats, [b.step_off for b in w.buckets], w.n_steps, w.step_params, w.cfg_off,
                       mults=[b.mult for b in w.buckets])
    assert all(np.array_equal(a, b_["lat"]) for a, b_ in zip(lat1, g))
    assert rel_err(step1[0], so).max() <= TOL_F32 and rel_err(tot1[0], to).max() <= TOL_F32
    assert rel_err(step1[0], step2[0]).max() <= 2e-6 and rel_err(tot1[0], tot2[0]).max() <= 2e-6
    assert np.array_equal(step0, step1) and np.array_equal(tot0, tot1)


def test_fused_six_buckets(ks):
    """More than four buckets (the closed loop's fine model slots make six): the eight-bucket instance."""
    B, D = ks
    rng = np.random.Generator(np.random.PCG64(5))
    w = W.config2(n=60_000)
    w.tier = W.TIER_NONE
    import copy
    w.buckets = w.buckets + [copy.deepcopy(b) for b in w.buckets]
    n_steps = 700
    for b in w.buckets:
        cnt = rng.multinomial(b.n - 7, np.full(n_steps, 1.0 / n_steps))
        b.step_off = np.concatenate([[0], np.cumsum(cnt)]).astype(np.int32)
    w.n_steps = n_steps
    w.cfg_off = np.array([0, 100, 700], np.int32)
    ctx = B.Context(0)
    try:
        db = D.to_device(w)
        g = D.predict(ctx, w, dbuckets=db)
        step2, tot2 = D.compose(ctx, w, [x["lat_dev"] for x in g], db)
        step1, tot1, lat1, launches = run_fused(B, D, ctx, w, db, True)
        assert launches == 2
    finally:
        ctx.close()
    lats, so, to = oracle_steps(w)
    assert rel_err(step1[0], so).max() <= TOL_F32 and rel_err(tot1[0], to).max() <= TOL_F32
    assert rel_err(step1[0], step2[0]).max() <= 2e-6
    for a, b_, bk in zip(lat1, g, w.buckets):
        used = int(bk.step_off[-1])
        assert np.array_equal(a[0, :used], b_["lat"][0, :used])


def test_fused_is_not_taken_with_several_specs(ks):
    """A spec sweep keeps the two-kernel path (three or more launches), with the same results as before."""
    B, D = ks
    import torch
    w = W.config4(n_steps=61, n_layers=6)
    w.specs = [W.spec_gb200(), W.spec_gb200(n_sm=132, peak_flops=1.0e15)]
    ctx = B.Context(0)
    try:
        db = D.to_device(w)
        n_cfg = len(w.cfg_off) - 1
        cfg = torch.from_numpy(np.ascontiguousarray(w.cfg_off, dtype=np.int32)).cuda()
        step = torch.empty((2, w.n_steps), dtype=torch.float32, device="cuda")
        tot = torch.empty((2, n_cfg), dtype=torch.float32, device="cuda")
        n0 = ctx.launch_count()
        ctx.run_steps(db, [b.step_off for b in db], w.specs, W.TIER_NONE, w.n_steps, w.step_params, cfg, n_cfg, step, tot)
        torch.cuda.synchronize()
        assert ctx.launch_count() - n0 >= 3
        step = step.cpu().numpy()
    finally:
        ctx.close()
    for s in range(2):
        lats = [O.predict_bucket(b, w.specs, W.TIER_NONE)["lat"][s] for b in w.buckets]
        so, _ = O.compose(lats, [b.step_off for b in w.buckets], w.n_steps, w.step_params, w.cfg_off)
        assert rel_err(step[s], so).max() <= TOL_F32
