"""-m gpu: parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(device-resident buffers, no auxiliary outputs unless noted), on sampled outputs the oracle computes
one by one (every k-th row of every bucket plus the first and last 300 rows: tile boundaries and
ragged tails), plus properties that hold at any size.  Tolerances as in test_gpu_parity.py.
"""
import numpy as np
import pytest

from oracle import oracle as O
import workloads as W

pytestmark = pytest.mark.gpu

TOL_F32 = 1e-5
TOL_MLP = 1e-2


@pytest.fixture(scope="module")
def ks():
    import torch
    from paper_2606_28565_b200 import binding as B
    from paper_2606_28565_b200 import build as ksbuild
    from paper_2606_28565_b200 import driver as D
    ksbuild.build()
    assert torch.cuda.is_available()
    return B, D


def sample_rows(n, stride, edge=300):
    r = np.unique(np.concatenate([np.arange(0, n, stride), np.arange(min(edge, n)), np.arange(max(n - edge, 0), n)]))
    return r.astype(np.int64)


def rel(got, want):
    want = np.asarray(want, np.float64)
    return np.abs(np.asarray(got, np.float64) - want) / np.maximum(np.abs(want), 1e-300)


def predict_full(ks, w, aux=False):
    B, D = ks
    ctx = B.Context(0)
    try:
        D.load_models(ctx, w)
        db = D.to_device(w)
        g = D.predict(ctx, w, dbuckets=db, aux=aux)
        step = tot = None
        if w.n_steps and all(b.step_off is not None for b in w.buckets):
            step, tot = D.compose(ctx, w, [x["lat_dev"] for x in g], db)
    finally:
        ctx.close()
    return g, step, tot


def check_sampled(w, g, stride, tol, tier=None):
    tier = w.tier if tier is None else tier
    heads = {f: O.Head(h) for f, h in w.heads.items()} if tier == W.TIER_A else {}
    grids = {f: O.Grid(x) for f, x in w.grids.items()} if tier == W.TIER_B else {}
    worst = 0.0
    for b, gi in zip(w.buckets, g):
        rows = sample_rows(b.n, stride)
        o = O.predict_bucket(b, w.specs, tier, head=heads.get(b.slot), grid=grids.get(b.slot), rows=rows)
        e = rel(gi["lat"][:, rows], o["lat"]).max(initial=0)
        assert e <= tol, f"{w.name} family {b.family}: sampled latency rel err {e}"
        assert np.all(np.isfinite(gi["lat"])) and np.all(gi["lat"] >= np.float32(w.specs[0]["t0"]) * (1 - 1e-6))
        worst = max(worst, float(e))
    return worst


def test_cfg2_full_tier_a_and_composition(ks):
    w = W.config2()                                   # 1,000,000 descriptors: the bench workload
    g, step, tot = predict_full(ks, w)
    print("cfg2 full: sampled max rel err", check_sampled(w, g, 997, TOL_MLP))
    # composition over ALL rows of the GPU latencies against the oracle's sums (same inputs)
    so, to = O.compose([x["lat"][0] for x in g], [b.step_off for b in w.buckets], w.n_steps, w.step_params, w.cfg_off)
    assert rel(step[0], so).max() <= TOL_F32 and rel(tot[0], to).max() <= TOL_F32


def check_composition(w, g, step, tot, specs=None):
    """Step and configuration latencies of ALL steps against the oracle's composer (O.compose: naive segment loops in
    double, Eq. 4) fed with the GPU's own per-kernel latencies, per spec."""
    n_cfg = len(w.cfg_off) - 1
    for s in (range(len(w.specs)) if specs is None else specs):
        so, to = O.compose([x["lat"][s] for x in g], [b.step_off for b in w.buckets], w.n_steps, w.step_params, w.cfg_off,
                           mults=[b.mult for b in w.buckets])
        assert rel(step[s], so).max() <= TOL_F32, f"{w.name}: step latencies of spec {s}"
        assert rel(tot[s][:n_cfg], to).max() <= TOL_F32, f"{w.name}: configuration totals of spec {s}"


def test_cfg3_full_tier_b(ks):
    w = W.config3()                                   # 4,194,304 grid queries
    g, step, tot = predict_full(ks, w, aux=True)
    print("cfg3 full: sampled max rel err", check_sampled(w, g, 4099, TOL_F32))
    check_composition(w, g, step, tot)                # 16,384 steps, 16 configurations
    t0 = w.specs[0]["t0"]
    for b, gi in zip(w.buckets, g):
        # interpolation never leaves [min, max] of the grid, so on EVERY row
        # max(t_roof / e_max, t0) <= t <= max(t_roof / e_min, t0)
        gmin, gmax = float(w.grids[b.slot].values.min()), float(w.grids[b.slot].values.max())
        tr = gi["troof"].astype(np.float64)
        assert np.all(gi["lat"] >= np.maximum(tr / gmax, t0) * (1 - 2e-6))
        assert np.all(gi["lat"] <= np.maximum(tr / gmin, t0) * (1 + 2e-6))


def test_cfg4_full_tier_none_closed_form(ks):
    w = W.config4()                                   # 100,000 steps, ~29.9M kernel instances
    g, step, tot = predict_full(ks, w)
    print("cfg4a full: sampled max rel err", check_sampled(w, g, 20011, TOL_F32))
    # every step: Tier NONE is the closed form sum(max(t_roof, t0)) + n c_disp, checked on
    # ALL steps against numpy segment sums of the GPU's own per-kernel latencies in fp64
    tot_ref = np.zeros(w.n_steps)
    cnt = np.zeros(w.n_steps)
    for b, gi in zip(w.buckets, g):
        cs = np.concatenate([[0.0], np.cumsum(gi["lat"][0].astype(np.float64))])
        tot_ref += cs[b.step_off[1:]] - cs[b.step_off[:-1]]
        cnt += np.diff(b.step_off)
    want = tot_ref + cnt * w.step_params["c_disp"]
    assert rel(step[0], want).max() <= TOL_F32
    cfg_ref = np.add.reduceat(want, w.cfg_off[:-1])
    assert rel(tot[0], cfg_ref).max() <= TOL_F32
    check_composition(w, g, step, tot)                # and against the oracle's own composer


def test_cfg4b_full_tier_a(ks):
    w = W.config4(tier=W.TIER_A)                      # the same 100,000 steps through the Tier-A heads (29.9M rows)
    g, step, tot = predict_full(ks, w)
    print("cfg4b full: sampled max rel err", check_sampled(w, g, 50021, TOL_MLP))
    check_composition(w, g, step, tot)


def test_cfg5_full_what_if_sweep(ks):
    w = W.config5()                                   # 64 specs x 4,194,304 rows = 268,435,456 predictions
    g, step, tot = predict_full(ks, w)
    print("cfg5 full: sampled max rel err", check_sampled(w, g, 65521, TOL_MLP))
    # a descriptor's latency is a function of (row, spec) only: rows that repeat (layer-homogeneous
    # descriptors within a step) must give bit-identical predictions under every spec
    b, gi = w.buckets[0], g[0]
    key = np.stack([c[:200000] for c in b.cols], axis=1)
    _, first, inv = np.unique(key, axis=0, return_index=True, return_inverse=True)
    assert np.array_equal(gi["lat"][:, :200000], gi["lat"][:, first[inv.ravel()]])
    # the 64-spec x 10.9k-step composition (spec_stride, chunk indexing): every step of every spec
    check_composition(w, g, step, tot)
