"""-m gpu: parity of the CUDA path (through the C ABI) against the CPU oracle, element by element
on the same seeded inputs.  Tolerances are BASELINE.json's: bit-exact integers (tiles, waves,
counts), <= 1e-5 relative for the fp32 roofline / interpolation / sum paths, <= 1e-2 relative on
latency for the bf16 tensor-core MLP path.
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


def rel_err(got, want):
    want = np.asarray(want, np.float64)
    return np.abs(np.asarray(got, np.float64) - want) / np.maximum(np.abs(want), 1e-300)


def oracle_all(w, tier=None, rows=None):
    tier = w.tier if tier is None else tier
    heads = {f: O.Head(h) for f, h in w.heads.items()} if tier == W.TIER_A else {}
    grids = {f: O.Grid(g) for f, g in w.grids.items()} if tier == W.TIER_B else {}
    out = []
    for i, b in enumerate(w.buckets):
        r = None if rows is None else rows[i]
        bnd = O.Bounded(w.bounded[b.slot]) if (tier == W.TIER_A and b.slot in getattr(w, "bounded", {})) else None
        ens = O.Ensemble(w.ensembles[b.slot]) if (tier == W.TIER_A and b.slot in getattr(w, "ensembles", {})) else None
        out.append(O.predict_bucket(b, w.specs, tier, head=heads.get(b.slot), grid=grids.get(b.slot), rows=r,
                                    bounded=bnd, ensemble=ens))
    return out


def check_bucket(g, o, tol, rows=None, what=""):
    sel = (lambda a: a) if rows is None else (lambda a: a[:, rows])
    assert np.array_equal(sel(g["tiles"]), o["tiles"]), f"{what}: tiles not bit-exact"
    assert np.array_equal(sel(g["waves"]), o["waves"]), f"{what}: waves not bit-exact"
    e_tr = rel_err(sel(g["troof"]), o["troof"])
    e_tr[o["troof"] == 0] = np.abs(sel(g["troof"]))[o["troof"] == 0]
    assert e_tr.max(initial=0) <= TOL_F32, f"{what}: t_roof rel err {e_tr.max()}"
    e = rel_err(sel(g["lat"]), o["lat"])
    assert e.max(initial=0) <= tol, f"{what}: latency rel err {e.max()}"
    return float(e.max(initial=0))


def run_and_check(ks, w, tol, tier=None, gelu_mode=0):
    B, D = ks
    ctx = B.Context(0)
    try:
        D.load_models(ctx, w)
        ctx.set_gelu_mode(gelu_mode)
        g = D.predict(ctx, w, tier=tier)
    finally:
        ctx.close()
    o = oracle_all(w, tier)
    return [check_bucket(gi, oi, tol, what=f"{w.name}/bucket{i}") for i, (gi, oi) in enumerate(zip(g, o))]


# ------------------------------------------------------------------ Tier NONE (S1, S2, S5)
@pytest.mark.parametrize("make", [lambda: W.config1(), lambda: W.config2(n=30011),
                                  lambda: W.config4(n_steps=60), lambda: W.config5(n_rows=20003, n_specs=3)])
def test_tier_none_parity(ks, make):
    w = make()
    run_and_check(ks, w, TOL_F32, tier=W.TIER_NONE)


def test_degenerate_rows_and_clamps(ks):
    spec = [W.spec_gb200(tile_m=96, tile_n=160, ctas_per_sm=2, ew_elems_per_cta=1000)]
    i32 = lambda *a: [np.asarray(x, np.int32) for x in a]
    buckets = [
        W.Bucket(W.FAM_GEMM, i32([0, 5, 1, 2 ** 20, 7], [8, 0, 1, 4096, 9], [8, 8, 0, 64, 3])),
        W.Bucket(W.FAM_GROUPED, i32([256] * 3, [64] * 3, *[[0, 1, 5000]] * 1, *[[0, 0, 17]] * 7)),
        W.Bucket(W.FAM_ATTN, i32([1, 3, 0, 2], [1, 700, 5, 64], [1, 100, 9, 64]), hq=32, hkv=8, head_dim=128),  # kv<q raised
        W.Bucket(W.FAM_ELEMWISE, i32([0, 1, 999, 1000, 1001, 5], [0, 1, 2, 3, 9, -4])),                       # subop clamped
    ]
    w = W.Workload("edge", buckets, spec, W.TIER_NONE)
    run_and_check(ks, w, TOL_F32)


@pytest.mark.parametrize("n", [1, 3, 4, 127, 128, 129, 1027])
def test_ragged_tails_and_misaligned_spec_stride(ks, n):
    w = W.config2(n=10 * n)      # buckets of 5n, 3n, 2n rows; n_specs = 3 makes spec rows start unaligned
    w.specs = [W.spec_gb200(), W.spec_gb200(n_sm=80, peak_bw=2e12), W.spec_gb200(tile_m=64, t0=1e-9)]
    run_and_check(ks, w, TOL_F32, tier=W.TIER_NONE)
    run_and_check(ks, w, TOL_MLP, tier=W.TIER_A)


def test_small_multi_bucket_call_equals_per_bucket_calls(ks):
    # a Tier-NONE call with several buckets and <= 32768 rows takes the one-launch thread-per-row kernel; the same
    # buckets one call each take the streaming kernel: same device functions, same bits (incl. Eq. 3 rows, fp32 columns)
    B, D = ks
    w = W.config4(n_steps=40, tp=4, n_layers=4)
    w.specs = [W.spec_gb200(), W.spec_gb200(n_sm=96, peak_bw=3e12, ar_beta_eff=4e11)]
    assert len(w.buckets) == 4 and sum(b.n for b in w.buckets) <= 32768
    ctx = B.Context(0)
    try:
        launches0 = ctx.launch_count()
        together = D.predict(ctx, w, tier=W.TIER_NONE)
        assert ctx.launch_count() - launches0 == 1
        for i, b in enumerate(w.buckets):
            one = W.Workload("one", [b], w.specs, W.TIER_NONE)
            alone = D.predict(ctx, one, tier=W.TIER_NONE)[0]
            for k in ("lat", "tiles", "waves", "troof"):
                assert np.array_equal(together[i][k], alone[k]), (i, k)
    finally:
        ctx.close()
    o = oracle_all(w, W.TIER_NONE)
    for i, (gi, oi) in enumerate(zip(together, o)):
        check_bucket(gi, oi, TOL_F32, what=f"small call / bucket {i}")


# ------------------------------------------------------------------ Tier B (S4b)
def test_tier_b_parity(ks):
    errs = run_and_check(ks, W.config3(n=60001), TOL_F32)
    print("tier B max rel err", errs)


def test_tier_b_nodes_exact_and_flat_axes(ks):
    B, D = ks
    rng = np.random.default_rng(11)
    # queries exactly on grid nodes (integer log2 coordinates) must return the node value
    vals = rng.uniform(0.2, 0.95, (8, 8, 8)).astype(np.float32)
    grid = W.Grid(np.array([8, 8, 8], np.int32), np.zeros(3, np.float32), np.full(3, 7, np.float32), vals)
    idx = rng.integers(0, 8, (500, 3))
    cols = [np.left_shift(1, idx[:, a]).astype(np.int32) for a in range(3)]
    spec = W.spec_gb200(t0=0.0)
    w = W.Workload("nodes", [W.Bucket(W.FAM_GEMM, cols)], [spec], W.TIER_B, grids={W.FAM_GEMM: grid})
    ctx = B.Context(0)
    D.load_models(ctx, w)
    g = D.predict(ctx, w)[0]
    e = g["troof"][0].astype(np.float64) / g["lat"][0].astype(np.float64)
    assert np.allclose(e, vals[idx[:, 0], idx[:, 1], idx[:, 2]], rtol=3e-7)
    # elementwise family: sub-op axis nodes + one flat axis
    ev = rng.uniform(0.2, 0.95, (32, 6, 1)).astype(np.float32)
    ge = W.Grid(np.array([32, 6, 1], np.int32), np.array([12, 0, 0], np.float32), np.array([25, 5, 0], np.float32), ev)
    ne, sub = W._elem_rows(rng, 5000)
    w2 = W.Workload("ew", [W.Bucket(W.FAM_ELEMWISE, W._i32(ne, sub))], [W.spec_gb200()], W.TIER_B,
                    grids={W.FAM_ELEMWISE: ge})
    D.load_models(ctx, w2)
    g2 = D.predict(ctx, w2)
    ctx.close()
    check_bucket(g2[0], oracle_all(w2)[0], TOL_F32, what="elementwise grid")


def _tierb_bucket(rng, fam, n, lo, hi, dtype=np.int32):
    """n rows whose axis values straddle the span [lo, hi] (log2), with zeros, ones, exact span ends and huge values."""
    lo, hi = np.asarray(lo, np.float64), np.asarray(hi, np.float64)
    x = rng.uniform(lo[None, :] - 1.5, hi[None, :] + 1.5, size=(n, 3))
    v = np.maximum(np.rint(np.exp2(x)), 0).astype(np.int64)
    k = min(n, 12)
    # (the CTA count B must stay below 2^31, Q1: the huge values go to the third axis, K or kv, which B ignores)
    special = np.array([0, 1, 2, 3, 2 ** 31 - 1, 2 ** 24 + 1, 2 ** 24 - 1, 255, 256, 257, 65535, 65537])[:k]
    for a in range(3):
        v[:k, a] = np.roll(np.minimum(special, 2 ** 31 - 1 if a == 2 else 65537), a)
        if n > 20:   # the exact span ends (integers there are hull corners) and one beyond each
            for j, e in enumerate((np.ceil(2.0 ** lo[a]), np.floor(2.0 ** hi[a]), np.floor(2.0 ** hi[a]) + 1)):
                v[12 + 3 * a + j if 12 + 3 * a + j < n else 0, a] = int(e)
    v = np.minimum(v, 2 ** 31 - 1)
    if fam == W.FAM_ATTN:
        kw = dict(hq=24, hkv=3, head_dim=96)
    else:
        kw = {}
    if dtype == np.float32:          # F32 columns hold exact integers < 2^24
        v = np.minimum(v, 2 ** 24 - 1)
    return W.Bucket(fam, [np.ascontiguousarray(v[:, a], dtype=dtype) for a in range(3)], **kw)


@pytest.mark.parametrize("dims,n_specs,dtype,n", [((7, 33, 5), 1, np.int32, 8191), ((2, 2, 300), 3, np.int32, 4097),
                                                  ((32, 1, 31), 1, np.float32, 5), ((1, 64, 64), 2, np.float32, 12289),
                                                  ((16, 16, 16), 1, np.int32, 1), ((2, 2, 8192), 1, np.int32, 3000)])
def test_tier_b_kernel_edge_cases(ks, dims, n_specs, dtype, n):
    # ks_tierb.cu away from the 32^3 / one-spec / int32 configuration: odd and flat dims (the zero tail behind the grid is
    # what the corners one past an axis read), fractional and large lo, several specs (the 512-thread instance), fp32
    # columns, ragged tails of 1..3 rows, values 0, 1, 2^31-1, span ends; five buckets = two launches of <= 4 buckets
    B, D = ks
    rng = np.random.Generator(np.random.PCG64(hash((dims, n_specs, n)) % 1000))
    spans = {W.FAM_GEMM: ((0.5, 3.25, 9.0), (11.75, 14.0, 20.5)), W.FAM_ATTN: ((0.0, 0.0, 1.3), (7.0, 12.6, 17.0))}
    specs = W.sweep_specs(rng, n_specs)
    specs[0].update(tile_m=96, tile_n=1, ctas_per_sm=3)           # divisors that are not powers of two, and a divisor of one
    buckets, grids = [], {}
    for i, fam in enumerate((W.FAM_GEMM, W.FAM_ATTN, W.FAM_GEMM, W.FAM_ATTN, W.FAM_GEMM)):
        lo, hi = spans[fam]
        slot = 8 + i                                               # five slots, five different grids
        b = _tierb_bucket(rng, fam, n if i != 3 else max(1, n // 3), lo, hi, dtype)
        b.model_slot = slot
        buckets.append(b)
        # (fp32 interpolation holds 1e-5 RELATIVE only where e is not tiny next to large neighbours: config-like values;
        # the last bucket's grid is a constant below the 2^-10 guard, so every row there comes out at t_roof * 2^10)
        vals = W.make_grid(rng, lo, hi, dims=dims).values if i < 4 else np.full(dims, 2.0 ** -12, np.float32)
        for a in range(3):          # an axis of hundreds of nodes asks more of an fp32 coordinate than 1e-5 leaves: flat there
            if dims[a] > 64:
                vals = np.ascontiguousarray(np.broadcast_to(np.take(vals, [0], axis=a), dims))
        grids[slot] = W.Grid(np.asarray(dims, np.int32), np.asarray(lo, np.float32), np.asarray(hi, np.float32), vals)
    w = W.Workload("tierb_edges", buckets, specs, W.TIER_B, grids=grids)
    errs = run_and_check(ks, w, TOL_F32)
    print(dims, n_specs, n, "tier-B edge max rel err", errs)


# ------------------------------------------------------------------ Tier A (S3, S4a)
@pytest.mark.parametrize("make", [lambda: W.config1(), lambda: W.config2(n=40013),
                                  lambda: W.config5(n_rows=12001, n_specs=3, n_layers=4),
                                  lambda: W.config4(n_steps=40, tier=W.TIER_A, n_layers=4)])
def test_tier_a_parity(ks, make):
    w = make()
    errs = run_and_check(ks, w, TOL_MLP)
    print(w.name, "tier A max rel err per bucket", errs)
    assert max(errs) < TOL_MLP


@pytest.mark.parametrize("n_in,h", [(12, 128), (32, 256), (8, 64)])
def test_tier_a_log_eta_output(ks, n_in, h):
    # heads whose output is log eta: eta = exp(max(z, 0)) instead of 1 / sigmoid(z); same kernels,
    # one branch-free epilogue.  Biases are spread so that both z < 0 (eta = 1: the bound) and z > 0 occur.
    w = W.config2(n=20011, n_in=n_in, h=h)
    rng = np.random.Generator(np.random.PCG64(300 + h))
    w.heads = {f: W.make_head(rng, n_in, h, bias_std=0.3) for f in w.heads}
    for hd in w.heads.values():
        hd.out_mode = W.HEAD_LOG_ETA
    B, D = ks
    ctx = B.Context(0)
    try:
        D.load_models(ctx, w)
        g = D.predict(ctx, w)
        # back to the utilisation convention on the same loaded weights: a different prediction
        for f in w.heads:
            ctx.set_head_output(f, B.KS_HEAD_UTILISATION)
        g0 = D.predict(ctx, w)
    finally:
        ctx.close()
    o = oracle_all(w)
    errs = [check_bucket(gi, oi, TOL_MLP, what=f"log-eta/bucket{i}") for i, (gi, oi) in enumerate(zip(g, o))]
    print(n_in, h, "log-eta max rel err", errs)
    at_bound = sum(int(np.sum(oi["lat"] == np.maximum(oi["troof"], w.specs[0]["t0"]))) for oi in o)
    above = sum(int(np.sum(oi["lat"] > 1.01 * np.maximum(oi["troof"], w.specs[0]["t0"]))) for oi in o)
    assert at_bound > 100 and above > 100                       # both regimes of max(z, 0) are exercised
    for hd in w.heads.values():
        hd.out_mode = W.HEAD_UTILISATION
    o0 = oracle_all(w)
    for gi, oi in zip(g0, o0):
        check_bucket(gi, oi, TOL_MLP, what="utilisation after switching back")
    assert any(np.max(rel_err(a["lat"], b_["lat"])) > 0.05 for a, b_ in zip(g, g0))


@pytest.mark.parametrize("tier", [W.TIER_A, W.TIER_B, W.TIER_B_ROUTED, W.TIER_NONE])
def test_model_slots_eight_paper_families(ks, tier):
    # PAPER.md:199 / Tables 2 and 4: eta is learned per kernel family — GEMM, LM head, attention prefill and decode,
    # RMSNorm, SiLU x Mul, RoPE, KV-cache write.  Eight buckets, eight model slots, eight different heads and grids
    # in ONE call; two buckets of one decode family must get their own model.
    w = W.config_families(n=40_000, tier=tier)
    B, D = ks
    ctx = B.Context(0)
    try:
        D.load_models(ctx, w)
        db = D.to_device(w)
        g = D.predict(ctx, w, dbuckets=db)
        step, tot = D.compose(ctx, w, [x["lat_dev"] for x in g], db)
        # a bucket whose slot holds no model is refused before anything runs
        if tier != W.TIER_NONE:
            bad = W.Bucket(W.FAM_GEMM, w.buckets[0].cols, model_slot=14)
            import torch
            lat = [torch.empty((1, bad.n), dtype=torch.float32, device="cuda:0")]
            with pytest.raises(B.KsError) as ei:
                ctx.predict_kernels(D.to_device(W.Workload("bad", [bad], w.specs, tier)), w.specs, tier, lat)
            assert ei.value.status == B.KS_ESTATE
    finally:
        ctx.close()
    heads = {s: O.Head(h) for s, h in w.heads.items()}
    grids = {s: O.Grid(x) for s, x in w.grids.items()}
    tol = TOL_F32 if tier in (W.TIER_B, W.TIER_NONE) else TOL_MLP
    lats = []
    for i, (b, gi) in enumerate(zip(w.buckets, g)):
        o = O.predict_bucket(b, w.specs, tier, head=heads.get(b.slot), grid=grids.get(b.slot))
        if tier == W.TIER_B_ROUTED:                               # in-hull rows: the fp32 path; routed rows: the bf16 path
            assert np.array_equal(gi["tiles"], o["tiles"]) and np.array_equal(gi["waves"], o["waves"])
            e, out = rel_err(gi["lat"], o["lat"]), o["routed"] == 1
            assert e[:, ~out].max(initial=0) <= TOL_F32 and e[:, out].max(initial=0) <= TOL_MLP, f"slot {b.slot}"
        else:
            check_bucket(gi, o, tol, what=f"slot {b.slot}")
        lats.append(gi["lat"][0])
        if tier == W.TIER_A and b.model_slot is not None:
            # priced with the decode family's default model instead, the bucket comes out different: the slot matters
            other = O.predict_bucket(b, w.specs, tier, head=heads[w.buckets[0].slot if b.family == W.FAM_GEMM else
                                                                  W.SLOT_ATTN_PREFILL if b.slot == W.SLOT_ATTN_DECODE else
                                                                  W.SLOT_ATTN_DECODE if b.slot == W.SLOT_ATTN_PREFILL else
                                                                  W.SLOT_RMSNORM if b.slot != W.SLOT_RMSNORM else W.SLOT_ROPE])
            assert np.max(rel_err(gi["lat"], other["lat"])) > 2 * TOL_MLP
    so, to = O.compose(lats, [b.step_off for b in w.buckets], w.n_steps, w.step_params, w.cfg_off)
    assert np.max(rel_err(step[0], so)) <= TOL_F32 and np.max(rel_err(tot[0], to)) <= TOL_F32


@pytest.mark.parametrize("n_in,h", [(8, 64), (8, 128), (12, 64), (12, 256), (32, 64), (32, 128), (8, 256)])
def test_tier_a_all_head_shapes_with_wide_weights(ks, n_in, h):
    # wider weights (std 0.25) push pre-activations to |x| ~ 2-3 where the tanh-form GELU differs most
    w = W.config2(n=6007, n_in=n_in, h=h)
    rng = np.random.Generator(np.random.PCG64(100 + n_in + h))
    w.heads = {f: W.make_head(rng, n_in, h, bias_std=0.2, w_std=0.25 if h < 256 else 0.15) for f in w.heads}
    errs = run_and_check(ks, w, TOL_MLP)
    print(n_in, h, "wide-weight max rel err", errs)


def test_tier_a_and_composition_are_bit_reproducible(ks):
    # no atomics, fixed reduction orders, one warp-specialized pipeline per SM: two runs of the same call (and a run
    # on a second context) give identical bits, for 128- and 256-wide heads and for the step composition
    B, D = ks
    for w in (W.config2(n=50021), W.config5(n_rows=30011, n_specs=3, n_layers=4)):
        outs = []
        for rep in range(3):
            ctx = B.Context(0)
            try:
                D.load_models(ctx, w)
                db = D.to_device(w)
                g = D.predict(ctx, w, dbuckets=db)
                step, tot = D.compose(ctx, w, [x["lat_dev"] for x in g], db)
                outs.append(([x["lat"].copy() for x in g], step.copy(), tot.copy()))
            finally:
                ctx.close()
        for o in outs[1:]:
            assert all(np.array_equal(a, b) for a, b in zip(o[0], outs[0][0]))
            assert np.array_equal(o[1], outs[0][1]) and np.array_equal(o[2], outs[0][2])


def test_tier_a_packed_gelu_mode_within_tolerance(ks):
    w = W.config2(n=40013)
    errs = run_and_check(ks, w, TOL_MLP, gelu_mode=1)
    print("gelu_mode=1 max rel err", errs)


def test_zero_weight_head_is_exact_closed_form(ks):
    B, D = ks
    w = W.config1()
    w.heads = {W.FAM_GEMM: W.make_head(np.random.default_rng(0), 8, 64, bias_std=0.0, w_std=0.0)}
    ctx = B.Context(0)
    D.load_models(ctx, w)
    g = D.predict(ctx, w)[0]
    ctx.close()
    want = np.maximum(2.0 * g["troof"][0], np.float32(2e-6))     # e = 0.5 exactly -> eta = 2
    assert np.array_equal(g["lat"][0], want.astype(np.float32))


# ------------------------------------------------------------------ S6 / S7
@pytest.mark.parametrize("params", [W.STEP_PARAMS_CFG4, W.STEP_PARAMS_HOSTBOUND,
                                    dict(c_disp=1e-6, floor_l=0.0, c_ovl=0.0, c_tail=1e-5, body_scale=1.25)])
def test_compose_parity(ks, params):
    B, D = ks
    w = W.config4(n_steps=700, n_cfg=9, step_params=params)
    ctx = B.Context(0)
    db = D.to_device(w)
    g = D.predict(ctx, w, dbuckets=db)
    step, tot = D.compose(ctx, w, [x["lat_dev"] for x in g], db)
    ctx.close()
    o = oracle_all(w)
    # same per-kernel inputs on both sides: feed the oracle's composer the GPU's fp32 latencies
    so, to = O.compose([x["lat"][0] for x in g], [b.step_off for b in w.buckets], w.n_steps, params, w.cfg_off)
    assert rel_err(step[0], so).max() <= TOL_F32
    assert rel_err(tot[0], to).max() <= TOL_F32
    # and end to end against the pure-oracle pipeline
    so2, to2 = O.compose([x["lat"][0] for x in o], [b.step_off for b in w.buckets], w.n_steps, params, w.cfg_off)
    assert rel_err(step[0], so2).max() <= TOL_F32 and rel_err(tot[0], to2).max() <= TOL_F32


def test_compose_ones_empty_segments_and_multi_spec(ks):
    import torch
    B, D = ks
    rng = np.random.default_rng(3)
    n_steps, ns = 257, 3
    ns_rows = [1000, 37]
    offs = [np.concatenate([[0], np.sort(rng.integers(0, n + 1, n_steps - 1)), [n]]).astype(np.int32) for n in ns_rows]
    lat = [rng.uniform(1e-6, 1e-3, (ns, n)).astype(np.float32) for n in ns_rows]
    cfg = np.array([0, 0, 100, 257], np.int32)                        # first config empty
    ctx = B.Context(0)
    dl = [torch.from_numpy(x).cuda() for x in lat]
    do = [torch.from_numpy(x).cuda() for x in offs]
    step = torch.empty((ns, n_steps), dtype=torch.float32, device="cuda")
    tot = torch.empty((ns, 3), dtype=torch.float32, device="cuda")
    ctx.compose_steps(dl, do, ns_rows, n_steps, ns, W.STEP_PARAMS_HOSTBOUND, torch.from_numpy(cfg).cuda(), 3, step, tot)
    torch.cuda.synchronize()
    for s in range(ns):
        so, to = O.compose([x[s] for x in lat], offs, n_steps, W.STEP_PARAMS_HOSTBOUND, cfg)
        assert rel_err(step[s].cpu().numpy(), so).max() <= TOL_F32
        assert np.allclose(tot[s].cpu().numpy(), to, rtol=TOL_F32, atol=0)
    ones = [torch.ones((1, n), dtype=torch.float32, device="cuda") for n in ns_rows]
    step1 = torch.empty((1, n_steps), dtype=torch.float32, device="cuda")
    tot1 = torch.empty((1, 3), dtype=torch.float32, device="cuda")
    ctx.compose_steps(ones, do, ns_rows, n_steps, 1, W.STEP_PARAMS_ZERO, torch.from_numpy(cfg).cuda(), 3, step1, tot1)
    torch.cuda.synchronize()
    ctx.close()
    assert np.array_equal(step1[0].cpu().numpy(), (np.diff(offs[0]) + np.diff(offs[1])).astype(np.float32))
    assert np.array_equal(tot1[0].cpu().numpy(), np.array([0, offs[0][100] + offs[1][100],
                                                           1037 - offs[0][100] - offs[1][100]], np.float32))


# ------------------------------------------------------------------ ABI behaviour on the device
def test_host_space_equals_device_space_and_run_steps(ks):
    import torch
    B, D = ks
    w = W.config2(n=20011)
    ctx = B.Context(0)
    D.load_models(ctx, w)
    db = D.to_device(w)
    g = D.predict(ctx, w, dbuckets=db)
    step_d, tot_d = D.compose(ctx, w, [x["lat_dev"] for x in g], db)
    n_cfg = w.cfg_off.shape[0] - 1
    # host space through ks_predict_kernels
    lat_h = [np.empty((1, b.n), np.float32) for b in w.buckets]
    tiles_h = [np.empty((1, b.n), np.int32) for b in w.buckets]
    ctx.predict_kernels(w.buckets, w.specs, w.tier, lat_h, tiles=tiles_h)
    for i in range(len(w.buckets)):
        assert np.array_equal(lat_h[i], g[i]["lat"]) and np.array_equal(tiles_h[i], g[i]["tiles"])
    # host space through the fused ks_run_steps
    step_h, tot_h = np.empty((1, w.n_steps), np.float32), np.empty((1, n_cfg), np.float32)
    lat_h2 = [np.empty((1, b.n), np.float32) for b in w.buckets]
    ctx.run_steps(w.buckets, [b.step_off for b in w.buckets], w.specs, w.tier, w.n_steps, w.step_params,
                  w.cfg_off, n_cfg, step_h, tot_h, latency=lat_h2)
    assert np.array_equal(step_h, step_d) and np.array_equal(tot_h, tot_d)
    assert all(np.array_equal(a, b["lat"]) for a, b in zip(lat_h2, g))
    # device space run_steps without returning per-kernel latencies; determinism (bit-identical rerun)
    cfg = torch.from_numpy(w.cfg_off).cuda()
    s1 = torch.empty((1, w.n_steps), dtype=torch.float32, device="cuda")
    t1 = torch.empty((1, n_cfg), dtype=torch.float32, device="cuda")
    for _ in range(2):
        ctx.run_steps(db, [b.step_off for b in db], w.specs, w.tier, w.n_steps, w.step_params, cfg, n_cfg, s1, t1)
        torch.cuda.synchronize()
        assert np.array_equal(s1.cpu().numpy(), step_d) and np.array_equal(t1.cpu().numpy(), tot_d)
    assert ctx.launch_count() > 0
    ctx.close()


def test_status_codes_on_device(ks):
    import torch
    B, D = ks
    w = W.config2(n=1000)
    ctx = B.Context(0)
    db = D.to_device(w)
    lat = [torch.empty((1, b.n), dtype=torch.float32, device="cuda") for b in db]
    with pytest.raises(B.KsError) as e:
        ctx.predict_kernels(db, w.specs, W.TIER_A, lat)              # heads not loaded
    assert e.value.status == B.KS_ESTATE
    with pytest.raises(B.KsError) as e:
        ctx.predict_kernels(db, w.specs, W.TIER_B, lat)              # grids not loaded
    assert e.value.status == B.KS_ESTATE
    bad = W.make_head(np.random.default_rng(0), 12, 96)
    with pytest.raises(B.KsError) as e:
        ctx.load_heads(W.FAM_GEMM, bad)
    assert e.value.status == B.KS_EUNSUPPORTED
    sentinel = torch.full((1, db[0].n + 1), -1.0, dtype=torch.float32, device="cuda")
    with pytest.raises(B.KsError) as e:                              # misaligned device output
        ctx.predict_kernels(db[:1], w.specs, W.TIER_NONE, [sentinel[0, 1:]])
    assert e.value.status == B.KS_EINVAL and bool((sentinel == -1.0).all())   # nothing was written
    badspec = [W.spec_gb200(n_sm=0)]
    with pytest.raises(B.KsError) as e:
        ctx.predict_kernels(db, badspec, W.TIER_NONE, lat)
    assert e.value.status == B.KS_EINVAL
    empty = W.Workload("empty", [W.Bucket(W.FAM_GEMM, W._i32([], [], []))], w.specs, W.TIER_NONE)
    ctx.predict_kernels(D.to_device(empty), w.specs, W.TIER_NONE, [torch.empty((1, 0), device="cuda")])   # n = 0 no-op
    ctx.close()


# ------------------------------------------------------------------ TP all-reduce rows (Eq. 3, NEXT-3)
@pytest.mark.parametrize("tier", [W.TIER_NONE, W.TIER_A])
def test_allreduce_family_and_tp_steps(ks, tier):
    B, D = ks
    w = W.config4(n_steps=37, n_layers=3, tier=tier, tp=4)
    w.specs = [W.spec_gb200(ar_alpha0=7e-6, ar_beta_eff=450e9), W.spec_gb200(ar_alpha0=0.0, ar_beta_eff=900e9, t0=5e-6)]
    ctx = B.Context(0)
    try:
        D.load_models(ctx, w)
        db = D.to_device(w)
        g = D.predict(ctx, w, dbuckets=db)
        step, tot = D.compose(ctx, w, [x["lat_dev"] for x in g], db)
    finally:
        ctx.close()
    o = oracle_all(w, tier)
    assert w.buckets[-1].family == W.FAM_ALLREDUCE
    for i, (gi, oi) in enumerate(zip(g, o)):
        check_bucket(gi, oi, TOL_F32 if (tier == W.TIER_NONE or i == 3) else TOL_MLP, what=f"{w.name}/bucket{i}")
    assert np.all(g[3]["tiles"] == 0) and np.all(g[3]["waves"] == 0)
    for s in range(2):                                 # the all-reduce rows enter the step sum like kernels
        so, to = O.compose([x["lat"][s] for x in g], [b.step_off for b in w.buckets], w.n_steps, w.step_params, w.cfg_off)
        assert rel_err(step[s], so).max() <= TOL_F32 and rel_err(tot[s], to).max() <= TOL_F32


def test_allreduce_degenerate_rows(ks):
    B, D = ks
    cols = [np.array([0, 1, 1 << 30, 4096, 4096, 4096], np.int32), np.array([8, 1, 2, 0, -3, 1 << 20], np.int32)]
    w = W.Workload("ar_edge", [W.Bucket(W.FAM_ALLREDUCE, cols)], [W.spec_gb200(ar_alpha0=3e-6, ar_beta_eff=100e9)], W.TIER_B)
    ctx = B.Context(0)
    try:
        g = D.predict(ctx, w)                          # Tier B without any grid loaded: Eq. 3 rows need none
    finally:
        ctx.close()
    o = oracle_all(w, W.TIER_NONE)
    check_bucket(g[0], o[0], TOL_F32, what="ar_edge")


# ------------------------------------------------------------------ bounded analytical head (NEXT-2)
TOL_BOUNDED = TOL_F32   # an fp32 path: features through MUFU log2 into two 22-term dot products (measured 1.3e-6)


@pytest.mark.parametrize("make,n_in", [(lambda: W.config2(n=30011), 12), (lambda: W.config1(), 8),
                                       (lambda: W.config5(n_rows=20003, n_specs=3, n_layers=4), 32)])
def test_bounded_head_parity(ks, make, n_in):
    B, D = ks
    w = make()
    rng = np.random.Generator(np.random.PCG64(11 + n_in))
    fams = [b.family for b in w.buckets]
    # every other family gets the bounded form, the rest keep their MLP heads: both kinds in one call
    w.bounded = {f: W.make_bounded_head(rng, n_in) for f in fams[::2]}
    w.heads = {f: h for f, h in w.heads.items() if f not in w.bounded}
    ctx = B.Context(0)
    try:
        D.load_models(ctx, w)
        g = D.predict(ctx, w)
    finally:
        ctx.close()
    o = oracle_all(w, W.TIER_A)
    errs = [check_bucket(gi, oi, TOL_BOUNDED if b.family in w.bounded else TOL_MLP, what=f"{w.name}/bucket{i}")
            for i, (b, gi, oi) in enumerate(zip(w.buckets, g, o))]
    print("bounded head max rel err per bucket", errs, "bounded families", sorted(w.bounded))


def test_bounded_head_closed_forms_and_replacement(ks):
    B, D = ks
    w = W.config1()
    fam = w.buckets[0].family
    zero = np.zeros(8, np.float32)
    ctx = B.Context(0)
    try:
        D.load_models(ctx, w)                                     # MLP head first ...
        ctx.load_bounded_head(fam, W.BoundedHead(8, zero, 0.0, zero, -1.0))   # ... replaced: gamma = 1/2, alpha = 0
        g = D.predict(ctx, w)
        half = np.maximum(2.0 * g[0]["troof"].astype(np.float64), w.specs[0]["t0"])
        assert rel_err(g[0]["lat"], half).max() <= 1e-6           # eta = 2 exactly, floor after eta
        ctx.load_bounded_head(fam, W.BoundedHead(8, zero, 60.0, zero, -1.0))  # gamma -> 1: attains the bound
        g = D.predict(ctx, w)
        assert rel_err(g[0]["lat"], np.maximum(g[0]["troof"].astype(np.float64), w.specs[0]["t0"])).max() <= 1e-6
        ctx.load_heads(fam, w.heads[fam])                         # and back to the MLP head
        g = D.predict(ctx, w)
    finally:
        ctx.close()
    check_bucket(g[0], oracle_all(w)[0], TOL_MLP, what="cfg1 after reloading the MLP head")
    with pytest.raises(Exception):
        c2 = B.Context(0)
        try:
            c2.load_bounded_head(fam, W.BoundedHead(9, np.zeros(9, np.float32), 0.0, np.zeros(9, np.float32), 0.0))
        finally:
            c2.close()


# ------------------------------------------------------------------ MLP ensembles (NEXT-2, Q17)
@pytest.mark.parametrize("n_in,h,k", [(12, 32, 4), (12, 64, 2), (8, 32, 2), (32, 64, 4), (32, 128, 2), (12, 32, 8)])
def test_ensemble_parity(ks, n_in, h, k):
    B, D = ks
    w = W.config2(n=20011, n_in=n_in, h=h * k) if n_in != 32 else W.config5(n_rows=12007, n_specs=3, n_layers=4, h=h * k)
    rng = np.random.Generator(np.random.PCG64(1000 + n_in + h + k))
    fams = [b.family for b in w.buckets]
    # every other family gets an ensemble of k members of width h, the rest keep a single head of width k h:
    # both kinds share the kernel launch
    w.ensembles = {f: W.make_ensemble(rng, n_in, h, k, bias_std=0.2, w_std=0.2) for f in fams[::2]}
    w.heads = {f: hd for f, hd in w.heads.items() if f not in w.ensembles}
    ctx = B.Context(0)
    try:
        D.load_models(ctx, w)
        g = D.predict(ctx, w)
    finally:
        ctx.close()
    o = oracle_all(w, W.TIER_A)
    errs = [check_bucket(gi, oi, TOL_MLP, what=f"{w.name}/bucket{i}") for i, (gi, oi) in enumerate(zip(g, o))]
    print("ensemble", (n_in, h, k), "max rel err per bucket", errs, "ensemble families", sorted(w.ensembles))


def test_ensemble_closed_forms_reductions_and_shapes(ks):
    B, D = ks
    w = W.config1()
    fam = w.buckets[0].family
    z = np.zeros

    def const_member(h, b3):
        return W.Head(8, h, h, z((8, h), np.float32), z(h, np.float32), z((h, h), np.float32), z(h, np.float32),
                      z(h, np.float32), float(b3))

    rng = np.random.Generator(np.random.PCG64(5))
    one = W.make_head(rng, 8, 64, bias_std=0.2, w_std=0.2)
    ctx = B.Context(0)
    try:
        # members with constant outputs 0.8 and 0.5: e = 0.65 (the mean of the efficiencies, Q17)
        ctx.load_head_ensemble(fam, [const_member(32, np.log(4.0)), const_member(32, 0.0)])
        g = D.predict(ctx, w)
        want = np.maximum(g[0]["troof"].astype(np.float64) / 0.65, w.specs[0]["t0"])
        assert rel_err(g[0]["lat"], want).max() <= 2e-6
        # two copies of one member = that member alone (different kernel shape, same arithmetic up to rounding)
        ctx.load_heads(fam, one)
        single = D.predict(ctx, w)[0]["lat"].copy()
        ctx.load_head_ensemble(fam, [one, one])
        twice = D.predict(ctx, w)[0]["lat"]
        assert rel_err(twice, single).max() <= 2e-6
        ctx.load_head_ensemble(fam, [one])                        # k = 1 is the plain head, bit for bit
        assert np.array_equal(D.predict(ctx, w)[0]["lat"], single)
        for h, k in ((16, 4), (32, 3), (64, 8), (128, 4), (32, 9)):
            with pytest.raises(B.KsError) as ei:
                ctx.load_head_ensemble(fam, [const_member(h, 0.0)] * k)
            assert ei.value.status == B.KS_EUNSUPPORTED
    finally:
        ctx.close()


# ------------------------------------------------------------------ density-routed Tier B (NEXT-1)
def routed_oracle(w):
    heads = {f: O.Head(h) for f, h in w.heads.items()}
    grids = {f: O.Grid(g) for f, g in w.grids.items()}
    return [O.predict_bucket(b, w.specs, W.TIER_B_ROUTED, head=heads.get(b.slot), grid=grids[b.slot],
                             bounded=O.Bounded(w.bounded[b.slot]) if b.slot in w.bounded else None)
            for b in w.buckets]


def check_routed(g, o, what):
    """In-hull rows are an fp32 path (1e-5), rows routed to an MLP head the bf16 path (1e-2)."""
    for i, (gi, oi) in enumerate(zip(g, o)):
        assert np.array_equal(gi["tiles"], oi["tiles"]) and np.array_equal(gi["waves"], oi["waves"])
        e = rel_err(gi["lat"], oi["lat"])
        out = oi["routed"] == 1
        assert e[:, ~out].max(initial=0) <= TOL_F32, f"{what}/bucket{i}: in-hull rel err {e[:, ~out].max()}"
        assert e[:, out].max(initial=0) <= TOL_MLP, f"{what}/bucket{i}: routed rel err {e[:, out].max()}"
        assert out.any() and (~out).any()


@pytest.mark.parametrize("n,n_specs", [(30011, 1), (5003, 3)])
def test_density_routing_parity(ks, n, n_specs):
    B, D = ks
    w = W.config3(n=n, routed=True)
    w.specs = [W.spec_gb200(), W.spec_gb200(n_sm=132, peak_flops=1.0e15, peak_bw=3.35e12, t0=3e-6),
               W.spec_gb200(ctas_per_sm=2)][:n_specs]
    ctx = B.Context(0)
    try:
        D.load_models(ctx, w)
        db = D.to_device(w)
        g = D.predict(ctx, w, dbuckets=db)
        g2 = D.predict(ctx, w, dbuckets=db)                           # the row lists are rebuilt per call
        step, tot = D.compose(ctx, w, [x["lat_dev"] for x in g], db)
    finally:
        ctx.close()
    o = routed_oracle(w)
    check_routed(g, o, w.name)
    for a, b_ in zip(g, g2):                                           # list order varies, results must not
        assert np.array_equal(a["lat"], b_["lat"])
    so, to = O.compose([x["lat"][0] for x in g], [b.step_off for b in w.buckets], w.n_steps, w.step_params, w.cfg_off)
    assert rel_err(step[0], so).max() <= TOL_F32 and rel_err(tot[0], to).max() <= TOL_F32


def test_density_routing_with_bounded_fallback_and_256_heads(ks):
    B, D = ks
    rng = np.random.Generator(np.random.PCG64(21))
    w = W.config3(n=9001, routed=True, n_in=32, h=256)                # attention keeps a 32->256->256->1 MLP head ...
    w.bounded = {W.FAM_GEMM: W.make_bounded_head(rng, 12)}             # ... GEMM falls back to the bounded form
    del w.heads[W.FAM_GEMM]
    ctx = B.Context(0)
    try:
        D.load_models(ctx, w)
        g = D.predict(ctx, w)
    finally:
        ctx.close()
    check_routed(g, routed_oracle(w), w.name)


def test_density_routing_host_space_and_missing_models(ks):
    B, D = ks
    import torch
    w = W.config3(n=4001, routed=True)
    ctx = B.Context(0)
    try:
        for fam, gr in w.grids.items():
            ctx.load_grid(fam, gr)
        db = D.to_device(w)
        lat = [torch.empty((1, b.n), dtype=torch.float32, device="cuda:0") for b in db]
        with pytest.raises(B.KsError) as ei:                           # grids alone are not enough: the fallback needs heads
            ctx.predict_kernels(db, w.specs, W.TIER_B_ROUTED, lat, space=B.KS_MEM_DEVICE)
        assert ei.value.status == B.KS_ESTATE
        D.load_models(ctx, w)
        g = D.predict(ctx, w, dbuckets=db, aux=False)
        hb = D.to_pinned(w)
        step_h = torch.empty((1, w.n_steps), dtype=torch.float32).pin_memory()
        tot_h = torch.empty((1, len(w.cfg_off) - 1), dtype=torch.float32).pin_memory()
        lat_h = [torch.empty((1, b.n), dtype=torch.float32).pin_memory() for b in hb]
        cfg_h = torch.from_numpy(np.ascontiguousarray(w.cfg_off, dtype=np.int32)).pin_memory()
        ctx.run_steps(hb, [b.step_off for b in hb], w.specs, W.TIER_B_ROUTED, w.n_steps, w.step_params, cfg_h,
                      len(w.cfg_off) - 1, step_h, tot_h, latency=lat_h, space=B.KS_MEM_HOST)
    finally:
        ctx.close()
    for a, b_ in zip(g, lat_h):
        assert np.array_equal(a["lat"], b_.numpy())                    # host space runs the same kernels


# ------------------------------------------------------------------ layer-homogeneous composition
@pytest.mark.parametrize("tier", [W.TIER_NONE, W.TIER_A])
def test_layer_homogeneous_steps_match_oracle_and_materialised_steps(ks, tier):
    B, D = ks
    import torch
    full = W.config4(n_steps=61, n_layers=6, tier=tier, tp=2)
    ded = W.config4(n_steps=61, n_layers=6, tier=tier, tp=2, dedupe=True)
    assert ded.n_rows * 4 < full.n_rows
    out = {}
    ctx = B.Context(0)
    try:
        for name, w in (("full", full), ("ded", ded)):
            D.load_models(ctx, w)
            db = D.to_device(w)
            g = D.predict(ctx, w, dbuckets=db)
            out[name] = (g,) + D.compose(ctx, w, [x["lat_dev"] for x in g], db)
        # the same through ks_run_steps in host space (multiplicities travel in ks_desc_batch.mult)
        hb = D.to_pinned(ded)
        n_cfg = len(ded.cfg_off) - 1
        step_h = torch.empty((1, ded.n_steps), dtype=torch.float32).pin_memory()
        tot_h = torch.empty((1, n_cfg), dtype=torch.float32).pin_memory()
        cfg_h = torch.from_numpy(np.ascontiguousarray(ded.cfg_off, dtype=np.int32)).pin_memory()
        ctx.run_steps(hb, [b.step_off for b in hb], ded.specs, tier, ded.n_steps, ded.step_params, cfg_h, n_cfg,
                      step_h, tot_h, space=B.KS_MEM_HOST)
    finally:
        ctx.close()
    g, step, tot = out["ded"]
    so, to = O.compose([x["lat"][0] for x in g], [b.step_off for b in ded.buckets], ded.n_steps, ded.step_params,
                       ded.cfg_off, mults=[b.mult for b in ded.buckets])
    assert rel_err(step[0], so).max() <= TOL_F32 and rel_err(tot[0], to).max() <= TOL_F32
    assert np.array_equal(step_h.numpy(), step) and np.array_equal(tot_h.numpy(), tot)
    # L identical kernels summed one by one or taken L times: the same step up to fp32 rounding of the sums
    assert rel_err(step[0], out["full"][1][0]).max() <= 2 * TOL_F32
    assert rel_err(tot[0], out["full"][2][0]).max() <= 2 * TOL_F32


# ------------------------------------------------------------------ holes named by the round-1 review
def grouped_grid_workload(n=20011, routed=False, seed=31):
    """A grouped-GEMM bucket (cfg5's MoE rows: N, K, m_0..m_7) against a 12 x 5 x 6 grid over (sum m, N, K) with a
    different span on every axis; about a fifth of the rows lie outside the hull (small or huge token totals)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    T = W._log_uniform_int(rng, 1, 1 << 15, n)                      # tokens routed top-2: sum m = 2 T
    m = rng.multinomial(2 * T, np.full(8, 1 / 8)).astype(np.int64)
    N = np.array([4096, 5120, 8192, 14336, 28672], np.int64)[rng.integers(0, 5, n)]
    K = np.array([2048, 4096, 8192, 14336], np.int64)[rng.integers(0, 4, n)]
    m[rng.random(n) < 0.01] = 0                                     # a few rows without any token (B = 0)
    grid = W.make_grid(rng, (3.0, 12.0, 11.0), (14.0, 15.0, 13.9), dims=(12, 5, 6))
    bk = W.Bucket(W.FAM_GROUPED, W._i32(N, K, *[m[:, e] for e in range(8)]))
    heads = {W.FAM_GROUPED: W.make_head(rng, 32, 256)} if routed else {}
    return W.Workload("grouped_grid", [bk], [W.spec_gb200(), W.spec_gb200(n_sm=132, tile_m=64, peak_bw=3.35e12)],
                      W.TIER_B_ROUTED if routed else W.TIER_B, grids={W.FAM_GROUPED: grid}, heads=heads)


def test_tier_b_grouped_gemm_bucket(ks):
    # the 512-thread Tier-B instance, grid axes (sum m, N, K) and the integer hull test of the grouped family
    w = grouped_grid_workload()
    errs = run_and_check(ks, w, TOL_F32)
    print("grouped-GEMM Tier B max rel err", errs)


def test_density_routing_grouped_gemm_bucket(ks):
    B, D = ks
    w = grouped_grid_workload(n=9001, routed=True)
    ctx = B.Context(0)
    try:
        D.load_models(ctx, w)
        g = D.predict(ctx, w)
    finally:
        ctx.close()
    o = routed_oracle(w)
    check_routed(g, o, w.name)
    frac = float(o[0]["routed"].mean())
    assert 0.05 < frac < 0.6, frac


@pytest.mark.parametrize("n_specs", [65, 130])
def test_more_specs_than_one_launch_holds(ks, n_specs):
    # n_specs > 64 is split into launches of <= 64 specs (output offset s0 x n; the routed row list is built once)
    B, D = ks
    rng = np.random.Generator(np.random.PCG64(77))
    specs = W.sweep_specs(rng, n_specs)
    for k in range(0, n_specs, 7):
        specs[k]["tile_m"], specs[k]["ctas_per_sm"] = 64, 2
    rows = [np.arange(0, 3001, 13)]
    # Tier NONE and Tier A on a cfg2-like mix (three buckets), spec 64 onward is the second launch
    w = W.config2(n=3001 * 2)
    w.specs = specs
    for tier, tol in ((W.TIER_NONE, TOL_F32), (W.TIER_A, TOL_MLP)):
        ctx = B.Context(0)
        try:
            D.load_models(ctx, w)
            db = D.to_device(w)
            g = D.predict(ctx, w, dbuckets=db, tier=tier)
            step, tot = D.compose(ctx, w, [x["lat_dev"] for x in g], db)
        finally:
            ctx.close()
        o = oracle_all(w, tier)
        for i, (gi, oi) in enumerate(zip(g, o)):
            check_bucket(gi, oi, tol, what=f"{n_specs} specs tier {tier} bucket {i}")
        for s in (0, 63, 64, n_specs - 1):
            so, to = O.compose([x["lat"][s] for x in g], [b.step_off for b in w.buckets], w.n_steps, w.step_params, w.cfg_off)
            assert rel_err(step[s], so).max() <= TOL_F32 and rel_err(tot[s], to).max() <= TOL_F32
    # density-routed Tier B
    w3 = W.config3(n=4001, routed=True)
    w3.specs = specs
    ctx = B.Context(0)
    try:
        D.load_models(ctx, w3)
        g = D.predict(ctx, w3)
    finally:
        ctx.close()
    check_routed(g, routed_oracle(w3), f"routed, {n_specs} specs")


@pytest.mark.parametrize("s", [1, 4])
def test_dtype_bytes_one_and_four(ks, s):
    # the element size s of the modelled kernel (fp8 / fp32 tensors) enters F_mem and feature 11
    for make, tier, tol in ((lambda: W.config2(n=9001), W.TIER_NONE, TOL_F32), (lambda: W.config2(n=9001), W.TIER_A, TOL_MLP),
                            (lambda: W.config5(n_rows=9001, n_specs=2, n_layers=4), W.TIER_A, TOL_MLP),
                            (lambda: W.config3(n=9001), W.TIER_B, TOL_F32)):
        w = make()
        for b in w.buckets:
            b.dtype_bytes = s
        run_and_check(ks, w, tol, tier=tier)
    # and it changes the answer: a memory-bound GEMM row moves s/2 times the bytes
    B, D = ks
    w = W.config1()
    ctx = B.Context(0)
    try:
        base = D.predict(ctx, w, tier=W.TIER_NONE)[0]["troof"]
        w.buckets[0].dtype_bytes = s
        got = D.predict(ctx, w, tier=W.TIER_NONE)[0]["troof"]
    finally:
        ctx.close()
    M = w.buckets[0].cols[0]
    mem_bound = M <= 16                                                # AI < ridge for these rows
    assert rel_err(got[0][mem_bound], base[0][mem_bound] * (s / 2)).max() <= 2e-6


def test_compose_many_steps_odd_stride_two_specs(ks):
    # n_steps x n_specs > 16384 takes the 32-step chunks; odd bucket sizes make spec 1's rows start unaligned
    import torch
    B, D = ks
    rng = np.random.default_rng(5)
    n_steps, ns = 9001, 2
    ns_rows = [270031, 90007, 13]
    offs = [np.concatenate([[0], np.sort(rng.integers(0, n + 1, n_steps - 1)), [n]]).astype(np.int32) for n in ns_rows]
    lat = [rng.uniform(1e-6, 1e-3, (ns, n)).astype(np.float32) for n in ns_rows]
    cfg = np.array([0, 17, 17, 4000, 9001], np.int32)
    ctx = B.Context(0)
    try:
        dl = [torch.from_numpy(x).cuda() for x in lat]
        do = [torch.from_numpy(x).cuda() for x in offs]
        step = torch.empty((ns, n_steps), dtype=torch.float32, device="cuda")
        tot = torch.empty((ns, 4), dtype=torch.float32, device="cuda")
        ctx.compose_steps(dl, do, ns_rows, n_steps, ns, W.STEP_PARAMS_HOSTBOUND, torch.from_numpy(cfg).cuda(), 4, step, tot)
        torch.cuda.synchronize()
    finally:
        ctx.close()
    for s in range(ns):
        so, to = O.compose([x[s] for x in lat], offs, n_steps, W.STEP_PARAMS_HOSTBOUND, cfg)
        assert rel_err(step[s].cpu().numpy(), so).max() <= TOL_F32
        assert np.allclose(tot[s].cpu().numpy(), to, rtol=TOL_F32, atol=0)
