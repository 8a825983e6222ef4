"""Pins for the oracle's density-routed Tier B: interpolate the
measured grid inside the hull, fall back to the learned head outside.  The hull is the grid's box,
decided on integers (Q16)."""
import numpy as np

from oracle import oracle as O
import workloads as W


def setup(n=4001):
    w = W.config3(n=n, routed=True)
    heads = {f: O.Head(h) for f, h in w.heads.items()}
    grids = {f: O.Grid(g) for f, g in w.grids.items()}
    return w, heads, grids


def box_mask(bucket, grid):
    """In-hull decision restated independently with integer numpy compares."""
    if bucket.family == W.FAM_GEMM:
        axes = [bucket.cols[0], bucket.cols[1], bucket.cols[2]]
    else:
        axes = [bucket.cols[0], bucket.cols[1], np.maximum(bucket.cols[2], bucket.cols[1])]
    m = np.ones(bucket.n, bool)
    for a, v in enumerate(axes):
        lo, hi = int(np.ceil(2.0 ** float(grid.lo_log2[a]))), int(np.floor(2.0 ** float(grid.hi_log2[a])))
        m &= (v.astype(np.int64) >= lo) & (v.astype(np.int64) <= hi) & (v > 0)
    return m


def test_routing_selects_per_row_between_the_two_tiers():
    w, heads, grids = setup()
    for b in w.buckets:
        r = O.predict_bucket(b, w.specs, W.TIER_B_ROUTED, head=heads[b.slot], grid=grids[b.slot])
        tb = O.predict_bucket(b, w.specs, W.TIER_B, grid=grids[b.slot])
        ta = O.predict_bucket(b, w.specs, W.TIER_A, head=heads[b.slot])
        inside = box_mask(b, w.grids[b.slot])
        assert 0.80 < inside.mean() < 0.99                      # the recipe pushes ~5-10 % of the queries outside
        assert np.array_equal(r["routed"] == 0, inside)
        assert np.array_equal(r["lat"][0][inside], tb["lat"][0][inside])      # dense interior: measured grid
        assert np.array_equal(r["lat"][0][~inside], ta["lat"][0][~inside])    # edge: learned extrapolation
        assert np.array_equal(r["tiles"], tb["tiles"]) and np.array_equal(r["waves"], tb["waves"])


def test_hull_boundary_is_inclusive_and_decided_on_integers():
    w, heads, grids = setup(n=64)
    g = w.grids[W.FAM_GEMM]                                     # spans log2 M [0,13], N [10,14], K [10,14]
    cols = [np.array([1, 8192, 8193, 1, 1, 1, 0], np.int32), np.array([1024, 16384, 1024, 1023, 16385, 4096, 4096], np.int32),
            np.array([1024, 16384, 1024, 1024, 1024, 1023, 4096], np.int32)]
    b = W.Bucket(W.FAM_GEMM, cols)
    r = O.predict_bucket(b, w.specs, W.TIER_B_ROUTED, head=heads[W.FAM_GEMM], grid=grids[W.FAM_GEMM])
    assert list(r["routed"]) == [0, 0, 1, 1, 1, 1, 1]           # corners in; one past any edge out; M = 0 out


def test_flat_axes_do_not_constrain_and_bounded_fallback():
    rng = np.random.Generator(np.random.PCG64(3))
    grid = W.Grid(np.array([4, 1, 1], np.int32), np.array([12, 0, 0], np.float32), np.array([20, 0, 0], np.float32),
                  rng.uniform(0.3, 0.9, (4, 1, 1)).astype(np.float32))
    b = W.Bucket(W.FAM_ELEMWISE, [np.array([4096, 1 << 20, 4095, (1 << 20) + 1], np.int32), np.array([0, 5, 2, 3], np.int32)])
    bh = O.Bounded(W.make_bounded_head(rng, 12))
    spec = [W.spec_gb200(t0=1e-9)]
    r = O.predict_bucket(b, spec, W.TIER_B_ROUTED, grid=O.Grid(grid), bounded=bh)
    assert list(r["routed"]) == [0, 0, 1, 1]
    ta = O.predict_bucket(b, spec, W.TIER_A, bounded=bh)
    assert np.array_equal(r["lat"][0][2:], ta["lat"][0][2:])


def test_all_inside_equals_tier_b_and_all_outside_equals_tier_a():
    w, heads, grids = setup(n=64)
    inside = W.Bucket(W.FAM_GEMM, [np.array([64, 512], np.int32), np.array([4096, 8192], np.int32), np.array([2048, 4096], np.int32)])
    outside = W.Bucket(W.FAM_GEMM, [np.array([64, 512], np.int32), np.array([512, 100000], np.int32), np.array([2048, 4096], np.int32)])
    h, g = heads[W.FAM_GEMM], grids[W.FAM_GEMM]
    assert np.array_equal(O.predict_bucket(inside, w.specs, 3, head=h, grid=g)["lat"], O.predict_bucket(inside, w.specs, 2, grid=g)["lat"])
    assert np.array_equal(O.predict_bucket(outside, w.specs, 3, head=h, grid=g)["lat"], O.predict_bucket(outside, w.specs, 1, head=h)["lat"])
