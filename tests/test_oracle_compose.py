"""Pins for the oracle's S6/S7 (segmented sums, Eq. 4, config totals) — PAPER.md:231-235."""
import numpy as np
import pytest

from oracle import oracle as O
import workloads as W

ZERO = dict(W.STEP_PARAMS_ZERO)


def _offs(rng, n, n_steps):
    return W.uniform_step_offsets(rng, n, n_steps)


def test_ones_give_segment_lengths_and_config_counts():
    rng = np.random.default_rng(0)
    offs = [_offs(rng, 1000, 37), _offs(rng, 333, 37)]
    lats = [np.ones(1000), np.ones(333)]
    cfg = W.cfg_offsets(rng, 37, 5)
    step, tot = O.compose(lats, offs, 37, ZERO, cfg)
    want = np.diff(offs[0]) + np.diff(offs[1])
    assert np.array_equal(step, want.astype(np.float64))
    assert np.array_equal(tot, np.add.reduceat(np.append(want, 0), cfg[:-1])[:5] * (np.diff(cfg) > 0))
    # config totals of all-ones step latencies = steps per config
    one_per_step = [np.ones(37)]
    step1, tot1 = O.compose(one_per_step, [np.arange(38)], 37, ZERO, cfg)
    assert np.array_equal(tot1, np.diff(cfg).astype(np.float64))


def test_segment_sums_vs_reduceat_and_cumsum():
    rng = np.random.default_rng(1)
    n, n_steps = 5000, 211
    lat = rng.uniform(1e-6, 1e-3, n)
    off = np.sort(rng.integers(0, n + 1, n_steps - 1))
    off = np.concatenate([[0], off, [n]]).astype(np.int64)           # includes empty segments
    step, _ = O.compose([lat], [off], n_steps, ZERO, np.array([0, n_steps]))
    cs = np.concatenate([[0.0], np.cumsum(lat)])
    assert np.allclose(step, cs[off[1:]] - cs[off[:-1]], rtol=1e-10, atol=1e-18)
    assert np.all(step[np.diff(off) == 0] == 0.0)


def test_eq4_regimes():
    # one step, t_gpu = 3e-3 from 3 kernels
    lat, off, cfg = [np.full(3, 1e-3)], [np.array([0, 3])], np.array([0, 1])
    gpu_bound = dict(c_disp=4e-6, floor_l=1e-3, c_ovl=2e-3, c_tail=5e-4, body_scale=1.0)
    s, _ = O.compose(lat, off, 1, gpu_bound, cfg)
    assert s[0] == pytest.approx(3e-3 + 3 * 4e-6 + 5e-4, rel=1e-14)   # t_gpu + n c_disp + c_tail
    host_bound = dict(c_disp=4e-6, floor_l=5e-3, c_ovl=8e-3, c_tail=5e-4, body_scale=1.0)
    s, _ = O.compose(lat, off, 1, host_bound, cfg)
    assert s[0] == pytest.approx(5e-3 + (8e-3 - 3e-3) + 5e-4, rel=1e-14)  # l + (c_ovl - t_gpu) + c_tail
    scaled = dict(c_disp=0.0, floor_l=0.0, c_ovl=0.0, c_tail=0.0, body_scale=1.25)
    s, _ = O.compose(lat, off, 1, scaled, cfg)
    assert s[0] == pytest.approx(1.25 * 3e-3, rel=1e-14)
    # empty step: t_gpu = 0, n = 0 -> max(0, l) + c_ovl + c_tail
    s, _ = O.compose([np.zeros(0)], [np.array([0, 0])], 1, host_bound, cfg)
    assert s[0] == pytest.approx(5e-3 + 8e-3 + 5e-4, rel=1e-14)
    # cfg-4 constants: sum t + 4e-6 n
    s, _ = O.compose(lat, off, 1, dict(W.STEP_PARAMS_CFG4), cfg)
    assert s[0] == pytest.approx(3e-3 + 12e-6, rel=1e-14)


def test_tier_none_pipeline_is_a_closed_form():
    # eta == 1: step latency = sum max(t_roof, t0) + n c_disp, t_roof from the golden GEMM cases
    spec = W.spec_gb200()
    b = W.Bucket(W.FAM_GEMM, [np.array([8192, 1, 1]), np.array([8192, 8192, 8]), np.array([8192, 8192, 8])])
    out = O.predict_bucket(b, [spec], W.TIER_NONE)
    assert np.array_equal(out["tiles"][0], [4096, 64, 1]) and np.array_equal(out["waves"][0], [28, 1, 1])
    want = [4.943984576284444e-04, 1.6781312e-05, 2e-6]
    assert np.allclose(out["lat"][0], want, rtol=1e-13)
    step, tot = O.compose([out["lat"][0]], [np.array([0, 2, 3])], 2, dict(W.STEP_PARAMS_CFG4), np.array([0, 2]))
    assert step[0] == pytest.approx(want[0] + want[1] + 8e-6, rel=1e-13)
    assert step[1] == pytest.approx(2e-6 + 4e-6, rel=1e-13)
    assert tot[0] == pytest.approx(step.sum(), rel=1e-14)


def test_batch_matches_single_and_spec_loop():
    w = W.config5(n_rows=3000, n_specs=3, n_layers=2)
    for b in w.buckets:
        out = O.predict_bucket(b, w.specs, W.TIER_NONE)
        assert out["lat"].shape == (3, b.n)
        for sp in (0, 2):
            for i in (0, b.n // 2, b.n - 1):
                d = O.make_desc(b.family, [int(c[i]) for c in b.cols], s=b.dtype_bytes, hq=b.hq, hkv=b.hkv,
                                d=b.head_dim)
                t, r, e = O.predict_one(d, O.make_spec(w.specs[sp]), W.TIER_NONE)
                assert out["lat"][sp, i] == t and out["tiles"][sp, i] == r.B and out["waves"][sp, i] == r.W
