"""Pins for the oracle's bounded analytical head (PAPER.md:197 Fig. 6, :201):
utilisation e = gamma(x) - alpha(x)/W, eta = 1/e, with gamma = sigmoid(w_gamma.x + b_gamma),
alpha = max(0, w_alpha.x + b_alpha) (Q15).  Closed forms and special cases.
"""
import numpy as np
import pytest
from scipy.special import expit

from oracle import oracle as O
import workloads as W

SPEC = W.spec_gb200()


def head(n_in=8, wg=0.0, bg=0.0, wa=0.0, ba=0.0):
    f = lambda v: np.full(n_in, v, np.float32) if np.isscalar(v) else np.asarray(v, np.float32)
    return O.Bounded(W.BoundedHead(n_in, f(wg), bg, f(wa), ba))


def test_constant_maps_give_fig6_curve():
    # with feature-independent maps the head is exactly Fig. 6's curve: e(W) = gamma - alpha / W
    # gamma = sigmoid(ln 4) = 0.8, alpha = 0.3 (both held in fp32 like the library does: 1e-7 slack)
    bh = head(bg=float(np.log(0.8 / 0.2)), ba=0.3)
    x = np.zeros(8)
    for Wv, want in [(1, 0.5), (2, 0.65), (3, 0.7), (10, 0.77), (300, 0.799)]:
        assert abs(O.bounded_e(bh, x, Wv) - want) < 1e-7
    es = [O.bounded_e(bh, x, Wv) for Wv in (1, 2, 4, 8, 64, 4096, 10 ** 9)]
    assert all(a < b for a, b in zip(es, es[1:]))             # efficiency climbs with the wave count ...
    gamma = O.bounded_e(bh, x, 0)                             # W = 0: no partial-wave term at all
    assert es[-1] < gamma and gamma - es[-1] < 1e-9 and abs(gamma - 0.8) < 1e-7               # ... towards the peak gamma


def test_no_partial_wave_overhead_means_gamma():
    bh = head(bg=0.0, ba=-5.0)                                # alpha = max(0, -5) = 0; gamma = sigmoid(0) = 1/2
    for Wv in (0, 1, 7, 10 ** 6):
        assert O.bounded_e(bh, np.zeros(8), Wv) == 0.5


def test_bounds_and_guard():
    assert O.bounded_e(head(bg=50.0, ba=0.0), np.zeros(8), 5) == 1.0                 # e <= 1  (eta >= 1)
    assert O.bounded_e(head(bg=0.0, ba=10.0), np.zeros(8), 1) == 2.0 ** -10          # guard at 2^-10 (Q3)
    assert abs(O.bounded_e(head(bg=0.0, ba=10.0), np.zeros(8), 40) - 0.25) < 1e-15   # 0.5 - 10/40


def test_linear_maps_against_numpy():
    rng = np.random.Generator(np.random.PCG64(7))
    for n_in in (8, 12, 32):
        h = W.make_bounded_head(rng, n_in)
        bh = O.Bounded(h)
        for _ in range(20):
            x = rng.uniform(-1, 1, n_in)
            Wv = int(rng.integers(1, 50))
            g = expit(np.dot(h.w_gamma.astype(np.float64), x) + np.float64(np.float32(h.b_gamma)))
            a = max(0.0, np.dot(h.w_alpha.astype(np.float64), x) + np.float64(np.float32(h.b_alpha)))
            want = min(max(g - a / Wv, 2.0 ** -10), 1.0)
            assert abs(O.bounded_e(bh, x, Wv) - want) < 1e-13


def test_prediction_uses_the_wave_count_of_the_kernel_and_the_floor():
    # GEMM 8192^3 on config 1's spec: B = 4096 tiles, W = 28 waves, t_roof = 4.943985e-4 s (golden case 1)
    b = W.Bucket(W.FAM_GEMM, [np.array([8192], np.int32)] * 3)
    bh = head(bg=float(np.log(0.8 / 0.2)), ba=0.3)
    o = O.predict_bucket(b, [SPEC], W.TIER_A, bounded=bh)
    e = 0.8 - 0.3 / 28
    assert o["waves"][0, 0] == 28
    assert abs(o["lat"][0, 0] - o["troof"][0, 0] / e) / o["lat"][0, 0] < 1e-7
    assert abs(o["troof"][0, 0] - 4.943985e-4) / 4.943985e-4 < 1e-6
    # tiny kernel: the launch floor wins and is not scaled by eta
    tiny = W.Bucket(W.FAM_ELEMWISE, [np.array([4096], np.int32), np.array([0], np.int32)])
    assert O.predict_bucket(tiny, [SPEC], W.TIER_A, bounded=bh)["lat"][0, 0] == SPEC["t0"]
    # a perfect head (gamma -> 1, alpha = 0) attains the bound: t = t_roof
    o1 = O.predict_bucket(b, [SPEC], W.TIER_A, bounded=head(bg=60.0, ba=-1.0))
    assert o1["lat"][0, 0] == o1["troof"][0, 0]


def test_features_enter_through_the_dot_products():
    # gamma must move with the features: raising w_gamma on feature 3 (occupancy B/(W S) = 1/u in (0,1]) raises e
    b = W.Bucket(W.FAM_GEMM, [np.array([576], np.int32), np.array([6144], np.int32), np.array([4096], np.int32)])
    wg = np.zeros(8, np.float32)
    lo = O.predict_bucket(b, [SPEC], W.TIER_A, bounded=head(wg=wg, ba=-1.0))["lat"][0, 0]
    wg[3] = 2.0
    hi = O.predict_bucket(b, [SPEC], W.TIER_A, bounded=head(wg=wg, ba=-1.0))["lat"][0, 0]
    x = O.features(O.make_desc(W.FAM_GEMM, [576, 6144, 4096]), O.make_spec(SPEC), 8)
    assert abs(x[3] - 240 / (2 * 148)) < 1e-12                # golden "mixed shape": B = 240, W = 2, S = 148
    assert abs(hi / lo - 0.5 / expit(2.0 * x[3])) < 1e-12     # e: 1/2 -> sigmoid(2 x3)
