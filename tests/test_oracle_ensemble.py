"""Pins for the oracle's MLP-ensemble head ("small MLP ensemble"; SURVEY.md §8(f) NEXT-2;
DESIGN.md Q17): k members of one shape, efficiency e = (1/k) sum_m sigmoid(z_m(x)), then the guard and
eta = 1/e.  Closed forms, reductions to the single head, and numpy/scipy written out independently.
"""
import numpy as np
from scipy.special import erf, expit

from oracle import oracle as O
import workloads as W

SPEC = W.spec_gb200()


def const_member(n_in, h, b3):
    z = np.zeros
    return W.Head(n_in, h, h, z((n_in, h), np.float32), z(h, np.float32), z((h, h), np.float32), z(h, np.float32),
                  z(h, np.float32), float(b3))


def test_mean_is_taken_over_efficiencies_not_logits_or_etas():
    # members with constant outputs 0.8 and 0.5: mean e = 0.65
    # (sigmoid of the mean logit would give 2/3, the mean of the etas 1/1.625 = 0.615)
    ens = O.Ensemble([const_member(8, 16, np.log(4.0)), const_member(8, 16, 0.0)])
    e = O.ensemble_e(ens, np.zeros(8))
    assert abs(e - 0.65) < 1e-7
    ens3 = O.Ensemble([const_member(8, 16, np.log(4.0)), const_member(8, 16, 0.0), const_member(8, 16, np.log(1 / 3))])
    assert abs(O.ensemble_e(ens3, np.ones(8)) - (0.8 + 0.5 + 0.25) / 3) < 1e-7


def test_one_member_and_identical_members_reduce_to_the_single_head():
    rng = np.random.Generator(np.random.PCG64(11))
    w = W.config2(n=600, seed=21)
    for b in w.buckets:
        h = W.make_head(rng, 12, 32)
        single = O.predict_bucket(b, w.specs, 1, head=O.Head(h))["lat"]
        one = O.predict_bucket(b, w.specs, 1, ensemble=O.Ensemble([h]))["lat"]
        four = O.predict_bucket(b, w.specs, 1, ensemble=O.Ensemble([h, h, h, h]))["lat"]
        assert np.array_equal(single, one)
        assert np.allclose(single, four, rtol=1e-15, atol=0)


def test_member_order_does_not_matter_and_mean_lies_between_members():
    rng = np.random.Generator(np.random.PCG64(12))
    ms = W.make_ensemble(rng, 12, 32, 4, w_std=0.4)
    for _ in range(10):
        x = rng.uniform(-1, 1, 12)
        e = O.ensemble_e(O.Ensemble(ms), x)
        assert abs(e - O.ensemble_e(O.Ensemble(ms[::-1]), x)) < 1e-15
        each = [O.ensemble_e(O.Ensemble([m]), x) for m in ms]
        assert min(each) <= e <= max(each) and max(each) - min(each) > 1e-4
        assert abs(e - float(np.mean(each))) < 1e-15


def test_against_numpy_written_out():
    rng = np.random.Generator(np.random.PCG64(13))
    gelu = lambda a: 0.5 * a * (1.0 + erf(a / np.sqrt(2.0)))
    for n_in, h, k in ((8, 16, 2), (12, 32, 4), (32, 64, 2), (12, 16, 8)):
        ms = W.make_ensemble(rng, n_in, h, k, w_std=0.3)
        ens = O.Ensemble(ms, round_weights=False)
        for _ in range(5):
            x = rng.uniform(-1, 1, n_in)
            es = []
            for m in ms:
                a1 = gelu(x @ m.W1.astype(np.float64) + m.b1)
                a2 = gelu(a1 @ m.W2.astype(np.float64) + m.b2)
                es.append(expit(a2 @ m.w3.astype(np.float64) + np.float64(np.float32(m.b3))))
            assert abs(O.ensemble_e(ens, x) - np.mean(es)) < 1e-13


def test_prediction_applies_guard_and_floor_after_the_mean():
    # GEMM 8192^3 on config 1's spec: t_roof = 4.943985e-4 s (golden case 1)
    b = W.Bucket(W.FAM_GEMM, [np.array([8192], np.int32)] * 3)
    ens = O.Ensemble([const_member(8, 16, np.log(4.0)), const_member(8, 16, 0.0)])
    out = O.predict_bucket(b, [SPEC], 1, ensemble=ens)
    assert abs(out["lat"][0, 0] - out["troof"][0, 0] / 0.65) < 1e-9 * out["lat"][0, 0]
    assert abs(out["troof"][0, 0] - 4.943985e-4) < 1e-9
    # both members at e ~ 0: the guard 2^-10 bounds eta (Q3)
    lo = O.Ensemble([const_member(8, 16, -60.0), const_member(8, 16, -60.0)])
    assert abs(O.predict_bucket(b, [SPEC], 1, ensemble=lo)["lat"][0, 0] - out["troof"][0, 0] * 1024.0) < 1e-12
    # a kernel far below the launch floor stays at t0 whatever the ensemble says (floor after eta)
    tiny = W.Bucket(W.FAM_GEMM, [np.array([16], np.int32)] * 3)
    assert O.predict_bucket(tiny, [SPEC], 1, ensemble=ens)["lat"][0, 0] == SPEC["t0"]
