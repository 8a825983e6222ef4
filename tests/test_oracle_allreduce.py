"""Pins for the oracle's tensor-parallel all-reduce term (Eq. 3):
t_ar = alpha0 + 2 (P - 1) / P * S / beta_eff.  Closed forms and special cases only — nothing here
re-types the oracle's own expression for a general (S, P).
"""
import ctypes as C

import numpy as np

from oracle import oracle as O
import workloads as W

SPEC = W.spec_gb200(ar_alpha0=12e-6, ar_beta_eff=900e9)   # NVLink 5 per-direction datasheet bandwidth


def ar(S, P, spec=SPEC):
    return O.lib().kso_allreduce(int(S), int(P), C.byref(O.make_spec(spec)))


def test_single_shard_moves_nothing():
    # the factor 2(P-1)/P is the per-GPU volume of reduce-scatter + all-gather: zero for P = 1
    for S in (0, 1, 8 << 20):
        assert ar(S, 1) == 12e-6


def test_two_shards_send_the_message_once():
    # P = 2: 2 (2 - 1) / 2 = 1  =>  t = alpha0 + S / beta
    S = 9_000_000                      # 9 MB at 900 GB/s = 10 us exactly
    assert abs(ar(S, 2) - (12e-6 + 10e-6)) < 1e-18


def test_hand_computed_case():
    # 64 tokens x 4096 hidden x 2 B = 524,288 B over P = 4: 2*3/4 = 1.5; 1.5 * 524288 / 9e11 = 8.738133...e-7 s
    assert abs(ar(524288, 4) - (12e-6 + 8.738133333333334e-07)) < 1e-18


def test_large_p_limit_and_monotonicity_in_p():
    S = 1 << 24
    vals = [ar(S, P) for P in (2, 3, 4, 8, 64, 4096)]
    assert all(a < b for a, b in zip(vals, vals[1:]))                     # 2(P-1)/P grows with P ...
    assert vals[-1] < 12e-6 + 2 * S / 900e9                               # ... towards, never reaching, 2 S / beta
    assert abs(vals[-1] - (12e-6 + 2 * S / 900e9)) / vals[-1] < 1e-3


def test_affine_in_message_size():
    # for fixed P the bandwidth term is linear in S: second differences vanish, zero message costs alpha0
    t = np.array([ar(S, 8) for S in (0, 1 << 20, 2 << 20, 3 << 20)])
    assert t[0] == 12e-6
    assert abs((t[2] - t[1]) - (t[1] - t[0])) < 1e-18 and abs((t[3] - t[2]) - (t[2] - t[1])) < 1e-18


def test_bandwidth_and_startup_enter_separately():
    base = ar(1 << 22, 4)
    assert abs(ar(1 << 22, 4, W.spec_gb200(ar_alpha0=0.0, ar_beta_eff=900e9)) - (base - 12e-6)) < 1e-18
    half_bw = ar(1 << 22, 4, W.spec_gb200(ar_alpha0=12e-6, ar_beta_eff=450e9))
    assert abs((half_bw - 12e-6) - 2 * (base - 12e-6)) < 1e-18


def test_batch_path_ignores_tier_and_floor_and_enters_the_step_sum():
    # an all-reduce row is Eq. 3 under every tier (no eta, no t0 floor) and is summed like a kernel
    b = W.Bucket(W.FAM_ALLREDUCE, [np.array([524288, 0, 1 << 20], np.int32), np.array([4, 4, 1], np.int32)])
    spec = W.spec_gb200(ar_alpha0=1e-7, ar_beta_eff=900e9, t0=2e-6)
    want = [1e-7 + 8.738133333333334e-07, 1e-7, 1e-7]                     # all below t0: the floor must not apply
    for tier in (W.TIER_NONE, W.TIER_A, W.TIER_B):
        o = O.predict_bucket(b, [spec], tier)
        assert np.allclose(o["lat"][0], want, rtol=1e-15, atol=0)
        assert np.all(o["tiles"] == 0) and np.all(o["waves"] == 0)
    step, _ = O.compose([o["lat"][0]], [np.array([0, 2, 3])], 2, W.STEP_PARAMS_ZERO, np.array([0, 2]))
    assert np.allclose(step, [want[0] + want[1], want[2]], rtol=1e-15)
