"""Pins for the oracle's log-eta head output (PAPER.md:193 "eta >= 1", :199 heads "trained against log eta";
DESIGN.md Q21): eta = exp(max(z, 0)), e = 1 / eta, then the same guard and floor as every other head."""
import numpy as np

from oracle import oracle as O
import workloads as W

SPEC = W.spec_gb200()


def const_head(b3, n_in=8, h=64, out_mode=W.HEAD_LOG_ETA):
    z = lambda *s: np.zeros(s, np.float32)
    return O.Head(W.Head(n_in, h, h, z(n_in, h), z(h), z(h, h), z(h), z(h), float(b3), out_mode))


def test_eta_from_log_closed_forms():
    assert O.eta_from_log(0.0) == 1.0
    assert O.eta_from_log(-3.0) == 1.0 and O.eta_from_log(-1e300) == 1.0     # the roofline is a lower bound
    assert abs(O.eta_from_log(np.log(2.0)) - 2.0) < 1e-15
    assert abs(O.eta_from_log(1.0) - np.e) < 1e-15
    zs = np.linspace(-2, 5, 50)
    es = [O.eta_from_log(z) for z in zs]
    assert all(b >= a for a, b in zip(es, es[1:])) and min(es) == 1.0           # monotone, never below 1
    # inverse of what the head is trained on: log eta_from_log(z) = z for z >= 0
    assert all(abs(np.log(O.eta_from_log(z)) - z) < 1e-14 for z in zs if z >= 0)


def test_zero_weight_head_is_the_constant_multiplier():
    # all-zero weights: z = b3.  b3 = ln 2 doubles the roofline time; b3 <= 0 attains the bound; the floor t0 is not scaled
    b = W.Bucket(W.FAM_GEMM, W._i32([8192, 1], [8192, 8], [8192, 8]))
    troof = O.predict_bucket(b, [SPEC], W.TIER_NONE)["troof"][0]
    two = O.predict_bucket(b, [SPEC], W.TIER_A, head=const_head(np.log(2.0)))["lat"][0]
    assert abs(two[0] / troof[0] - 2.0) < 1e-12                                   # t = 2 t_roof
    assert two[1] == SPEC["t0"]                                                    # a tiny kernel: floor after eta
    for b3 in (0.0, -0.7, -50.0):
        one = O.predict_bucket(b, [SPEC], W.TIER_A, head=const_head(b3))["lat"][0]
        assert one[0] == troof[0] and one[1] == SPEC["t0"]                         # eta = 1 attains the bound
    # the same weights read as a utilisation: e = sigmoid(ln 2) = 2/3, eta = 1.5 — a different convention
    util = O.predict_bucket(b, [SPEC], W.TIER_A, head=const_head(np.log(2.0), out_mode=W.HEAD_UTILISATION))["lat"][0]
    assert abs(util[0] / troof[0] - 1.5) < 1e-12


def test_guard_caps_eta_at_2_pow_10():
    b = W.Bucket(W.FAM_GEMM, W._i32([8192], [8192], [8192]))
    troof = O.predict_bucket(b, [SPEC], W.TIER_NONE)["troof"][0]
    big = O.predict_bucket(b, [SPEC], W.TIER_A, head=const_head(20.0))["lat"][0]   # exp(20) >> 2^10
    assert abs(big[0] / troof[0] - 1024.0) < 1e-9                                   # guard e >= 2^-10 (Q3) applies here too


def test_head_e_against_numpy_and_scipy():
    from scipy.special import erf
    rng = np.random.Generator(np.random.PCG64(21))
    for n_in, h in ((8, 64), (12, 128)):
        hd = W.make_head(rng, n_in, h, bias_std=0.3)
        hd.out_mode = W.HEAD_LOG_ETA
        oh = O.Head(hd)
        gelu = lambda v: 0.5 * v * (1.0 + erf(v / np.sqrt(2.0)))
        for _ in range(20):
            x = O.bf16(rng.uniform(-1, 1, n_in))
            z = float(gelu(gelu(x @ oh.W1 + oh.b1) @ oh.W2 + oh.b2) @ oh.w3 + float(hd.b3))
            want = 1.0 / np.exp(max(z, 0.0))
            assert abs(O.head_e(oh, x) - want) < 1e-13
