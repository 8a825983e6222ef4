"""Pins for the oracle's efficiency models (S3 features, S4a MLP head, S4b grid) and S5 floor.

PAPER.md:191-201 (Eq. 2, heads), :211 (Tier B).  Expected values come from closed forms, special
cases, and independent library routines (numpy matmul + scipy erf, scipy RegularGridInterpolator,
torch bfloat16 casting) — never from the oracle itself.
"""
import math

import numpy as np
import pytest
import torch
from scipy.interpolate import RegularGridInterpolator
from scipy.special import erf, expit

from oracle import oracle as O
import workloads as W

SPECD = W.spec_gb200()
SPEC = O.make_spec(SPECD)


# ------------------------------------------------------------------ bf16 rounding
def test_bf16_matches_torch_rne():
    rng = np.random.default_rng(0)
    x = np.concatenate([rng.normal(0, 1, 5000), rng.normal(0, 1e-3, 2000), rng.uniform(-300, 300, 2000),
                        [0.0, 1.0, -1.0, 1.00390625, 1.01171875, 0.1, 3.0e38, 1e-30]]).astype(np.float32)
    want = torch.from_numpy(x).to(torch.bfloat16).to(torch.float64).numpy()
    got = O.bf16(x.astype(np.float64))
    assert np.array_equal(got, want)
    # ties to even: 1 + 2^-8 is halfway between 1 and 1 + 2^-7 -> 1 ; 1 + 3*2^-8 -> 1 + 2^-6
    assert O.bf16(1.0 + 2.0 ** -8) == 1.0
    assert O.bf16(1.0 + 3 * 2.0 ** -8) == 1.0 + 2.0 ** -6


def test_activation_closed_forms():
    L = O.lib()
    assert L.kso_gelu(0.0) == 0.0
    assert L.kso_sigmoid(0.0) == 0.5
    assert L.kso_gelu(10.0) == pytest.approx(10.0, rel=1e-15)      # GELU(x) -> x
    assert abs(L.kso_gelu(-10.0)) < 1e-20                          # GELU(x) -> 0-
    xs = np.linspace(-6, 6, 241)
    got = np.array([L.kso_gelu(float(v)) for v in xs])
    assert np.allclose(got, 0.5 * xs * (1 + erf(xs / math.sqrt(2))), rtol=1e-14, atol=1e-300)
    # Phi(1) = 0.841344746068543 (standard normal table)
    assert L.kso_gelu(1.0) == pytest.approx(0.841344746068543, rel=1e-14)


# ------------------------------------------------------------------ MLP head
def _numpy_mlp(h, x):
    g = lambda a: 0.5 * a * (1 + erf(a / math.sqrt(2)))
    a1 = g(x @ h.W1 + h.b1)
    a2 = g(a1 @ h.W2 + h.b2)
    return a2 @ h.w3 + h.c.b3


@pytest.mark.parametrize("n_in,hdim", [(8, 64), (12, 128), (32, 256)])
def test_mlp_vs_numpy_matmul(n_in, hdim):
    rng = np.random.Generator(np.random.PCG64(5))
    h = O.Head(W.make_head(rng, n_in, hdim, w_std=0.3))
    for _ in range(20):
        x = rng.uniform(-1, 1, n_in)
        assert O.mlp_z(h, x) == pytest.approx(_numpy_mlp(h, x), rel=1e-12, abs=1e-13)


def test_mlp_zero_weights_gives_half_efficiency():
    # all-zero weights -> z = b3 = 0 -> e = 0.5 -> eta = 2 -> t = max(2 t_roof, t0) exactly
    hd = W.make_head(np.random.default_rng(0), 8, 64, bias_std=0.0, w_std=0.0)
    h = O.Head(hd)
    d = O.make_desc(W.FAM_GEMM, [8192, 8192, 8192])
    t, r, e = O.predict_one(d, SPEC, W.TIER_A, head=h)
    assert e == 0.5 and t == 2.0 * r.t_roof
    tiny = O.make_desc(W.FAM_GEMM, [1, 8, 8])
    t, r, e = O.predict_one(tiny, SPEC, W.TIER_A, head=h)
    assert 2 * r.t_roof < SPECD["t0"] and t == SPECD["t0"]


def test_mlp_one_hidden_unit_by_hand():
    # n_in=8, only unit 0 alive in each layer: z = w3 * g(w2 * g(w1 * x0 + b1) + b2) + b3
    hd = W.make_head(np.random.default_rng(0), 8, 64, bias_std=0.0, w_std=0.0)
    hd.W1[0, 0], hd.b1[0], hd.W2[0, 0], hd.b2[0], hd.w3[0], hd.b3 = 0.5, 0.25, -1.5, 0.125, 2.0, -0.5
    h = O.Head(hd)
    x = np.zeros(8); x[0] = 0.75
    g = lambda a: 0.5 * a * (1 + math.erf(a / math.sqrt(2)))
    want = 2.0 * g(-1.5 * g(0.5 * 0.75 + 0.25) + 0.125) - 0.5
    assert O.mlp_z(h, x) == pytest.approx(want, rel=1e-14)


def test_mlp_transposition_is_detected():
    # W1[i][j]: input i -> hidden j.  A transposed read would mix these up.
    hd = W.make_head(np.random.default_rng(0), 8, 64, bias_std=0.0, w_std=0.0)
    hd.W1[3, 5] = 1.0          # input 3 feeds hidden 5
    hd.W2[5, 7] = 1.0          # hidden 5 feeds hidden 7
    hd.w3[7] = 1.0
    h = O.Head(hd)
    x = np.zeros(8); x[3] = 1.0
    g = lambda a: 0.5 * a * (1 + math.erf(a / math.sqrt(2)))
    assert O.mlp_z(h, x) == pytest.approx(g(g(1.0)), rel=1e-14)
    x = np.zeros(8); x[5] = 1.0
    assert O.mlp_z(h, x) == 0.0


def test_head_weights_are_bf16_rounded_features_too():
    rng = np.random.Generator(np.random.PCG64(7))
    hd = W.make_head(rng, 12, 128)
    h = O.Head(hd)
    want = torch.from_numpy(hd.W2).to(torch.bfloat16).to(torch.float64).numpy()
    assert np.array_equal(h.W2, want)
    # end-to-end Tier A == numpy pipeline on bf16-rounded oracle features
    d = O.make_desc(W.FAM_ATTN, [64, 1, 4096], hq=32, hkv=8, d=128)
    t, r, e = O.predict_one(d, SPEC, W.TIER_A, head=h)
    x = O.features(d, SPEC, 12)
    xb = torch.from_numpy(x.astype(np.float32)).to(torch.bfloat16).to(torch.float64).numpy()
    z = _numpy_mlp(h, xb)
    assert e == pytest.approx(float(expit(z)), rel=1e-12)
    assert t == pytest.approx(max(r.t_roof / float(expit(z)), SPECD["t0"]), rel=1e-12)


# ------------------------------------------------------------------ features (Q2)
def test_features_closed_forms():
    d = O.make_desc(W.FAM_GEMM, [8192, 8192, 8192])
    r = O.roofline(d, SPEC)
    x = O.features(d, SPEC, 12)
    AI = 1099511627776 / 402653184                       # golden F / Y
    assert x[0] == pytest.approx(math.log2(AI) / 16, rel=1e-14)
    assert x[1] == pytest.approx(math.log2(AI / 281.25) / 16, rel=1e-13)   # ridge = 2.25e15/8e12
    assert x[2] == pytest.approx(math.log2(28) / 16, rel=1e-14)
    assert x[3] == pytest.approx(1 / 1.01171875, rel=1e-14)               # occupancy = 1/u
    assert x[4] == pytest.approx(math.log2(4.943984576284444e-04 / 2e-6) / 16, rel=1e-12)
    assert x[5] == pytest.approx(126e6 / 402653184, rel=1e-14)
    assert x[6] == pytest.approx(math.log2(4.943984576284444e-04 / 5.0331648e-05) / 20, rel=1e-12)
    assert x[7] == pytest.approx(math.log2(4096 / 148) / 16, rel=1e-14)
    assert list(x[8:11]) == [13 / 16] * 3 and x[11] == 0.5
    assert np.all(np.abs(x) <= 1.0)
    # first 8 are shared between feature-set sizes; 32-wide pads with zeros for non-grouped
    assert np.array_equal(O.features(d, SPEC, 8), x[:8])
    x32 = O.features(d, SPEC, 32)
    assert np.array_equal(x32[:12], x) and not x32[12:].any()


def test_features_ridge_is_zero_and_small_kernel_resident():
    d = O.make_desc(W.FAM_GEMM, [148 * 128, 128, 4096])   # u = 1
    r0 = O.roofline(d, SPEC)
    spec = O.make_spec(W.spec_gb200(peak_bw=1e12, peak_flops=1e12 * r0.F / r0.Y))
    x = O.features(d, spec, 8)
    assert abs(x[1]) < 1e-15 and abs(x[6]) < 1e-15        # on the ridge
    assert x[3] == 1.0 and x[2] == 0.0                    # one full wave
    small = O.make_desc(W.FAM_ELEMWISE, [4096, W.SUB_RMSNORM])
    xs = O.features(small, SPEC, 12)
    assert xs[5] == 1.0                                   # fits L2
    assert xs[9] == 2 / 4 and xs[10] == 4 / 8 and xs[8] == 12 / 32


def test_features_grouped_and_degenerate():
    m = [10, 0, 30, 0, 0, 0, 0, 40]
    d = O.make_desc(W.FAM_GROUPED, [4096, 1024] + m)
    x = O.features(d, SPEC, 32)
    assert np.allclose(x[12:20], np.array(m) / 80.0, rtol=1e-15)
    assert x[20] == pytest.approx(40 / 80, rel=1e-15)     # (max/mean)/8 with 8 experts = max/sum
    assert x[21] == 3 / 8
    assert not x[22:].any()
    assert x[8] == pytest.approx(math.log2(80) / 16)
    z = O.features(O.make_desc(W.FAM_GROUPED, [4096, 1024] + [0] * 8), SPEC, 32)
    assert not z.any()                                    # B = 0 -> all-zero features


# ------------------------------------------------------------------ Tier-B grid
def _grid(values, lo=(0, 0, 0), hi=(13, 14, 15)):
    v = np.asarray(values, np.float32)
    return W.Grid(np.asarray(v.shape, np.int32), np.asarray(lo, np.float32), np.asarray(hi, np.float32), v)


def test_trilinear_nodes_exact():
    rng = np.random.default_rng(1)
    gd = _grid(rng.uniform(0.2, 0.95, (32, 32, 32)), lo=(0, 0, 0), hi=(31, 31, 31))
    g = O.Grid(gd)
    for _ in range(200):
        i, j, k = (int(v) for v in rng.integers(0, 32, 3))
        assert O.trilinear(g, [2.0 ** i, 2.0 ** j, 2.0 ** k]) == float(gd.values[i, j, k])


def test_trilinear_reproduces_multilinear_function_and_scipy():
    rng = np.random.default_rng(2)
    lo, hi = np.array([0.0, 10.0, 10.0]), np.array([13.0, 14.0, 14.0])
    ax = [np.linspace(lo[a], hi[a], 32) for a in range(3)]
    A, B, Cc = np.meshgrid(*ax, indexing="ij")
    lin = 0.3 + 0.01 * A - 0.02 * B + 0.03 * Cc
    g_lin = O.Grid(_grid(lin.astype(np.float64), lo, hi))
    g_lin.values[...] = lin                    # keep the function's full double precision
    rnd = rng.uniform(0.2, 0.95, (32, 32, 32)).astype(np.float32)
    g_rnd = O.Grid(_grid(rnd, lo, hi))
    rgi = RegularGridInterpolator(ax, rnd.astype(np.float64), method="linear")
    for _ in range(300):
        x = rng.uniform(lo, hi)
        v = 2.0 ** x
        assert O.trilinear(g_lin, v) == pytest.approx(0.3 + 0.01 * x[0] - 0.02 * x[1] + 0.03 * x[2], rel=1e-12)
        got = O.trilinear(g_rnd, v)
        assert got == pytest.approx(float(rgi(x[None, :])[0]), rel=1e-11)
        i = [min(int(np.floor((x[a] - lo[a]) / (hi[a] - lo[a]) * 31)), 30) for a in range(3)]
        corners = rnd[i[0]:i[0] + 2, i[1]:i[1] + 2, i[2]:i[2] + 2]
        assert corners.min() - 1e-12 <= got <= corners.max() + 1e-12


def test_trilinear_clamp_constant_and_flat_axes():
    rng = np.random.default_rng(3)
    lo, hi = (0.0, 10.0, 10.0), (13.0, 14.0, 14.0)
    rnd = rng.uniform(0.2, 0.95, (32, 32, 32)).astype(np.float32)
    g = O.Grid(_grid(rnd, lo, hi))
    inside = [2.0 ** 5.3, 2.0 ** 12.1, 2.0 ** 13.7]
    for a in range(3):
        below, above = list(inside), list(inside)
        below[a], above[a] = 2.0 ** (lo[a] - 1.7), 2.0 ** (hi[a] + 1.2)
        at_lo, at_hi = list(inside), list(inside)
        at_lo[a], at_hi[a] = 2.0 ** lo[a], 2.0 ** hi[a]
        assert O.trilinear(g, below) == pytest.approx(O.trilinear(g, at_lo), rel=1e-14)
        assert O.trilinear(g, above) == pytest.approx(O.trilinear(g, at_hi), rel=1e-14)
    const = O.Grid(_grid(np.full((32, 32, 32), 0.625, np.float32), lo, hi))
    assert O.trilinear(const, inside) == pytest.approx(0.625, rel=1e-15)
    # elementwise family: axis 1 is the sub-op node (6 nodes), axis 2 is flat (1 node)
    ev = rng.uniform(0.2, 0.95, (32, 6, 1)).astype(np.float32)
    ge = O.Grid(_grid(ev, (12, 0, 0), (25, 5, 0)))
    d = O.make_desc(W.FAM_ELEMWISE, [2 ** 20, 4])
    t, r, e = O.predict_one(d, SPEC, W.TIER_B, grid=ge)
    c = (20 - 12) / 13 * 31
    i = int(np.floor(c)); f = c - i
    assert e == pytest.approx(float(ev[i, 4, 0]) * (1 - f) + float(ev[i + 1, 4, 0]) * f, rel=1e-13)


def test_tier_b_latency_and_axes():
    rng = np.random.default_rng(4)
    gd = W.make_grid(rng, *W.ATTN_SPAN)
    g = O.Grid(gd)
    d = O.make_desc(W.FAM_ATTN, [64, 1, 4096], hq=32, hkv=8, d=128)    # log2 = (6, 0, 12)
    t, r, e = O.predict_one(d, SPEC, W.TIER_B, grid=g)
    ax = [np.linspace(W.ATTN_SPAN[0][a], W.ATTN_SPAN[1][a], 32) for a in range(3)]
    want_e = float(RegularGridInterpolator(ax, gd.values.astype(np.float64))([[6.0, 0.0, 12.0]])[0])
    assert e == pytest.approx(want_e, rel=1e-12)
    assert t == pytest.approx(1.343488e-04 / want_e, rel=1e-12)          # golden t_roof / e
    assert t >= r.t_roof                                                 # eta >= 1 since e <= 1


def test_grouped_gemm_grid_axes_are_total_tokens_then_n_then_k():
    # DESIGN.md Q5: a grouped GEMM's grid coordinates are (sum_e m_e, N, K).  A 5 x 3 x 2 grid whose node (i, j, k)
    # holds 0.1 + 0.1 i + 0.02 j + 0.3 k, with a different span on every axis: sum m over 2^4..2^8, N over 2^10..2^12,
    # K over 2^6..2^7.  Queries on nodes name their value; swapping N and K, or taking one expert's tokens for the
    # total, lands on another node (or off the grid) and fails.
    val = np.array([[[0.1 + 0.1 * i + 0.02 * j + 0.3 * k for k in range(2)] for j in range(3)] for i in range(5)])
    g = O.Grid(_grid(val, lo=(4, 10, 6), hi=(8, 12, 7)))
    for i in range(5):
        for j in range(3):
            for k in range(2):
                tot = 2 ** (4 + i)
                m = [tot // 2, 0, tot // 4, 0, 0, tot // 8, 0, tot // 8]           # eight experts, three idle
                assert sum(m) == tot
                d = O.make_desc(W.FAM_GROUPED, [2 ** (10 + j), 2 ** (6 + k)] + m)
                _, _, e = O.predict_one(d, SPEC, W.TIER_B, grid=g)
                assert e == pytest.approx(float(np.float32(val[i, j, k])), rel=1e-12)
    # between nodes, by hand: sum m = 48 -> coordinate log2(48) - 4 = 1.58496 on axis 0 (cell 1, f = 0.58496);
    # N = 2^11 (node 1), K = 2^6 (node 0): e = v[1,1,0] + f (v[2,1,0] - v[1,1,0]) = 0.22 + 0.058496
    d = O.make_desc(W.FAM_GROUPED, [2048, 64, 40, 8, 0, 0, 0, 0, 0, 0])
    _, _, e = O.predict_one(d, SPEC, W.TIER_B, grid=g)
    f = math.log2(48) - 5
    assert e == pytest.approx(float(np.float32(val[1, 1, 0])) * (1 - f) + float(np.float32(val[2, 1, 0])) * f, rel=1e-12)
    # negative token counts are ignored by the total (like everywhere else in the family)
    d = O.make_desc(W.FAM_GROUPED, [2048, 64, 40, 8, -7, 0, 0, 0, 0, 0])
    assert O.predict_one(d, SPEC, W.TIER_B, grid=g)[2] == pytest.approx(e, rel=1e-15)


# ------------------------------------------------------------------ floor
def test_floor_applied_after_eta():
    d = O.make_desc(W.FAM_ELEMWISE, [4096, W.SUB_RMSNORM])
    t, r, e = O.predict_one(d, SPEC, W.TIER_NONE)
    assert r.t_roof < 1e-8 and t == SPECD["t0"]
    nofloor = O.make_spec(W.spec_gb200(t0=1e-30))
    big = O.make_desc(W.FAM_GEMM, [8192, 8192, 8192])
    t, r, e = O.predict_one(big, nofloor, W.TIER_NONE)
    assert e == 1.0 and t == r.t_roof                                    # eta = 1 attains the bound
    # the floor is never scaled by eta: tiny kernel, e = 0.5 head -> still exactly t0
    hd = W.make_head(np.random.default_rng(0), 8, 64, bias_std=0.0, w_std=0.0)
    t, r, e = O.predict_one(d, SPEC, W.TIER_A, head=O.Head(hd))
    assert t == SPECD["t0"]
