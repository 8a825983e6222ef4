"""Pins for the oracle's S1/S2 (work, wave quantization, Eq. 2) — PAPER.md:88, :191-193, :249.

Every expected value is the paper's (Fig. 2), a hand-computed constant (tests/golden), a brute-force
count, or an invariant — never the oracle's own formula retyped.
"""
import itertools
import os

import numpy as np
import pytest

from oracle import oracle as O
import workloads as W

SPEC = O.make_spec(W.spec_gb200())
GOLD = os.path.join(os.path.dirname(__file__), "golden", "roofline_cases.txt")


def test_fig2_worked_example():
    # 9 blocks on 4 SMs span 3 waves; u = ceil(9/4)*4/9
    Wv, u = O.wave(9, 4)
    assert Wv == 3
    assert u == pytest.approx(4.0 / 3.0, rel=1e-15)


def _simulate_waves(B, S):
    """Round-robin block placement: brute-force wave count and time inflation."""
    slots = [0] * S
    for b in range(B):
        slots[b % S] += 1
    waves = max(slots)
    return waves, waves * S / B


@pytest.mark.parametrize("S", [1, 2, 3, 4, 7, 16, 64])
def test_wave_bruteforce(S):
    for B in range(1, 65):
        Wv, u = O.wave(B, S)
        wb, ub = _simulate_waves(B, S)
        assert Wv == wb
        assert u == pytest.approx(ub, rel=1e-15)
        assert u >= 1.0
        assert (u == 1.0) == (B % S == 0)          # partial only if S does not divide B


def test_wave_tiny_grids_and_degenerate():
    S = 148
    assert O.wave(S, S) == (1, 1.0)
    Wv, u = O.wave(S + 1, S)
    assert Wv == 2 and u == pytest.approx(2 * S / (S + 1))
    Wv, u = O.wave(1, S)
    assert Wv == 1 and u == pytest.approx(S)
    assert O.wave(0, S) == (0, 1.0)                 # DESIGN.md Q4


def _golden():
    fam = {"gemm": W.FAM_GEMM, "attn": W.FAM_ATTN, "elem": W.FAM_ELEMWISE}
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        lhs, rhs = line.split("|")
        f, a, b, c = lhs.split()
        yield fam[f], [int(a), int(b), int(c)], rhs.split()


@pytest.mark.parametrize("family,v,exp", list(_golden()))
def test_golden_roofline(family, v, exp):
    F, Y, B, Wv, u, troof = exp
    if family == W.FAM_ELEMWISE:
        d = O.make_desc(family, v[:2])
    else:
        d = O.make_desc(family, v, hq=32, hkv=8, d=128)
    r = O.roofline(d, SPEC)
    assert r.F == float(F) and r.Y == float(Y)
    assert r.B == int(B) and r.W == int(Wv)
    assert r.u == pytest.approx(float(u), rel=1e-15)
    assert r.t_roof == pytest.approx(float(troof), rel=1e-13)


def test_attn_pairs_bruteforce():
    # chunk query i (0-based) sees keys j <= hist + i
    for q, kv in itertools.product(range(0, 13), range(0, 20)):
        if kv < q:
            continue
        hist = kv - q
        brute = sum(1 for i in range(q) for j in range(kv) if j <= hist + i)
        assert O.lib().kso_attn_pairs(q, kv) == brute
    assert O.lib().kso_attn_pairs(1, 4096) == 4096          # decode: pairs = kv
    assert O.lib().kso_attn_pairs(7, 7) == 7 * 8 // 2        # no history: causal triangle


def test_gemm_bruteforce_flops_bytes_tiles():
    spec = O.make_spec(W.spec_gb200(tile_m=4, tile_n=8))
    for M, N, K in [(1, 1, 1), (3, 5, 7), (4, 8, 2), (9, 17, 3), (5, 16, 4)]:
        macs = sum(1 for _ in itertools.product(range(M), range(N), range(K)))
        tiles = len({(i // 4, j // 8) for i in range(M) for j in range(N)})
        elems = M * K + K * N + M * N
        r = O.roofline(O.make_desc(W.FAM_GEMM, [M, N, K], s=2), spec)
        assert r.F == 2 * macs and r.Y == 2 * elems and r.B == tiles


def test_grouped_reduces_to_gemm_and_skips_empty_experts():
    # one active expert with m tokens == a plain GEMM(m, N, K)
    g = O.roofline(O.make_desc(W.FAM_GROUPED, [4096, 1024, 300, 0, 0, 0, 0, 0, 0, 0]), SPEC)
    p = O.roofline(O.make_desc(W.FAM_GEMM, [300, 4096, 1024]), SPEC)
    assert (g.F, g.Y, g.B) == (p.F, p.Y, p.B)
    # two experts: tiles add per expert (ceil per expert), weights read once per ACTIVE expert
    g2 = O.roofline(O.make_desc(W.FAM_GROUPED, [256, 64, 1, 129, 0, 0, 0, 0, 0, 0]), SPEC)
    assert g2.B == (1 + 2) * 2
    assert g2.F == 2 * 256 * 64 * 130
    assert g2.Y == 2 * (64 * 130 + 2 * 64 * 256 + 256 * 130)
    z = O.roofline(O.make_desc(W.FAM_GROUPED, [256, 64] + [0] * 8), SPEC)
    assert (z.F, z.Y, z.B, z.W, z.u, z.t_roof) == (0, 0, 0, 0, 1.0, 0.0)


def test_ridge_and_bound_regimes():
    # at AI == P/BW the two ceilings meet.  Pick F, Y with F/Y = ridge via a spec.
    d = O.make_desc(W.FAM_GEMM, [148 * 128, 128, 4096])          # B = 148 -> u = 1
    r0 = O.roofline(d, SPEC)
    assert r0.u == 1.0
    spec = O.make_spec(W.spec_gb200(peak_bw=1e12, peak_flops=1e12 * r0.F / r0.Y))
    r = O.roofline(d, spec)
    assert r.t_comp == pytest.approx(r.t_mem, rel=1e-14)
    lo = O.roofline(d, O.make_spec(W.spec_gb200(peak_bw=1e12, peak_flops=2e12 * r0.F / r0.Y)))
    assert lo.t_roof == lo.t_mem                                   # above-ridge machine: memory-bound
    hi = O.roofline(d, O.make_spec(W.spec_gb200(peak_bw=1e12, peak_flops=0.5e12 * r0.F / r0.Y)))
    assert hi.t_roof == hi.t_comp * hi.u                           # compute-bound


def test_troof_monotone_in_each_dim():
    rng = np.random.default_rng(0)
    for _ in range(200):
        M, N, K = (int(x) for x in rng.integers(1, 5000, 3))
        base = O.roofline(O.make_desc(W.FAM_GEMM, [M, N, K]), SPEC)
        # wave quantization makes t_roof non-monotone in M,N (that is the point of u), but
        # F, Y, B are monotone, and t_roof is monotone in K (B unchanged).
        up = O.roofline(O.make_desc(W.FAM_GEMM, [M, N, K + 1]), SPEC)
        assert up.t_roof >= base.t_roof and up.B == base.B
        for v in ([M + 1, N, K], [M, N + 1, K]):
            r = O.roofline(O.make_desc(W.FAM_GEMM, v), SPEC)
            assert r.F > base.F and r.Y > base.Y and r.B >= base.B


def test_elementwise_table_and_ctas():
    # RMSNorm 2 words/elem; SiLU*Mul 3 (two reads, one write); KV-write 2 words, 0 FLOPs
    n = 10000
    rm = O.roofline(O.make_desc(W.FAM_ELEMWISE, [n, W.SUB_RMSNORM]), SPEC)
    sm = O.roofline(O.make_desc(W.FAM_ELEMWISE, [n, W.SUB_SILU_MUL]), SPEC)
    kw = O.roofline(O.make_desc(W.FAM_ELEMWISE, [n, W.SUB_KV_WRITE]), SPEC)
    assert rm.Y == 2 * 2 * n and sm.Y == 2 * 3 * n and kw.Y == 2 * 2 * n and kw.F == 0
    assert rm.B == 3                                               # ceil(10000/4096)
    assert kw.t_roof == kw.t_mem


def test_ctas_per_sm_generalisation():
    # DESIGN.md Q4: S = N_SM * c; c = 1 reduces to the paper's u
    d = O.make_desc(W.FAM_GEMM, [128 * 200, 128, 512])             # B = 200
    r1 = O.roofline(d, O.make_spec(W.spec_gb200(ctas_per_sm=1)))
    r2 = O.roofline(d, O.make_spec(W.spec_gb200(ctas_per_sm=2)))
    assert (r1.W, r2.W) == (2, 1)
    assert r1.u == pytest.approx(296 / 200) and r2.u == pytest.approx(296 / 200)
