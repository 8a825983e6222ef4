"""The seeded generators: shapes, determinism, and the structure DESIGN.md §4 promises."""
import numpy as np

import workloads as W


def test_deterministic_and_sized():
    a, b = W.config2(n=5000), W.config2(n=5000)
    for x, y in zip(a.buckets, b.buckets):
        assert all(np.array_equal(p, q) for p, q in zip(x.cols, y.cols))
    assert [bk.n for bk in a.buckets] == [2500, 1500, 1000]
    assert np.array_equal(a.heads[W.FAM_ATTN].W2, b.heads[W.FAM_ATTN].W2)


def test_cfg1_fp32_exact_ints():
    w = W.config1()
    M, N, K = w.buckets[0].cols
    assert M.dtype == np.float32 and w.buckets[0].n == 4096
    assert np.all(M == np.rint(M)) and M.max() <= 8192 and set(np.unique(N)) <= set(W.GEMM_NK.astype(np.float32))
    h = w.heads[W.FAM_GEMM]
    assert (h.n_in, h.h1, h.h2) == (8, 64, 64) and not h.b1.any() and h.b3 == 0.0


def test_cfg2_attention_ranges():
    w = W.config2(n=20000)
    B_, q, kv = w.buckets[1].cols
    assert B_.min() >= 1 and B_.max() <= 256 and np.all(kv >= q) and kv.max() <= 32768
    assert np.all((q == 1) | ((q >= 128) & (q <= 8192)))
    ne, sub = w.buckets[2].cols
    assert ne.min() >= 4096 and ne.max() <= 32 * 2 ** 20 and set(np.unique(sub)) <= set(range(6))


def test_cfg3_grids_and_oob_fraction():
    w = W.config3(n=40000)
    g = w.grids[W.FAM_GEMM]
    assert g.values.shape == (32, 32, 32) and g.values.dtype == np.float32
    assert 0.2 <= g.values.min() and g.values.max() <= 0.95
    M, N, K = (c.astype(np.float64) for c in w.buckets[0].cols)
    lo, hi = W.GEMM_SPAN
    oob = ((np.log2(M) < lo[0] - 1e-9) | (np.log2(M) > hi[0] + 1e-9) | (np.log2(N) < lo[1] - 0.01)
           | (np.log2(N) > hi[1] + 0.01) | (np.log2(K) < lo[2] - 0.01) | (np.log2(K) > hi[2] + 0.01))
    assert 0.04 < oob.mean() < 0.12
    B_, q, kv = w.buckets[1].cols
    assert np.all(kv >= q)


def test_cfg4_step_structure():
    w = W.config4(n_steps=200)
    gemm, attn, elem = w.buckets
    assert np.all(np.diff(gemm.step_off) == 129) and np.all(np.diff(elem.step_off) == 130)
    per = np.diff(attn.step_off)
    assert set(np.unique(per)) <= {32, 64}
    for b in w.buckets:
        assert b.step_off[0] == 0 and b.step_off[-1] == b.n and b.step_off.shape[0] == 201
    # nine kernels per layer (+1 prefill attention) + 3 per-step rows
    assert np.all(np.diff(gemm.step_off) + np.diff(elem.step_off) + per == 9 * 32 + 3 + (per - 32))
    assert w.cfg_off[0] == 0 and w.cfg_off[-1] == 200
    M = gemm.cols[0].reshape(200, 129)
    assert np.all(M[:, 0] == M[:, 127]) and np.all(M[:, 128] <= 257)      # LM head sees one token per sequence


def test_cfg5_exact_row_count_and_csr():
    w = W.config5(n_rows=12345, n_specs=4)
    assert w.n_rows == 12345 and len(w.specs) == 4
    for b in w.buckets:
        assert b.step_off[-1] == b.n and b.step_off.shape[0] == w.n_steps + 1
        assert np.all(np.diff(b.step_off) >= 0)
    grp = [b for b in w.buckets if b.family == W.FAM_GROUPED][0]
    assert len(grp.cols) == 10
    for s in w.specs:
        assert 80 <= s["n_sm"] <= 160 and 0.3e15 <= s["peak_flops"] <= 2.5e15 and 2e12 <= s["peak_bw"] <= 8e12
