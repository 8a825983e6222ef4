"""Pins for the layer-homogeneous form of step composition (t_gpu = L t_layer + t_lm_head +
t_embed): rows carry multiplicities; the weighted sum must equal the sum over the materialised rows."""
import numpy as np

from oracle import oracle as O
import workloads as W


def test_multiplicity_equals_repetition():
    rng = np.random.Generator(np.random.PCG64(5))
    lat = rng.uniform(1e-6, 1e-3, 37)
    mult = rng.integers(0, 5, 37)
    off = np.array([0, 10, 10, 25, 37])
    rep = np.repeat(lat, mult)                                     # the same kernels written out m_k times
    roff = np.concatenate([[0], np.cumsum(mult)])[off]
    for params in (W.STEP_PARAMS_ZERO, W.STEP_PARAMS_CFG4, W.STEP_PARAMS_HOSTBOUND):
        sw, cw = O.compose([lat], [off], 4, params, np.array([0, 3, 4]), mults=[mult])
        sr, cr = O.compose([rep], [roff], 4, params, np.array([0, 3, 4]))
        assert np.allclose(sw, sr, rtol=1e-13, atol=0) and np.allclose(cw, cr, rtol=1e-13, atol=0)


def test_paper_formula_l_times_layer_plus_head_plus_embed():
    # one step: a layer of two kernels (3 us, 5 us) repeated L = 32 times, an LM head (7 us), an embedding (1 us)
    lat = np.array([3e-6, 5e-6, 7e-6, 1e-6])
    step, _ = O.compose([lat], [np.array([0, 4])], 1, W.STEP_PARAMS_ZERO, np.array([0, 1]), mults=[np.array([32, 32, 1, 1])])
    assert abs(step[0] - (32 * (3e-6 + 5e-6) + 7e-6 + 1e-6)) < 1e-18
    # Eq. 4's n counts launches, i.e. multiplicities: 66 launches x 4 us
    step, _ = O.compose([lat], [np.array([0, 4])], 1, W.STEP_PARAMS_CFG4, np.array([0, 1]), mults=[np.array([32, 32, 1, 1])])
    assert abs(step[0] - (32 * 8e-6 + 8e-6 + 66 * 4e-6)) < 1e-18


def test_missing_multiplicities_are_ones_and_zero_drops_a_row():
    lat = [np.array([1.0, 2.0, 4.0]), np.array([8.0, 16.0])]
    offs = [np.array([0, 2, 3]), np.array([0, 1, 2])]
    s1, _ = O.compose(lat, offs, 2, W.STEP_PARAMS_ZERO, np.array([0, 2]), mults=[None, np.array([1, 0])])
    assert list(s1) == [11.0, 4.0]


def test_layer_homogeneous_config4_equals_the_materialised_one():
    full = W.config4(n_steps=23, n_layers=5)
    ded = W.config4(n_steps=23, n_layers=5, dedupe=True)
    assert ded.n_rows * 4 < full.n_rows
    def steps(w):
        lats = [O.predict_bucket(b, w.specs, W.TIER_NONE)["lat"][0] for b in w.buckets]
        return O.compose(lats, [b.step_off for b in w.buckets], w.n_steps, w.step_params, w.cfg_off,
                         mults=[b.mult for b in w.buckets])
    sf, cf = steps(full)
    sd, cd = steps(ded)
    assert np.allclose(sf, sd, rtol=1e-12, atol=0) and np.allclose(cf, cd, rtol=1e-12, atol=0)
