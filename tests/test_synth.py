"""Input generator self-tests: shapes of BASELINE.json's configs, element
balance of every reaction, determinism, state recipe.  No GPU, no method arithmetic."""
import numpy as np
import pytest

from paper_1309_2710_b200 import synth


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_mechanism_shape_and_balance(cfg):
    spec = synth.CONFIGS[cfg]
    m = synth.make_mechanism(cfg)
    assert (m.n_species, m.n_reactions) == (spec.K, spec.R)
    assert m.n_third_body == 2 * spec.n_tb_pairs
    assert len({tuple(r) for r in m.elem_counts}) == spec.K and m.elem_counts.min() >= 0 and m.elem_counts.max() <= 4
    aw = np.array([synth.ATOMIC_WEIGHT[e] for e in m.elements])
    assert np.allclose(m.mol_weight, m.elem_counts @ aw)
    seen = set()
    for j in range(m.n_reactions):
        rs = slice(m.reac_ptr[j], m.reac_ptr[j + 1])
        ps = slice(m.prod_ptr[j], m.prod_ptr[j + 1])
        lhs = (m.elem_counts[m.reac_species[rs]] * m.reac_nu[rs, None]).sum(0)
        rhs = (m.elem_counts[m.prod_species[ps]] * m.prod_nu[ps, None]).sum(0)
        assert np.array_equal(lhs, rhs)
        assert 1 <= m.reac_nu[rs].sum() <= spec.max_side and 1 <= m.prod_nu[ps].sum() <= spec.max_side
        assert not set(m.reac_species[rs]) & set(m.prod_species[ps])
        key = (tuple(m.reac_species[rs]), tuple(m.reac_nu[rs]), tuple(m.prod_species[ps]), tuple(m.prod_nu[ps]))
        assert key not in seen
        seen.add(key)
    # forward/reverse pairs: reaction 2i+1 is reaction 2i reversed
    for j in range(0, m.n_reactions, 2):
        assert np.array_equal(m.reac_species[m.reac_ptr[j]:m.reac_ptr[j + 1]],
                              m.prod_species[m.prod_ptr[j + 1]:m.prod_ptr[j + 2]])
    for r, j in enumerate(m.tb_reaction):
        assert m.reac_nu[m.reac_ptr[j]:m.reac_ptr[j + 1]].sum() <= 2
        eff = m.tb_eff[m.tb_ptr[r]:m.tb_ptr[r + 1]]
        assert len(eff) == min(3, spec.K) and eff.min() >= 0.5 and eff.max() <= 3.0
    assert m.arr_beta.min() >= -1 and m.arr_beta.max() <= 2 and m.arr_E.min() >= 0 and m.arr_E.max() <= 30000
    T = np.linspace(300, 2500, 50)[:, None]
    cpR = sum(m.nasa[:, i] * T ** i for i in range(5))
    assert cpR.min() > 3.0 and cpR.max() < 8.0


def test_determinism_and_calibration_applied():
    a, b = synth.make_mechanism(3), synth.make_mechanism(3)
    assert np.array_equal(a.arr_A, b.arr_A) and np.array_equal(a.reac_species, b.reac_species)
    raw = synth.make_mechanism(3, calibrated=False)
    cal = synth.load_calibration()["mech3_seed0"]
    assert np.allclose(a.arr_A, raw.arr_A * cal["g"]) and a.rate_factor == cal["g"]
    lo, hi = cal["target_span"]
    p5, p95 = cal["sigma_min_p5_p50_p95_max"][1], cal["sigma_min_p5_p50_p95_max"][3]
    assert lo <= p5 and p95 <= hi and cal["recheck_max_rel_dev"] < 1e-6


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_states(cfg):
    spec = synth.CONFIGS[cfg]
    st, p = synth.make_states(cfg, 300)
    assert st.shape == (spec.K + 1, 300) and p == synth.P_ATM
    assert st[0].min() >= spec.T_range[0] and st[0].max() <= spec.T_range[1]
    assert np.allclose(st[1:].sum(0), 1.0) and st[1:].min() >= 0
    st2, _ = synth.make_states(cfg, 100)
    assert np.array_equal(st2, st[:, :100])                     # sweeps nest
    sim, _ = synth.make_states(cfg, 300, ordering="similar")
    assert np.all(np.diff(sim[0]) >= 0) and np.allclose(np.sort(st[0]), sim[0])
