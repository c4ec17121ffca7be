"""Pins for the oracle's two-range NASA thermodynamics (reading R30: species k uses the high-range
coefficients where T > T_mid[k]).  None retypes the oracle's selection: the pins reduce the two-range f(y) to the one-range
f(y) (pinned in test_oracle_chem.py) on mechanisms assembled in numpy, and check the conservation laws that only hold if
the SAME range supplies c_p and h (total enthalpy at constant pressure, internal energy at constant volume)."""
import copy

import numpy as np
import pytest

import oracle
from paper_1309_2710_b200 import synth

RU = 8.314462618e7


def _two(cfg):
    spec = synth.CONFIGS[cfg]
    return synth.with_two_range_thermo(synth.make_mechanism(cfg), spec.T_range)


def _one_range(mech, nasa):
    m = copy.copy(mech)
    m.nasa, m.nasa_high, m.T_mid = np.ascontiguousarray(nasa), None, None
    return m


def _h_mass(mech, y):
    """Specific enthalpy (erg/g) with the range chosen per species in numpy."""
    T, Y = y[0], y[1:]
    a = np.where((T > mech.T_mid)[:, None], mech.nasa_high, mech.nasa)
    h_rt = a[:, 0] + a[:, 1] * T / 2 + a[:, 2] * T ** 2 / 3 + a[:, 3] * T ** 3 / 4 + a[:, 4] * T ** 4 / 5 + a[:, 5] / T
    return float((Y * RU * T * h_rt / mech.mol_weight).sum()), float((Y * RU * T * (h_rt - 1.0) / mech.mol_weight).sum())


def test_recipe_is_continuous_and_straddled():
    mech = _two(2)
    T = mech.T_mid
    cp = lambda a: a[:, 0] + a[:, 1] * T + a[:, 2] * T ** 2 + a[:, 3] * T ** 3 + a[:, 4] * T ** 4
    h = lambda a: a[:, 0] + a[:, 1] * T / 2 + a[:, 2] * T ** 2 / 3 + a[:, 3] * T ** 3 / 4 + a[:, 4] * T ** 4 / 5 + a[:, 5] / T
    assert np.allclose(cp(mech.nasa_high), cp(mech.nasa), rtol=1e-12)
    assert np.allclose(h(mech.nasa_high), h(mech.nasa), rtol=1e-12)
    assert not np.allclose(mech.nasa_high[:, 1:5], mech.nasa[:, 1:5])
    states, _ = synth.make_states(2, 256)
    above = (states[0][None, :] > mech.T_mid[:, None]).mean()
    assert 0.2 < above < 0.8


@pytest.mark.parametrize("cfg", [0, 2, 3])
def test_reduces_to_one_range_per_species(cfg):
    """f(y) of the two-range mechanism at state y equals f(y) of a ONE-range mechanism whose coefficient rows were
    picked per species in numpy for that y's temperature (a wrong comparison direction, a per-mechanism instead of
    per-species switch, or mixing c_p of one range with h of the other all fail)."""
    mech = _two(cfg)
    om = oracle.OracleMech(mech)
    states, p = synth.make_states(cfg, 24)
    n_mixed = 0
    for i in range(24):
        y = states[:, i].copy()
        use_hi = y[0] > mech.T_mid
        n_mixed += int(0 < use_hi.sum() < len(use_hi))
        ref = oracle.OracleMech(_one_range(mech, np.where(use_hi[:, None], mech.nasa_high, mech.nasa)))
        for cv, arg in ((False, p), (True, 1.3e-4)):
            assert np.array_equal(om.rhs(y, arg, cv=cv), ref.rhs(y, arg, cv=cv))
        lo_only = oracle.OracleMech(_one_range(mech, mech.nasa)).rhs(y, p)
        if use_hi.any():
            assert lo_only[0] != om.rhs(y, p)[0]
    assert n_mixed >= 4                                              # states between two species' T_mid


def test_limits_of_the_switch():
    mech = _two(0)
    states, p = synth.make_states(0, 6)
    for tm, nasa in ((1e9, mech.nasa), (0.0, mech.nasa_high)):
        m2 = copy.copy(mech)
        m2.T_mid = np.full(mech.n_species, tm)
        a, b = oracle.OracleMech(m2), oracle.OracleMech(_one_range(mech, nasa))
        for i in range(6):
            assert np.array_equal(a.rhs(states[:, i].copy(), p), b.rhs(states[:, i].copy(), p))
    # identical ranges: the switch is invisible
    m3 = copy.copy(mech)
    m3.nasa_high = mech.nasa.copy()
    a, b = oracle.OracleMech(m3), oracle.OracleMech(_one_range(mech, mech.nasa))
    y1 = a.integrate(states, p, 1e-6, 1e-8, 1e-12, "rkck")
    y2 = b.integrate(states, p, 1e-6, 1e-8, 1e-12, "rkck")
    assert np.array_equal(y1[0], y2[0]) and np.array_equal(y1[2], y2[2])


@pytest.mark.parametrize("method", ["rkck", "rkc"])
def test_enthalpy_and_energy_conserved_across_the_switch(method):
    """Adiabatic reactors conserve h (constant pressure) / u (constant volume); with continuous fits that holds through
    T_mid, and only if c_p in the denominator belongs to the same range as h_k in the numerator."""
    mech = _two(0)
    om = oracle.OracleMech(mech)
    states, p = synth.make_states(0, 64)
    rho = synth.make_densities(mech, states, p)
    for cv in (False, True):
        y1, st, _ = om.integrate(states, 0.0 if cv else p, 2e-5, 1e-9, 1e-13, method, pressure=rho if cv else None, cv=cv)
        assert (st == 0).all()
        crossed = 0
        for i in range(64):
            e0, e1 = _h_mass(mech, states[:, i])[int(cv)], _h_mass(mech, y1[:, i])[int(cv)]
            assert abs(e1 - e0) <= 3e-7 * RU * states[0, i] * 4.0 / mech.mol_weight.min()
            crossed += int(((states[0, i] > mech.T_mid) != (y1[0, i] > mech.T_mid)).any())
        assert crossed >= 3                                          # some systems do pass a T_mid while reacting
