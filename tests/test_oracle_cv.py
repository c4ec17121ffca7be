"""Pins for the constant-volume closure of the oracle (reading R29: the paper only mentions the
variant).  Nothing here retypes the oracle's formula: the pins are the conservation law the closure exists to
satisfy (internal energy of an adiabatic constant-volume reactor), evaluated from the NASA fits in numpy, a linear
special case with a closed form, and the relation to the constant-pressure closure."""
import numpy as np
import pytest

import oracle
from paper_1309_2710_b200 import synth

RU = 8.314462618e7   # erg/(mol K)


def _u_mass(mech, y):
    """Specific internal energy (erg/g) from the NASA fits: u = sum_k Y_k (h_k - Ru T) / W_k."""
    T, Y = y[0], y[1:]
    a = mech.nasa
    h_rt = a[:, 0] + a[:, 1] * T / 2 + a[:, 2] * T ** 2 / 3 + a[:, 3] * T ** 3 / 4 + a[:, 4] * T ** 4 / 5 + a[:, 5] / T
    return float((Y * RU * T * (h_rt - 1.0) / mech.mol_weight).sum())


def _cv_mass(mech, y):
    T, Y = y[0], y[1:]
    a = mech.nasa
    cp_r = a[:, 0] + a[:, 1] * T + a[:, 2] * T ** 2 + a[:, 3] * T ** 3 + a[:, 4] * T ** 4
    return float((Y * RU * (cp_r - 1.0) / mech.mol_weight).sum())


def _rho(mech, y, p):
    return p / (RU * y[0] * (y[1:] / mech.mol_weight).sum())


@pytest.mark.parametrize("cfg", [0, 2, 3])
def test_rhs_conserves_internal_energy_identically(cfg):
    """du/dt = sum_k u_k/W_k dY_k/dt + c_v dT/dt must vanish for every state: an algebraic identity of f(y) that a
    wrong sign, a missing -Ru T, c_p in place of c_v or a wrong density all break at O(1)."""
    mech = synth.make_mechanism(cfg)
    om = oracle.OracleMech(mech)
    states, p = synth.make_states(cfg, 24)
    for i in range(24):
        y = states[:, i].copy()
        rho = _rho(mech, y, p) * (0.5 + 0.1 * i)          # any density, not just the one p would give
        f = om.rhs(y, rho, cv=True)
        T = y[0]
        a = mech.nasa
        h_rt = a[:, 0] + a[:, 1] * T / 2 + a[:, 2] * T ** 2 / 3 + a[:, 3] * T ** 3 / 4 + a[:, 4] * T ** 4 / 5 + a[:, 5] / T
        u_k = RU * T * (h_rt - 1.0) / mech.mol_weight
        terms = np.append(u_k * f[1:], _cv_mass(mech, y) * f[0])
        assert abs(terms.sum()) <= 1e-11 * np.abs(terms).sum()
        assert abs(f[1:].sum()) <= 1e-12 * np.abs(f[1:]).sum() + 1e-300     # mass conserved


def test_species_rates_match_constant_pressure_at_equal_density():
    """The closure only changes the energy equation: with rho = p Wbar/(Ru T) the species rates are those of the
    constant-pressure f(y), and dT/dt differs by the factor (sum h_k w_k / c_p) -> (sum u_k w_k / c_v)."""
    mech = synth.make_mechanism(2)
    om = oracle.OracleMech(mech)
    states, p = synth.make_states(2, 16)
    for i in range(16):
        y = states[:, i].copy()
        fp, fv = om.rhs(y, p), om.rhs(y, _rho(mech, y, p), cv=True)
        assert np.allclose(fv[1:], fp[1:], rtol=1e-13, atol=0)
        assert fv[0] != fp[0]


@pytest.mark.parametrize("method", ["rkck", "rkc"])
def test_integration_conserves_internal_energy(method):
    mech = synth.make_mechanism(0)
    om = oracle.OracleMech(mech)
    states, p = synth.make_states(0, 64)
    rho = np.array([_rho(mech, states[:, i], p) for i in range(64)])
    y1, st, _ = om.integrate(states, 0.0, 2e-5, 1e-9, 1e-13, method, pressure=rho, cv=True)
    assert (st == 0).all()
    moved = np.abs(y1[0] - states[0]).max()
    assert moved > 1.0                                           # the batch does react (kelvins of change)
    for i in range(64):
        u0, u1 = _u_mass(mech, states[:, i]), _u_mass(mech, y1[:, i])
        scale = _cv_mass(mech, states[:, i]) * states[0, i]
        assert abs(u1 - u0) <= 2e-7 * scale                      # nonlinear invariant: kept to the tolerance
    assert np.abs(y1[1:].sum(0) - 1.0).max() < 1e-12


@pytest.mark.parametrize("method", ["rkck", "rkc"])
def test_constant_cv_closed_form(method):
    """A -> B, equal W, temperature-independent c_p/R = a1 for both, heats of formation a6: then
    (a1 - 1) T + Y_A a6_A + Y_B a6_B is a LINEAR invariant of the constant-volume system, which Runge-Kutta methods
    keep to round-off; at constant pressure the invariant has a1 in place of a1 - 1."""
    nasa = np.zeros((2, 7))
    nasa[:, 0] = 4.0
    nasa[0, 5], nasa[1, 5] = 3000.0, -2000.0
    mech = synth.toy_mechanism(2, [({0: 1}, {1: 1}, 4e5, 0.0, 3000.0)], W=[20.0, 20.0], nasa=nasa)
    om = oracle.OracleMech(mech)
    N = 16
    states = np.zeros((3, N))
    states[0] = np.linspace(900.0, 1600.0, N)
    states[1] = np.linspace(0.2, 1.0, N)
    states[2] = 1.0 - states[1]
    inv = lambda s_, c: c * s_[0] + s_[1] * 3000.0 + s_[2] * (-2000.0)
    yv, st, _ = om.integrate(states, 1e-4, 5e-6, 1e-8, 1e-12, method, cv=True)
    assert (st == 0).all() and (yv[1] < states[1]).all()
    assert np.allclose(inv(yv, 3.0), inv(states, 3.0), rtol=1e-13, atol=0)
    assert not np.allclose(inv(yv, 4.0), inv(states, 4.0), rtol=1e-6, atol=0)
    yp, st, _ = om.integrate(states, synth.P_ATM, 5e-6, 1e-8, 1e-12, method)
    assert np.allclose(inv(yp, 4.0), inv(states, 4.0), rtol=1e-13, atol=0)     # the constant-pressure counterpart
    # the heat released raises T more at constant volume (c_v < c_p)
    assert ((yv[0] - states[0]) > 0).all()
