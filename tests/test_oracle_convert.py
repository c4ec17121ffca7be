"""Pins for the oracle's Appendix-A converter: reverse Arrhenius parameters from
k_f / K_c at three temperatures.  No GPU.

Eq. A.10-A.12 are closed forms of a 3 x 3 linear system, so three points taken FROM an Arrhenius law must give that law
back to round-off (exact round trip) -- with numpy's linear solve as the independent route.  The equilibrium constant
(reading R32, Chemkin form) is pinned on hand-built species whose NASA fits have only a1, a6, a7: there K_c is itself of
Arrhenius form, so the reverse parameters are known in closed form (signs of Delta s and Delta h, the (P_atm/RuT)^dnu factor and
the direction of the division all show).
"""
import numpy as np
import pytest

import oracle
from paper_1309_2710_b200 import synth

RU, RC, PATM = 8.314462618e7, 1.98720425864, 1.01325e6


@pytest.mark.parametrize("A,beta,Tar", [(3.2e13, 0.0, 8000.0), (1.7e-4, 2.7, -350.0), (5.0e20, -1.9, 22000.0), (1.0, 0.0, 0.0)])
def test_fit_reverse_round_trip_and_linear_solve(A, beta, Tar):
    for T3 in ([1000.0, 1500.0, 2000.0], [2400.0, 300.0, 900.0], [800.0, 810.0, 3000.0]):
        T = np.array(T3)
        kr = A * T ** beta * np.exp(-Tar / T)
        got = oracle.fit_reverse(T, kr)
        assert abs(got[0] / A - 1) < 2e-9 and abs(got[1] - beta) < 3e-10 and abs(got[2] - Tar) < 3e-7 * max(1.0, abs(Tar))
        # independent route: ln k = ln A + beta ln T - Tar / T as a 3 x 3 linear system
        sol = np.linalg.solve(np.stack([np.ones(3), np.log(T), -1.0 / T], axis=1), np.log(kr))
        assert abs(got[1] - sol[1]) < 3e-10 and abs(got[2] - sol[2]) < 3e-7 * max(1.0, abs(Tar)) and abs(np.log(got[0]) - sol[0]) < 2e-9


def test_fit_interpolates_a_non_arrhenius_curve_at_the_three_temperatures():
    T = np.array([900.0, 1400.0, 2300.0])
    kr = 1e9 * T ** 1.3 * np.exp(-4000.0 / T) * (1 + 0.3 * np.sin(T / 300.0))
    A, b, Tar = oracle.fit_reverse(T, kr)
    assert np.max(np.abs(A * T ** b * np.exp(-Tar / T) / kr - 1)) < 1e-10


def _two_level_mech(dnu_case):
    """A <-> B (dnu = 0) or A <-> 2 B (dnu = +1), NASA fits with a1, a6, a7 only."""
    nasa = np.zeros((2, 7))
    nasa[0, [0, 5, 6]] = [4.5, -2500.0, 3.2]
    nasa[1, [0, 5, 6]] = [3.1, 1800.0, 5.7]
    prod = {1: 2} if dnu_case else {1: 1}
    return synth.toy_mechanism(2, [({0: 1}, prod, 4.0e11, 0.7, 12000.0)], W=[20.0, 10.0 if dnu_case else 20.0], nasa=nasa), nasa


@pytest.mark.parametrize("dnu_case", [0, 1])
def test_reverse_parameters_closed_form(dnu_case):
    mech, nasa = _two_level_mech(dnu_case)
    om = oracle.OracleMech(mech)
    nuB = 2 if dnu_case else 1
    da1 = nuB * nasa[1, 0] - nasa[0, 0]
    da6 = nuB * nasa[1, 5] - nasa[0, 5]
    da7 = nuB * nasa[1, 6] - nasa[0, 6]
    dnu = nuB - 1
    for T in (700.0, 1300.0, 2600.0):
        # ln K_p = da1 (ln T - 1) + da7 - da6 / T   (s/R - h/RT with a1, a6, a7 only)
        Kc = np.exp(da1 * (np.log(T) - 1.0) + da7 - da6 / T) * (PATM / (RU * T)) ** dnu
        assert abs(om.equilibrium_constant(0, T) / Kc - 1) < 1e-12
    # k_r = k_f / K_c = A T^beta e^(-E/RcT) e^(da1 - da7) T^(-da1) e^(da6/T) (Ru T / P_atm)^dnu : exactly Arrhenius
    A_r = 4.0e11 * np.exp(da1 - da7) * (RU / PATM) ** dnu
    beta_r = 0.7 - da1 + dnu
    E_r = 12000.0 - da6 * RC
    got = om.reverse_parameters(0, [1000.0, 1600.0, 2200.0])
    assert abs(got[0] / A_r - 1) < 1e-8 and abs(got[1] - beta_r) < 1e-9 and abs(got[2] - E_r) < 1e-5


def test_forward_and_fitted_reverse_reach_the_equilibrium_of_kc():
    """A <-> B at fixed T (equal, constant cp; equal enthalpies: isothermal): integrating the pair of irreversible
    reactions (forward, fitted reverse) to steady state gives C_B / C_A = K_c."""
    nasa = np.zeros((2, 7))
    nasa[0, [0, 5, 6]] = [3.5, 500.0, 3.0]
    nasa[1, [0, 5, 6]] = [3.5, 500.0, 4.1]         # same h: no heat release, T stays
    fwd = ({0: 1}, {1: 1}, 3.0e6, 0.0, 2000.0)
    m1 = synth.toy_mechanism(2, [fwd], W=[15.0, 15.0], nasa=nasa)
    Ar, br, Er = oracle.OracleMech(m1).reverse_parameters(0, [900.0, 1200.0, 1500.0])
    m2 = synth.toy_mechanism(2, [fwd, ({1: 1}, {0: 1}, Ar, br, Er)], W=[15.0, 15.0], nasa=nasa)
    om = oracle.OracleMech(m2)
    T0 = 1100.0
    y, st, _ = om.integrate(np.array([[T0], [1.0], [0.0]]), PATM, 2e-3, 1e-10, 1e-14, "rkck")
    assert st[0] == 0 and abs(y[0, 0] - T0) < 1e-6
    Kc = oracle.OracleMech(m1).equilibrium_constant(0, T0)
    assert abs((y[2, 0] / y[1, 0]) / Kc - 1) < 1e-6
    assert abs(Kc - np.exp(1.1)) < 1e-12           # ds/R = 1.1, dh = 0, dnu = 0
