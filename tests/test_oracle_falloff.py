"""Pins for the oracle's fall-off reactions (reading R31: the Chemkin-manual form the paper refers to,
P:80).  The oracle and its pins were committed before the CUDA path (ckb_mech_load3; parity in tests/test_gpu_falloff.py).

The pins reduce the fall-off rate to paths pinned elsewhere (third-body and plain reactions, test_oracle_chem.py) in its
two limits, and fix the constants of the blending function at the points where it has closed-form values:
Lindemann at P_r = 1 gives k_inf / 2; Troe gives F = F_cent at log10 P_r = -c, F = sqrt(F_cent) where the bracket is 1,
and F -> F_cent^(1 / (1 + 1/0.14^2)) as P_r -> infinity."""
import copy

import numpy as np
import pytest

import oracle
from paper_1309_2710_b200 import synth

RU, RC = 8.314462618e7, 1.98720425864
A_INF, B_INF, E_INF = 3.0e10, 0.5, 9000.0
A_0, B_0, E_0 = 4.0e16, -1.2, 3000.0
W = [20.0, 20.0, 30.0]


def _mech(troe=None, third_body=None, falloff=True, low_as_plain=False):
    """A (+M) -> B with an inert C; species 0 = A."""
    if low_as_plain:
        rx = [({0: 1}, {1: 1}, A_0, B_0, E_0)]
    else:
        rx = [({0: 1}, {1: 1}, A_INF, B_INF, E_INF)]
    m = synth.toy_mechanism(3, rx, W=W, third_body=third_body)
    if falloff:
        m.fo_reaction = np.array([0], dtype=np.int32)
        m.fo_low = np.array([[A_0, B_0, E_0]])
        m.fo_troe = np.array([[np.nan, 0, 0, 0]] if troe is None else [troe], dtype=np.float64)
    return m


def _k(A, b, E, T):
    return A * T ** b * np.exp(-E / (RC * T))


def _rate_A(om, T, Y, p):
    """-dC_A/dt / C_A = the effective first-order coefficient k (s^-1) the oracle applied."""
    y = np.array([T, *Y])
    f = om.rhs(y, p)
    rho = p / (RU * T * sum(Yk / Wk for Yk, Wk in zip(Y, W)))
    return -f[1] / Y[0], rho


def _p_for_M(M, T):
    return M * RU * T                       # all efficiencies 1: [M] = C_tot = p / (Ru T)


@pytest.mark.parametrize("T", [900.0, 1400.0])
def test_lindemann_half_at_unit_reduced_pressure(T):
    om = oracle.OracleMech(_mech())
    kinf, k0 = _k(A_INF, B_INF, E_INF, T), _k(A_0, B_0, E_0, T)
    k, _ = _rate_A(om, T, [0.3, 0.2, 0.5], _p_for_M(kinf / k0, T))
    assert k == pytest.approx(kinf / 2.0, rel=1e-13)
    # general P_r: k = k_inf k_0 M / (k_inf + k_0 M)
    for M in (1e-9, 3e-6, 2e-3):
        k, _ = _rate_A(om, T, [0.3, 0.2, 0.5], _p_for_M(M, T))
        assert k == pytest.approx(kinf * k0 * M / (kinf + k0 * M), rel=1e-13)


def test_limits_reduce_to_third_body_and_plain_reactions():
    """P_r -> 0: the third-body reaction with (A_0, beta_0, E_0) and the same efficiencies; P_r -> infinity: the plain
    reaction with the high-pressure parameters.  Both comparison mechanisms go through paths pinned in test_oracle_chem."""
    eff = {0: {2: 2.5, 1: 0.7}}
    fo = oracle.OracleMech(_mech(third_body=eff))
    tb = oracle.OracleMech(_mech(third_body=eff, falloff=False, low_as_plain=True))
    plain = oracle.OracleMech(_mech(falloff=False))
    T, Y = 1200.0, [0.25, 0.05, 0.7]
    y = np.array([T, *Y])
    lo = 1e-12 * synth.P_ATM                                  # P_r ~ 1e-9
    assert np.allclose(fo.rhs(y, lo), tb.rhs(y, lo), rtol=1e-7, atol=0)
    hi = 1e14 * synth.P_ATM                                   # P_r ~ 1e+11
    assert np.allclose(fo.rhs(y, hi), plain.rhs(y, hi), rtol=1e-7, atol=0)
    mid = synth.P_ATM
    assert not np.allclose(fo.rhs(y, mid), plain.rhs(y, mid), rtol=1e-3)
    assert not np.allclose(fo.rhs(y, mid), tb.rhs(y, mid), rtol=1e-3)
    # the efficiencies enter through [M]: without them the rate differs
    assert not np.allclose(oracle.OracleMech(_mech()).rhs(y, mid), fo.rhs(y, mid), rtol=1e-3)


@pytest.mark.parametrize("troe", [(0.6, 100.0, 2000.0, 5000.0), (0.35, 250.0, 1500.0, np.inf)])
def test_troe_closed_form_points(troe):
    a, T3, T1, T2 = troe
    om = oracle.OracleMech(_mech(troe=troe))
    T = 1000.0
    kinf, k0 = _k(A_INF, B_INF, E_INF, T), _k(A_0, B_0, E_0, T)
    Fcent = (1 - a) * np.exp(-T / T3) + a * np.exp(-T / T1) + (np.exp(-T2 / T) if np.isfinite(T2) else 0.0)
    lF = np.log10(Fcent)
    c, n = -0.4 - 0.67 * lF, 0.75 - 1.27 * lF

    def k_at(Pr):
        return _rate_A(om, T, [0.4, 0.1, 0.5], _p_for_M(Pr * kinf / k0, T))[0]

    Pr = 10.0 ** (-c)                                        # bracket = 0: F = F_cent
    assert k_at(Pr) == pytest.approx(kinf * Pr / (1 + Pr) * Fcent, rel=1e-12)
    Pr = 10.0 ** (n / 1.14 - c)                              # (x) / (n - 0.14 x) = 1 at x = n / 1.14: F = sqrt(F_cent)
    assert k_at(Pr) == pytest.approx(kinf * Pr / (1 + Pr) * np.sqrt(Fcent), rel=1e-12)
    Pr = 10.0 ** (-n / 0.86 - c)                             # ratio = -1 at x = -n / 0.86: again sqrt(F_cent)
    assert k_at(Pr) == pytest.approx(kinf * Pr / (1 + Pr) * np.sqrt(Fcent), rel=1e-12)
    # far limit: x / (n - 0.14 x) -> -1/0.14, so F -> F_cent^(1/(1 + 1/0.14^2)); approached like 1/log10(P_r)
    Pr = 1e280
    lim = Fcent ** (1.0 / (1.0 + 1.0 / 0.14 ** 2))
    assert k_at(Pr) / kinf == pytest.approx(lim, rel=2e-2 * abs(np.log(Fcent)))
    # Lindemann is the F_cent = 1 case: (a, T***, T*) = (1, *, inf) gives F_cent = exp(0) = 1 exactly
    one = oracle.OracleMech(_mech(troe=(1.0, 300.0, np.inf, np.inf)))
    lin = oracle.OracleMech(_mech())
    y = np.array([T, 0.4, 0.1, 0.5])
    assert np.allclose(one.rhs(y, synth.P_ATM), lin.rhs(y, synth.P_ATM), rtol=1e-14, atol=0)


def test_only_listed_reactions_change_and_integration_runs():
    """In a full synthetic mechanism, turning some third-body reactions into fall-off reactions changes f(y) only through
    those reactions: with k_0 = k_inf * 1e30 (P_r huge, Lindemann) they become plain reactions -- compare with the mechanism
    that has those reactions removed from the third-body list."""
    base = synth.make_mechanism(0)
    pick = base.tb_reaction[:3]
    fo = copy.copy(base)
    fo.fo_reaction = np.ascontiguousarray(pick, dtype=np.int32)
    fo.fo_low = np.stack([base.arr_A[pick] * 1e30, base.arr_beta[pick], base.arr_E[pick]], axis=1)
    fo.fo_troe = np.full((3, 4), np.nan)
    plain = copy.copy(base)
    keep = [i for i, j in enumerate(base.tb_reaction) if j not in set(pick.tolist())]
    ptr = [0]
    sp, eff = [], []
    for i in keep:
        sp += base.tb_species[base.tb_ptr[i]:base.tb_ptr[i + 1]].tolist()
        eff += base.tb_eff[base.tb_ptr[i]:base.tb_ptr[i + 1]].tolist()
        ptr.append(len(sp))
    plain.tb_reaction = np.array([base.tb_reaction[i] for i in keep], dtype=np.int32)
    plain.tb_ptr, plain.tb_species, plain.tb_eff = np.array(ptr, dtype=np.int32), np.array(sp, dtype=np.int32), np.array(eff)
    a, b = oracle.OracleMech(fo), oracle.OracleMech(plain)
    states, p = synth.make_states(0, 16)
    for i in range(16):
        assert np.allclose(a.rhs(states[:, i].copy(), p), b.rhs(states[:, i].copy(), p), rtol=1e-12, atol=0)
    y1, st, _ = a.integrate(states, p, 1e-6, 1e-8, 1e-12, "rkck")
    assert (st == 0).all() and np.abs(y1[1:].sum(0) - 1.0).max() < 1e-12
