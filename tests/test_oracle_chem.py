"""Pins for the oracle's chemistry source term (Eq. 2-6) and the batch drivers.  No GPU.

Closed forms on hand-built mechanisms fix units, signs and indices of every term; linear invariants
and the adiabatic enthalpy fix the stoichiometric bookkeeping and the energy equation on the
synthetic mechanisms; a brute-force fixed-step run and an independent library integrator (scipy
Radau) fix the adaptive drivers end to end.
"""
import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_1309_2710_b200 import synth

RU = 8.314462618e7
RC = 1.98720425864
P = synth.P_ATM


def _integrate(mech, y0, dt, method="rkck", rtol=1e-11, atol=1e-16):
    om = oracle.OracleMech(mech)
    out, status, stats = om.integrate(np.asarray(y0, dtype=float).reshape(-1, 1), P, dt, rtol, atol, method)
    assert status[0] == 0
    return out[:, 0]


@pytest.mark.parametrize("method", ["rkck", "rkc"])
def test_first_order_A_to_B_with_heat_release(method):
    """A -> B, equal W, beta = 0, E = 0: Y_A = Y_A0 exp(-A t) independent of rho; with cp/R = a1 and
    a6_A != a6_B the adiabatic temperature is T0 + (a6_A - a6_B)(Y_A0 - Y_A)/a1."""
    nasa = np.zeros((2, 7))
    nasa[:, 0] = 4.0
    nasa[0, 5], nasa[1, 5] = 500.0, -1500.0
    k = 3.0e5
    mech = synth.toy_mechanism(2, [({0: 1}, {1: 1}, k, 0.0, 0.0)], W=[20.0, 20.0], nasa=nasa)
    dt = 4e-6
    rtol = 1e-11 if method == "rkck" else 1e-9
    y = _integrate(mech, [1200.0, 0.7, 0.3], dt, method, rtol=rtol)
    ya = 0.7 * np.exp(-k * dt)
    tol = 1e-8 if method == "rkck" else 2e-6       # 2nd-order RKC: global error ~ steps x rtol
    assert abs(y[1] / ya - 1) < tol and abs(y[2] - (1.0 - ya)) < tol
    T = 1200.0 + (500.0 + 1500.0) * (0.7 - ya) / 4.0
    assert abs(y[0] / T - 1) < tol


def test_bateman_chain():
    """A -> B -> C: Y_B(t) = Y_A0 k1/(k2-k1) (e^{-k1 t} - e^{-k2 t}) + Y_B0 e^{-k2 t} (equal W, same thermo)."""
    k1, k2 = 4.0e5, 1.5e5
    mech = synth.toy_mechanism(3, [({0: 1}, {1: 1}, k1, 0.0, 0.0), ({1: 1}, {2: 1}, k2, 0.0, 0.0)])
    dt = 5e-6
    y = _integrate(mech, [1000.0, 0.6, 0.1, 0.3], dt)
    ya = 0.6 * np.exp(-k1 * dt)
    yb = 0.6 * k1 / (k2 - k1) * (np.exp(-k1 * dt) - np.exp(-k2 * dt)) + 0.1 * np.exp(-k2 * dt)
    assert abs(y[0] - 1000.0) < 1e-9
    assert abs(y[1] / ya - 1) < 1e-9 and abs(y[2] / yb - 1) < 1e-9 and abs(y[3] - (1 - ya - yb)) < 1e-9


def test_bimolecular_A_plus_B():
    """A + B -> C + D, all W equal, same thermo: rho and T constant; with a = C_A0, b = C_B0,
    xi = a b (e^{(b-a)kt} - 1)/(b e^{(b-a)kt} - a).  Pins rho = P Wbar/(Ru T) and C_k = rho Y_k/W_k."""
    W, T0, k = 25.0, 1500.0, 2.0e12
    mech = synth.toy_mechanism(4, [({0: 1, 1: 1}, {2: 1, 3: 1}, k, 0.0, 0.0)], W=[W] * 4)
    rho = P * W / (RU * T0)
    a, b = rho * 0.3 / W, rho * 0.5 / W
    dt = 2e-6
    y = _integrate(mech, [T0, 0.3, 0.5, 0.15, 0.05], dt)
    e = np.exp((b - a) * k * dt)
    xi = a * b * (e - 1) / (b * e - a)
    assert xi / a > 0.2                                  # the reaction actually progressed
    assert abs(y[0] - T0) < 1e-9
    for idx, c0, sgn in ((1, a, -1), (2, b, -1), (3, rho * 0.15 / W, 1), (4, rho * 0.05 / W, 1)):
        assert abs(y[idx] / ((c0 + sgn * xi) * W / rho) - 1) < 1e-9


def test_third_body():
    """A + M -> B + M: unit efficiencies give first order with k_eff = k P/(Ru T); one alpha != 1 gives
    [M] = C_tot + (alpha-1) C_k (checked on f at t = 0).  P:80 / R22."""
    W, T0, k = 30.0, 1100.0, 5.0e10
    rx = [({0: 1}, {1: 1}, k, 0.0, 0.0)]
    mech = synth.toy_mechanism(3, rx, W=[W] * 3, third_body={0: {}})
    dt = 3e-6
    y = _integrate(mech, [T0, 0.8, 0.1, 0.1], dt)
    keff = k * P / (RU * T0)
    assert 0.05 < keff * dt < 5
    assert abs(y[1] / (0.8 * np.exp(-keff * dt)) - 1) < 1e-9
    mech2 = synth.toy_mechanism(3, rx, W=[W] * 3, third_body={0: {0: 2.5, 2: 0.5}})
    f = oracle.OracleMech(mech2).rhs([T0, 0.8, 0.1, 0.1], P)
    rho = P * W / (RU * T0)
    C = rho * np.array([0.8, 0.1, 0.1]) / W
    M = C.sum() + 1.5 * C[0] - 0.5 * C[2]
    assert abs(f[1] / (-k * M * C[0] * W / rho) - 1) < 1e-14
    assert abs(f[2] + f[1]) < 1e-14 * abs(f[1]) and f[3] == 0.0


def test_stoichiometric_coefficients_and_unequal_weights():
    """2A + B -> 3C with W_C = (2 W_A + W_B)/3: f from Eq. 2-4 by hand; mass is conserved."""
    WA, WB = 2.0, 32.0
    WC = (2 * WA + WB) / 3
    k, T0 = 7.0e15, 900.0
    mech = synth.toy_mechanism(3, [({0: 2, 1: 1}, {2: 3}, k, 0.0, 0.0)], W=[WA, WB, WC])
    Y = np.array([0.2, 0.5, 0.3])
    f = oracle.OracleMech(mech).rhs(np.concatenate([[T0], Y]), P)
    rho = P / (RU * T0 * np.sum(Y / np.array([WA, WB, WC])))
    C = rho * Y / np.array([WA, WB, WC])
    Om = k * C[0] ** 2 * C[1]
    expect = np.array([-2 * Om * WA, -Om * WB, 3 * Om * WC]) / rho
    assert np.allclose(f[1:], expect, rtol=1e-14, atol=0)
    assert abs(f[1:].sum()) < 1e-13 * np.abs(f[1:]).max()


def test_arrhenius_against_mpmath():
    """k(T) = A T^beta exp(-E/(R T)) (Eq. 5) at three temperatures, 40-digit reference."""
    mp.mp.dps = 40
    for (A, beta, E) in ((3.2e13, -0.7, 17041.0), (5.0e4, 2.0, 0.0), (1.0e9, 1.3, 29999.0)):
        mech = synth.toy_mechanism(2, [({0: 1}, {1: 1}, A, beta, E)])
        om = oracle.OracleMech(mech)
        for T in (800.0, 1234.5, 2400.0):
            f = om.rhs([T, 0.4, 0.6], P)
            kref = mp.mpf(A) * mp.mpf(T) ** mp.mpf(beta) * mp.exp(-mp.mpf(E) / (mp.mpf(RC) * mp.mpf(T)))
            assert abs(-f[1] / 0.4 / float(kref) - 1) < 5e-15


def _enthalpy(mech, y):
    T, Y = y[0], y[1:]
    a = mech.nasa
    hRT = a[:, 0] + a[:, 1] * T / 2 + a[:, 2] * T ** 2 / 3 + a[:, 3] * T ** 3 / 4 + a[:, 4] * T ** 4 / 5 + a[:, 5] / T
    return np.sum(Y * RU * T * hRT / mech.mol_weight)


@pytest.mark.parametrize("cfg,method", [(0, "rkck"), (0, "rkc"), (2, "rkc"), (2, "rkck"), (3, "rkc")])
def test_invariants_on_synthetic_mechanisms(cfg, method):
    """Sum Y and every element mass fraction are linear invariants (element-balanced reactions, W from
    the element counts): conserved to round-off by any Runge-Kutta step sequence.  Total enthalpy is
    conserved to O(tolerance)."""
    mech = synth.make_mechanism(cfg)
    N = 24 if cfg < 3 else 6
    st, p = synth.make_states(cfg, N)
    out, status, stats = oracle.OracleMech(mech).integrate(st, p, 1e-6, 1e-8, 1e-12, method)
    assert np.all((status == 0) | (status == 4))
    assert np.max(np.abs(out[1:].sum(0) - 1.0)) < 5e-14
    aw = np.array([synth.ATOMIC_WEIGHT[e] for e in mech.elements])
    Z0 = (mech.elem_counts * aw).T @ (st[1:] / mech.mol_weight[:, None])
    Z1 = (mech.elem_counts * aw).T @ (out[1:] / mech.mol_weight[:, None])
    assert np.max(np.abs(Z1 - Z0)) < 5e-14
    assert np.allclose(Z0.sum(0), 1.0, atol=1e-13)       # W_k = sum_e n_ek A_e
    for i in range(N):
        h0, h1 = _enthalpy(mech, st[:, i]), _enthalpy(mech, out[:, i])
        scale = RU * st[0, i] / mech.mol_weight.min()
        assert abs(h1 - h0) < 2e-6 * scale
    assert np.abs(out[0] - st[0]).max() > 0.5            # something happened


def test_adaptive_drivers_against_brute_force_and_library():
    """cfg0 mechanism, 3 states, dt = 1e-6: adaptive RKCK and RKC at rtol 1e-8 against (a) the oracle's
    own single-step RKCK applied 4000 times with fixed h (controller off) and (b) scipy Radau at
    rtol 1e-12 over the oracle's RHS -- an independent integrator."""
    from scipy.integrate import solve_ivp
    mech = synth.make_mechanism(0)
    om = oracle.OracleMech(mech)
    st, p = synth.make_states(1, 3)
    dt = 1e-6
    f = lambda t, y: om.rhs(y, p)
    for i in range(3):
        y0 = st[:, i].copy()
        y = y0.copy()
        n = 4000
        for s in range(n):
            y, _ = oracle.rkck_step(f, 0.0, y, dt / n)
        sol = solve_ivp(f, (0.0, dt), y0, method="Radau", rtol=1e-12, atol=1e-18)
        assert np.allclose(sol.y[:, -1], y, rtol=1e-9, atol=1e-15)
        for method, rt in (("rkck", 10.0), ("rkc", 300.0)):
            out, status, stats = om.integrate(y0.reshape(-1, 1), p, dt, 1e-8, 1e-12, method)
            assert status[0] == 0
            err = np.abs(out[:, 0] - y)
            assert np.all(err <= rt * 1e-8 * np.abs(y) + rt * 1e-12), (method, err / (1e-8 * np.abs(y) + 1e-12))


@pytest.mark.parametrize("cfg", [0, 2])
def test_rkck_and_rkc_agree(cfg):
    """Two independent integrators over one RHS at tight tolerance agree to ~1e-6 relative (RKC global error ~ steps x rtol) on Y > 1e-8."""
    mech = synth.make_mechanism(cfg)
    st, p = synth.make_states(cfg, 8)
    om = oracle.OracleMech(mech)
    a, sa, _ = om.integrate(st, p, 1e-6, 1e-10, 1e-14, "rkck")
    b, sb, _ = om.integrate(st, p, 1e-6, 1e-10, 1e-14, "rkc")
    assert np.all(sa == 0)
    big = np.abs(a) > 1e-8
    assert np.max(np.abs(b[big] / a[big] - 1)) < 2e-6


def test_batch_entry_layout_and_threads():
    """SoA layout, per-system pressure array, thread count independence (bitwise)."""
    mech = synth.make_mechanism(0)
    om = oracle.OracleMech(mech)
    st, p = synth.make_states(0, 40)
    a, _, sa = om.integrate(st, p, 1e-6, 1e-8, 1e-12, "rkck", nthreads=1)
    b, _, sb = om.integrate(st, p, 1e-6, 1e-8, 1e-12, "rkck", nthreads=4, pressure=np.full(40, p))
    assert np.array_equal(a, b) and np.array_equal(sa, sb)
    one, _, _ = om.integrate(st[:, 17:18], p, 1e-6, 1e-8, 1e-12, "rkck")
    assert np.array_equal(one[:, 0], a[:, 17])
    with pytest.raises(ValueError):
        om.integrate(st, p, -1.0, 1e-8, 1e-12, "rkck")
