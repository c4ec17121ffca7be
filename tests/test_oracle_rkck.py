"""Pins for the oracle's RKCK (section 2.3; Table 1).  No GPU.

Nothing here compares the oracle with itself: Table 1 is pinned by the rooted-tree order conditions in
exact rational arithmetic, the step by the closed-form stability polynomial on y' = lambda y, the order
by a measured slope on a problem with an analytic solution, the driver by invariants.
"""
from fractions import Fraction
from itertools import product

import numpy as np

import oracle


def _table():
    a, b, c, cs = oracle.rkck_tableau()
    fr = lambda x: Fraction(float(x)).limit_denominator(10 ** 7)
    A = [fr(x) for x in a]
    B = [[fr(x) for x in row] for row in b]          # B[i][j], i = 0..5 (stage i+1), j = 0..4
    return A, B, [fr(x) for x in c], [fr(x) for x in cs], (a, b, c, cs)


def test_table1_entries_are_the_rationals_they_round_to():
    A, B, Cw, Cs, (a, b, c, cs) = _table()
    for fr, x in zip(A + [q for row in B for q in row] + Cw + Cs,
                     list(a) + list(b.ravel()) + list(c) + list(cs)):
        assert float(fr) == float(x)                 # the double IS the nearest double of a small rational
    # fragments legible in P:96-101
    legible = {Fraction(37, 378), Fraction(2825, 27648), Fraction(250, 621), Fraction(18575, 48384),
               Fraction(125, 594), Fraction(13525, 55296), Fraction(277, 14336), Fraction(512, 1771),
               Fraction(1, 4), Fraction(-9, 10), Fraction(6, 5), Fraction(-11, 54), Fraction(5, 2),
               Fraction(-70, 27), Fraction(35, 27), Fraction(1631, 55296), Fraction(175, 512),
               Fraction(575, 13824), Fraction(44275, 110592), Fraction(253, 4096), Fraction(7, 8),
               Fraction(1, 5), Fraction(3, 10), Fraction(3, 40), Fraction(9, 40)}
    have = set(A) | {q for row in B for q in row} | set(Cw) | set(Cs)
    assert legible <= have


def _order_conditions(A, B, w, order):
    """Rooted-tree order conditions up to `order` for weights w (exact Fractions).
    Returns the list of (tree name, residual)."""
    s = 6
    M = [[B[i][j] if j < 5 else Fraction(0) for j in range(s)] for i in range(s)]
    one = [Fraction(1)] * s
    c = A
    mv = lambda v: [sum(M[i][j] * v[j] for j in range(s)) for i in range(s)]
    had = lambda u, v: [x * y for x, y in zip(u, v)]
    dot = lambda v: sum(wi * vi for wi, vi in zip(w, v))
    c2, c3, c4 = had(c, c), had(had(c, c), c), had(had(c, c), had(c, c))
    Ac, Ac2, Ac3 = mv(c), mv(c2), mv(c3)
    AAc, AAc2 = mv(Ac), mv(Ac2)
    AAAc = mv(AAc)
    conds = [("t1", dot(one) - 1)]
    if order >= 2:
        conds += [("t2", dot(c) - Fraction(1, 2))]
    if order >= 3:
        conds += [("t31", dot(c2) - Fraction(1, 3)), ("t32", dot(Ac) - Fraction(1, 6))]
    if order >= 4:
        conds += [("t41", dot(c3) - Fraction(1, 4)), ("t42", dot(had(c, Ac)) - Fraction(1, 8)),
                  ("t43", dot(Ac2) - Fraction(1, 12)), ("t44", dot(AAc) - Fraction(1, 24))]
    if order >= 5:
        conds += [("t51", dot(c4) - Fraction(1, 5)),
                  ("t52", dot(had(c2, Ac)) - Fraction(1, 10)),
                  ("t53", dot(had(c, Ac2)) - Fraction(1, 15)),
                  ("t54", dot(had(c, AAc)) - Fraction(1, 30)),
                  ("t55", dot(had(Ac, Ac)) - Fraction(1, 20)),
                  ("t56", dot(Ac3) - Fraction(1, 20)),
                  ("t57", dot(mv(had(c, Ac))) - Fraction(1, 40)),
                  ("t58", dot(AAc2) - Fraction(1, 60)),
                  ("t59", dot(AAAc) - Fraction(1, 120))]
    return conds


def test_table1_order_conditions_exact():
    """17 conditions to order 5 for c, 8 to order 4 for c*, row sums, and failure one order higher."""
    A, B, Cw, Cs, _ = _table()
    for i in range(6):
        assert sum(B[i]) == A[i]
    assert sum(Cw) == 1 and sum(Cs) == 1
    c5 = _order_conditions(A, B, Cw, 5)
    assert len(c5) == 17 and all(r == 0 for _, r in c5), [n for n, r in c5 if r != 0]
    c4 = _order_conditions(A, B, Cs, 4)
    assert len(c4) == 8 and all(r == 0 for _, r in c4)
    assert any(r != 0 for _, r in _order_conditions(A, B, Cs, 5)[8:])      # embedded is NOT 5th order
    # 6th-order bushy tree fails for c
    c5v = [a ** 5 for a in A]
    assert sum(w * v for w, v in zip(Cw, c5v)) != Fraction(1, 6)
    # error weights c - c* as printed in SURVEY C1
    diff = [x - y for x, y in zip(Cw, Cs)]
    assert diff == [Fraction(-277, 64512), 0, Fraction(6925, 370944), Fraction(-6925, 202752),
                    Fraction(-277, 14336), Fraction(277, 7084)]


def test_single_step_linear_closed_form():
    """y' = lambda y: y1/y0 = R(z) = sum z^k/k! (k<=5) + z^6/800; embedded R*(z) (Eq. 13-15)."""
    for z in (-0.7, -0.1, 0.3, 1.1):
        lam, h = z / 0.25, 0.25
        ynew, delta = oracle.rkck_step(lambda t, y: lam * y, 0.0, [2.0], h)
        R = 1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24 + z ** 5 / 120 + z ** 6 / 800
        Rs = 1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24 + 10517 / 1228800 * z ** 5 + 1771 / 1638400 * z ** 6
        assert abs(ynew[0] / 2.0 - R) < 4e-15 * max(1, abs(R))
        assert abs((ynew[0] - delta[0]) / 2.0 - Rs) < 4e-15 * max(1, abs(Rs))


def test_stage_times_a_i():
    """Non-autonomous f(t) only: y1 - y0 = h * sum c_i f(t + a_i h) is a 6-node quadrature of degree 4+."""
    for p in range(0, 5):
        ynew, _ = oracle.rkck_step(lambda t, y: np.array([t ** p]), 0.5, [0.0], 0.4)
        exact = ((0.9) ** (p + 1) - 0.5 ** (p + 1)) / (p + 1)
        assert abs(ynew[0] - exact) < 1e-15


def _fixed_steps(step, n_steps, T=1.0):
    y = np.array([1.0])
    h = T / n_steps
    ye = np.array([1.0])
    for i in range(n_steps):
        yn, d = step(lambda t, y: -y * y, i * h, y, h)
        ye = yn - d if i == n_steps - 1 else ye
        y = yn
    return y[0]


def test_measured_order_5_and_4():
    """y' = -y^2, y(0)=1, y = 1/(1+t): global error slope 5 (Eq. 13); local embedded error slope 5 (order 4)."""
    errs = []
    ns = [16, 32, 64, 128]
    for n in ns:
        errs.append(abs(_fixed_steps(oracle.rkck_step, n) - 0.5))
    slopes = [np.log2(errs[i] / errs[i + 1]) for i in range(len(ns) - 1)]
    assert all(4.8 < s < 5.2 for s in slopes), slopes
    # one-step local errors on y' = cos(t) y, y = exp(sin t): 5th-order ~ h^6, embedded 4th-order ~ h^5
    loc5, loc4 = [], []
    t0 = 0.3
    for h in (0.4, 0.2, 0.1, 0.05):
        yn, d = oracle.rkck_step(lambda t, y: np.cos(t) * y, t0, [np.exp(np.sin(t0))], h)
        ex = np.exp(np.sin(t0 + h))
        loc5.append(abs(yn[0] - ex))
        loc4.append(abs(yn[0] - d[0] - ex))
    s5 = [np.log2(loc5[i] / loc5[i + 1]) for i in range(3)]
    s4 = [np.log2(loc4[i] / loc4[i + 1]) for i in range(3)]
    assert all(5.8 < s < 6.3 for s in s5), s5
    assert all(4.8 < s < 5.4 for s in s4), s4


def test_driver_tolerance_proportionality_and_k1_reuse():
    """Global error ~ rtol (slope about 1 over 6 decades); nfe = accepted + 5*(accepted+rejected) (R25)."""
    f = lambda t, y: np.array([y[1], -y[0]])          # harmonic oscillator, y = (cos t, -sin t)
    errs = []
    tols = [1e-4, 1e-6, 1e-8, 1e-10]
    for tol in tols:
        y, status, st = oracle.rkck_generic(f, [1.0, 0.0], 0.0, 10.0, tol, tol * 1e-3)
        assert status == 0
        assert st[0] == st[1] + 5 * (st[1] + st[2])
        errs.append(np.hypot(y[0] - np.cos(10.0), y[1] + np.sin(10.0)))
    slope = np.log10(errs[0] / errs[-1]) / 6.0
    assert 0.8 < slope < 1.25, (errs, slope)
    assert errs[2] < 1e-6


def test_driver_hits_end_exactly_and_first_step_is_global_step():
    """R4/R5: smooth problem, loose tolerance -> a single step of the whole interval, 6 evaluations."""
    y, status, st = oracle.rkck_generic(lambda t, y: -0.01 * y, [1.0], 0.0, 1.0, 1e-8, 1e-12)
    assert status == 0 and list(st[:3]) == [6, 1, 0]
    assert abs(y[0] - np.exp(-0.01)) < 1e-14


def test_driver_nonfinite_rejects_then_fails_cleanly():
    """R6/R7: an RHS that is NaN everywhere ends in status 3 (non-finite) with y untouched."""
    y, status, st = oracle.rkck_generic(lambda t, y: np.array([np.nan]), [1.0], 0.0, 1.0, 1e-8, 1e-12)
    assert status == 3 and y[0] == 1.0 and st[1] == 0
