"""Pins for the step-size controllers of the oracle's drivers, read from their step traces.  No GPU.

`ora_rkck_trace` / `ora_rkc_trace` are the generic drivers with one record per step attempt
(t, step size, error measure, accepted, stages, sigma refreshed, sigma).  Everything below is computed in the
test from the traced numbers with the constants of the paper, typed here from PAPER.md:

  RKCK  Eq. 16, Eq. 17 and "increases limited to five, decreases to ten", S = 0.9
  RKC   Eq. 30-32, Eq. 33-35, Eq. 36-38, Eq. 39,
        "estimated every 25 (internal) steps or after a step rejection"

A wrong exponent (1/5 <-> 1/4), a wrong limit, Eq. 34 with its ratios upside down, a missing [0.1, 10] clamp, a wrong
0.1 or square root in Eq. 38 or a refresh count other than 25 each fail one of these (checked on scratch copies of the
oracle while writing them).
"""
import mpmath as mp
import numpy as np

import oracle

mp.mp.dps = 40


def _next_expected(tr, i, t_end, fac):
    """Step size of attempt i+1 given the factor the controller must apply after attempt i, incl. the end clip R5."""
    t_next = tr["t"][i] + (tr["h"][i] if tr["accepted"][i] else 0.0)
    h = tr["h"][i] * fac
    if 1.1 * h >= t_end - t_next:
        h = t_end - t_next
    return h


# ------------------------------------------------------------------------------------------------ RKCK
def _rkck_cases():
    lam = -1000.0
    yield "transient", (lambda t, y: lam * y), [1.0], 1.0, 1e-6, 1e-9
    yield "forced", (lambda t, y: np.array([-50.0 * (y[0] - np.cos(t)), y[0] * np.sin(3 * t)])), [0.0, 1.0], 3.0, 1e-6, 1e-9
    # a jump in f: the steps across it are cut down hard, the ones behind it are far too small and grow at the limit
    yield "jump", (lambda t, y: np.sin(t) - 0.01 * y + (5.0 if t >= 0.3 else 0.0)), [1.0], 2.0, 1e-6, 1e-9
    yield "orbit", (lambda t, y: np.array([y[1], -y[0] * (1 + 20 * np.exp(-30 * (t - 1.3) ** 2))])), [1.0, 0.0], 4.0, 1e-7, 1e-12


def test_rkck_step_factor_follows_eq17_with_both_exponents_and_both_limits():
    seen = dict(acc_free=0, acc_clamp5=0, rej_free=0, rej_clamp10=0)
    for name, f, y0, t_end, rtol, atol in _rkck_cases():
        y, status, st, tr = oracle.rkck_trace(f, y0, 0.0, t_end, rtol, atol)
        assert status == 0
        n = len(tr["t"])
        assert n == st[1] + st[2] and np.sum(tr["accepted"]) == st[1]
        assert tr["h"][0] == t_end                                        # R4: first trial step is the whole interval
        for i in range(n - 1):
            e = tr["err"][i]
            if tr["accepted"][i]:
                assert e <= 1.0
                raw = 0.9 * e ** (-1.0 / 5.0) if e > 0 else np.inf        # Eq. 17, accepted branch, S = 0.9
                fac = min(5.0, raw)                                       # P:144 "increases ... limited to five"
                seen["acc_clamp5" if raw > 5.0 else "acc_free"] += 1
                assert abs(tr["t"][i + 1] - (tr["t"][i] + tr["h"][i])) <= 1e-15 * t_end
            else:
                assert e > 1.0
                raw = 0.9 * e ** (-1.0 / 4.0)                             # Eq. 17, rejected branch
                fac = max(0.1, raw)                                       # P:144 "decreases ... limited to ten"
                seen["rej_clamp10" if raw < 0.1 else "rej_free"] += 1
                assert tr["t"][i + 1] == tr["t"][i]
            expect = _next_expected(tr, i, t_end, fac)
            assert abs(tr["h"][i + 1] / expect - 1.0) < 1e-13, (name, i, tr["h"][i + 1], expect)
        # the last attempt is accepted and ends exactly at t_end (R5)
        assert tr["accepted"][-1] == 1 and abs(tr["t"][-1] + tr["h"][-1] - t_end) <= 2e-16 * t_end
        ratios = tr["h"][1:] / tr["h"][:-1]
        assert np.all(ratios <= 5.0 * (1 + 1e-13)) and np.all(ratios >= 0.1 * (1 - 1e-13))
    assert all(v >= 3 for v in seen.values()), seen


def test_rkck_traced_error_is_eq16_eq17_of_the_pinned_single_step():
    """errmax of every attempt = max_i |Delta_i| / (rtol (|y_i| + |dt f_i|) + atol), with Delta from ora_rkck_step (pinned
    by the closed forms of tests/test_oracle_rkck.py) replayed along the accepted steps of the trace."""
    f = lambda t, y: np.array([-50.0 * (y[0] - np.cos(t)), y[0] * np.sin(3 * t)])
    rtol, atol = 1e-6, 1e-9
    yend, status, st, tr = oracle.rkck_trace(f, [0.0, 1.0], 0.0, 3.0, rtol, atol)
    y = np.array([0.0, 1.0])
    for i in range(len(tr["t"])):
        t, h = tr["t"][i], tr["h"][i]
        ynew, delta = oracle.rkck_step(f, t, y, h)
        d0 = rtol * (np.abs(y) + np.abs(h * f(t, y))) + atol               # Eq. 16 (R2: eps = rtol, eps*delta = atol)
        errmax = np.max(np.abs(delta) / d0)
        assert abs(tr["err"][i] / errmax - 1.0) < 1e-9, (i, tr["err"][i], errmax)
        if tr["accepted"][i]:
            y = ynew
    assert np.max(np.abs(y - yend)) < 1e-13


# ------------------------------------------------------------------------------------------------ RKC
def _kink(t):
    """forcing with a kink in its second derivative at t = 0.7 and a bump: the local error varies from step to step"""
    return np.cos(t) + 0.3 * np.abs(t - 0.7) ** 3 + 0.2 * np.exp(-200.0 * (t - 1.4) ** 2)


def _dkink(t):
    return -np.sin(t) + 0.9 * np.abs(t - 0.7) * (t - 0.7) - 80.0 * (t - 1.4) * np.exp(-200.0 * (t - 1.4) ** 2)


def _rkc_cases():
    lam = -100.0
    yield "kink", (lambda t, y: lam * (y - _kink(t)) + _dkink(t)), [1.0], 2.0, 1e-5, 1e-8
    A = np.array([[-2000.0, 1500.0], [3.0, -4.0]])
    yield "stiff2", (lambda t, y: A @ y + np.array([np.sin(40 * t), 1.0])), [1.0, 0.5], 1.5, 1e-4, 1e-7
    yield "vdp", (lambda t, y: np.array([y[1], 30.0 * (1 - y[0] ** 2) * y[1] - y[0]])), [2.0, 0.0], 1.2, 1e-5, 1e-8


def test_rkc_step_factor_follows_eq33_35_with_memory_and_clamp():
    seen = dict(memory=0, memory_differs=0, no_memory=0, rejected=0, clamp_lo=0, clamp_hi=0)
    for name, f, y0, t_end, rtol, atol in _rkc_cases():
        y, status, st, tr = oracle.rkc_trace(f, y0, 0.0, t_end, rtol, atol)
        assert status in (0, 4)
        n = len(tr["t"])
        assert n == st[1] + st[2]
        for i in range(n - 1):
            e = tr["err"][i]
            if tr["accepted"][i]:
                assert e <= 1.0
                prev_ok = i >= 1 and tr["accepted"][i - 1] == 1                  # R13: memory only after an accepted step
                if prev_ok:
                    e_old, h_old = tr["err"][i - 1], tr["h"][i - 1]
                    # Eq. 34 with p = 2: 0.8 (||D_n||^(1/3) / ||D_n+1||^(1/3)) (dt_n / dt_n-1) / ||D_n+1||^(1/3)
                    raw = 0.8 * (e_old ** (1 / 3) / e ** (1 / 3)) * (tr["h"][i] / h_old) / e ** (1 / 3)
                    seen["memory"] += 1
                    if abs(raw / (0.8 / e ** (1 / 3)) - 1) > 0.05:
                        seen["memory_differs"] += 1
                else:
                    raw = 0.8 / e ** (1 / 3)
                    seen["no_memory"] += 1
            else:
                assert e > 1.0
                raw = 0.8 / e ** (1 / 3)                                         # Eq. 35
                seen["rejected"] += 1
            fac = min(10.0, max(0.1, raw))                                       # Eq. 33
            seen["clamp_lo"] += raw < 0.1
            seen["clamp_hi"] += raw > 10.0
            expect = _next_expected(tr, i, t_end, fac)
            if tr["s"][i + 1] == 0:
                continue
            assert abs(tr["h"][i + 1] / expect - 1.0) < 1e-12, (name, i, tr["h"][i + 1], expect, raw)
        ratios = tr["h"][1:] / tr["h"][:-1]
        assert np.all(ratios <= 10.0 * (1 + 1e-12))
        assert tr["accepted"][-1] == 1 and abs(tr["t"][-1] + tr["h"][-1] - t_end) <= 2e-16 * t_end
    assert seen["memory"] > 50 and seen["memory_differs"] > 20 and seen["no_memory"] >= 3 and seen["rejected"] >= 3, seen
    assert seen["clamp_lo"] >= 1 and seen["clamp_hi"] >= 1, seen


def test_rkc_first_step_is_eq36_38_by_hand():
    """dt_0 = 1/sigma (Eq. 36), Delta_0 = dt_0 (f(t0 + dt_0, y0 + dt_0 f0) - f0) (Eq. 37), dt_1 = 0.1 dt_0 / sqrt(||Delta_0||)
    (Eq. 38) with the norm of Eq. 31 and the weights atol + rtol |y_0| (R14), evaluated here with numpy."""
    A = np.array([[-2000.0, 1500.0], [3.0, -4.0]])
    f = lambda t, y: A @ y + np.array([np.sin(40 * t), 1.0])
    y0 = np.array([1.0, 0.5])
    rtol, atol = 1e-4, 1e-7
    _, status, st, tr = oracle.rkc_trace(f, y0, 0.0, 1.5, rtol, atol)
    sigma = tr["sigma"][0]
    rho = np.max(np.abs(np.linalg.eigvals(A)))
    assert 1.2 * 0.98 < sigma / rho < 1.2 * 1.001                               # R18 on a linear problem
    dt0 = 1.0 / sigma
    f0 = f(0.0, y0)
    D0 = dt0 * (f(dt0, y0 + dt0 * f0) - f0)
    est = np.sqrt(np.mean((D0 / (atol + rtol * np.abs(y0))) ** 2))
    assert abs(tr["est0"][0] / est - 1) < 1e-12
    assert abs(tr["h"][0] / (0.1 * dt0 / np.sqrt(est)) - 1) < 1e-12
    assert tr["sigma_refreshed"][0] == 1


def test_rkc_sigma_refresh_every_25_accepted_steps_and_after_a_rejection_when_stale():
    refreshes_by_count = refreshes_after_reject = fresh_rejects = 0
    for name, f, y0, t_end, rtol, atol in _rkc_cases():
        _, status, st, tr = oracle.rkc_trace(f, y0, 0.0, t_end, rtol, atol)
        since, fresh = 0, True
        for i in range(len(tr["t"])):
            must = False
            if i > 0:
                if tr["accepted"][i - 1]:
                    since += 1
                    fresh = False
                    must = since >= 25                                           # P:233 "every 25 (internal) steps"
                else:
                    must = (since >= 25) or (not fresh)                          # P:233 "or after a step rejection"; R16
                    fresh_rejects += fresh
            got = bool(tr["sigma_refreshed"][i]) if i > 0 else False
            assert got == must, (name, i, since, fresh)
            if got:
                refreshes_by_count += since >= 25
                refreshes_after_reject += since < 25
                since, fresh = 0, True
            if i > 0 and not got:
                assert tr["sigma"][i] == tr["sigma"][i - 1]
    assert refreshes_by_count >= 5 and refreshes_after_reject >= 3, (refreshes_by_count, refreshes_after_reject)


def test_rkc_stage_count_is_eq39_truncated_and_inside_the_stability_interval():
    lam = np.array([-1.0, -50.0, -2.0e4])
    cases = list(_rkc_cases()) + [("decay", (lambda t, y: lam * y), [1.0, 1.0, 1.0], 1.0, 1e-4, 1e-10)]
    s_seen = set()
    for name, f, y0, t_end, rtol, atol in cases:
        _, status, st, tr = oracle.rkc_trace(f, y0, 0.0, t_end, rtol, atol)
        s = tr["s"].astype(int)
        expect = np.maximum(2, 1 + np.floor(np.sqrt(1 + 1.54 * tr["h"] * tr["sigma"])).astype(int))   # Eq. 39, R12
        assert np.array_equal(s, expect)
        assert st[3] == s.max()
        s_seen |= set(s.tolist())
        for sv in np.unique(s):
            co = oracle.rkc_coeffs(int(sv))
            beta = (1 + co["w0"]) / co["w1"]
            sel = s == sv
            assert np.all(tr["h"][sel] * tr["sigma"][sel] <= beta)               # SURVEY C7 "Eq. 39 + truncation"
    assert len(s_seen) >= 8 and max(s_seen) >= 20, s_seen


def _P(s, z):
    """stability polynomial a_s + b_s T_s(w0 + w1 z) through the cosh/acosh closed forms (mpmath), not the recurrences"""
    w0 = 1 + mp.mpf(2) / 13 / (s * s)
    th = mp.acosh(w0)
    dT = lambda j: j * mp.sinh(j * th) / mp.sinh(th)
    d2T = lambda j: (j * j * mp.cosh(j * th) - w0 * dT(j)) / (w0 * w0 - 1)
    w1 = dT(s) / d2T(s)
    b = d2T(s) / dT(s) ** 2
    a = 1 - b * mp.cosh(s * th)
    x = w0 + w1 * z
    T = mp.cos(s * mp.acos(x)) if abs(x) <= 1 else mp.cosh(s * mp.acosh(x))
    return a + b * T


def test_rkc_traced_error_is_eq30_32_closed_form_on_a_linear_problem():
    """y' = lambda y, atol = 0: ||err|| = |0.8 (1 - P) + 0.4 z (1 + P)| / (rtol max(1, |P|)), P = P_s(z), z = dt lambda,
    independent of y_n.  Two identical decoupled components give the same value (the 1/sqrt(N) of Eq. 31)."""
    lam, rtol = -300.0, 1e-4
    for ncomp in (1, 2):
        _, status, st, tr = oracle.rkc_trace(lambda t, y: lam * y, [1.0] * ncomp, 0.0, 0.5, rtol, 0.0)
        assert status == 0 and len(tr["t"]) > 20
        for i in range(len(tr["t"])):
            z = mp.mpf(tr["h"][i]) * lam
            P = _P(int(tr["s"][i]), z)
            expect = abs(mp.mpf("0.8") * (1 - P) + mp.mpf("0.4") * z * (1 + P)) / (rtol * max(1, abs(P)))
            # Eq. 30 cancels to O(z^3): round-off of its terms is u |z| / rtol in absolute terms
            assert abs(tr["err"][i] - float(expect)) < 1e-6 * float(expect) + 1e-10, (ncomp, i, tr["err"][i], float(expect))
