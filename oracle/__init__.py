"""ctypes access to the CPU oracle (oracle/ckoracle.c).  TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this
package.  It imports nothing from the CUDA path (paper_1309_2710_b200.binding / csrc); mechanisms are
passed in as any object that carries the arrays of ``ora_mech_desc`` as numpy attributes.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ckoracle.c")
_LIB = os.path.join(_HERE, "libckoracle.so")
CFLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall"]

RHS_FN = C.CFUNCTYPE(None, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_void_p)


def build(force: bool = False) -> str:
    """Compile ckoracle.c -> libckoracle.so with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.run(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


class _Desc(C.Structure):
    _fields_ = [
        ("n_species", C.c_int32), ("n_reactions", C.c_int32),
        ("mol_weight", C.c_void_p), ("nasa", C.c_void_p), ("arr_A", C.c_void_p),
        ("arr_beta", C.c_void_p), ("arr_E", C.c_void_p),
        ("reac_ptr", C.c_void_p), ("reac_species", C.c_void_p), ("reac_nu", C.c_void_p),
        ("prod_ptr", C.c_void_p), ("prod_species", C.c_void_p), ("prod_nu", C.c_void_p),
        ("n_third_body", C.c_int32),
        ("tb_reaction", C.c_void_p), ("tb_ptr", C.c_void_p), ("tb_species", C.c_void_p),
        ("tb_eff", C.c_void_p),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        ip = C.POINTER(C.c_int32)
        L.ora_mech_load.argtypes = [C.POINTER(_Desc), C.POINTER(C.c_void_p)]
        L.ora_mech_load.restype = C.c_int
        L.ora_mech_free.argtypes = [C.c_void_p]
        L.ora_mech_free.restype = None
        L.ora_rhs.argtypes = [C.c_void_p, dp, C.c_double, dp]
        L.ora_rhs.restype = None
        L.ora_integrate.argtypes = [C.c_void_p, dp, dp, C.c_double, C.c_int64, C.c_int64, C.c_double,
                                    C.c_double, C.c_double, C.c_double, C.c_int32, ip, ip, C.c_int32]
        L.ora_integrate.restype = C.c_int
        L.ora_mech_set_thermo2.argtypes = [C.c_void_p, dp, dp]
        L.ora_mech_set_thermo2.restype = C.c_int
        L.ora_mech_set_falloff.argtypes = [C.c_void_p, C.c_int32, ip, dp, dp]
        L.ora_mech_set_falloff.restype = C.c_int
        L.ora_rhs_cv.argtypes = L.ora_rhs.argtypes
        L.ora_rhs_cv.restype = None
        L.ora_integrate_cv.argtypes = L.ora_integrate.argtypes
        L.ora_integrate_cv.restype = C.c_int
        L.ora_rkck_tableau.argtypes = [dp]
        L.ora_rkck_tableau.restype = None
        L.ora_rkck_step.argtypes = [RHS_FN, C.c_void_p, C.c_int, C.c_double, dp, C.c_double, dp, dp]
        L.ora_rkck_step.restype = None
        L.ora_rkck_generic.argtypes = [RHS_FN, C.c_void_p, C.c_int, dp, C.c_double, C.c_double,
                                       C.c_double, C.c_double, ip]
        L.ora_rkck_generic.restype = C.c_int
        L.ora_rkc_generic.argtypes = L.ora_rkck_generic.argtypes
        L.ora_rkc_generic.restype = C.c_int
        L.ora_rkck_trace.argtypes = L.ora_rkck_generic.argtypes + [dp, C.c_int64, C.POINTER(C.c_int64)]
        L.ora_rkck_trace.restype = C.c_int
        L.ora_rkc_trace.argtypes = L.ora_rkck_trace.argtypes
        L.ora_rkc_trace.restype = C.c_int
        L.ora_rkc_coeffs.argtypes = [C.c_int, dp, dp, dp, dp, dp, dp, dp, dp, dp]
        L.ora_rkc_coeffs.restype = C.c_int
        L.ora_rkc_step.argtypes = [RHS_FN, C.c_void_p, C.c_int, C.c_double, dp, C.c_double, C.c_int, dp, dp]
        L.ora_rkc_step.restype = None
        L.ora_spectral_radius.argtypes = [RHS_FN, C.c_void_p, C.c_int, C.c_double, dp, dp, C.c_int, ip, ip]
        L.ora_spectral_radius.restype = C.c_double
        L.ora_fit_reverse.argtypes = [dp, dp, dp]
        L.ora_fit_reverse.restype = None
        L.ora_equilibrium_constant.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.ora_equilibrium_constant.restype = C.c_double
        L.ora_reverse_parameters.argtypes = [C.c_void_p, C.c_int, dp, dp]
        L.ora_reverse_parameters.restype = None
        L.ora_num_threads.argtypes = []
        L.ora_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def wrap_rhs(fn, n):
    """Python f(t, y) -> dydt as a C callback for the generic drivers."""
    def cb(t, yp, dp, _ctx):
        y = np.ctypeslib.as_array(yp, shape=(n,))
        out = np.ctypeslib.as_array(dp, shape=(n,))
        out[:] = fn(t, y)
    return RHS_FN(cb)


class OracleMech:
    """ora_mech handle; `mech` is any object with the ora_mech_desc arrays as attributes."""

    def __init__(self, mech):
        self.K = int(len(mech.mol_weight))
        self.R = int(len(mech.arr_A))
        keep = dict(
            mol_weight=_f64(mech.mol_weight), nasa=_f64(mech.nasa), arr_A=_f64(mech.arr_A),
            arr_beta=_f64(mech.arr_beta), arr_E=_f64(mech.arr_E),
            reac_ptr=_i32(mech.reac_ptr), reac_species=_i32(mech.reac_species), reac_nu=_i32(mech.reac_nu),
            prod_ptr=_i32(mech.prod_ptr), prod_species=_i32(mech.prod_species), prod_nu=_i32(mech.prod_nu),
            tb_reaction=_i32(mech.tb_reaction), tb_ptr=_i32(mech.tb_ptr), tb_species=_i32(mech.tb_species),
            tb_eff=_f64(mech.tb_eff))
        d = _Desc()
        d.n_species, d.n_reactions, d.n_third_body = self.K, self.R, int(len(keep["tb_reaction"]))
        for k, v in keep.items():
            setattr(d, k, v.ctypes.data)
        h = C.c_void_p()
        rc = lib().ora_mech_load(C.byref(d), C.byref(h))
        if rc != 0:
            raise ValueError(f"ora_mech_load failed: {rc}")
        self._h = h
        # optional second temperature range of the NASA fits (reading R30)
        if getattr(mech, "nasa_high", None) is not None:
            hi, tm = _f64(mech.nasa_high), _f64(mech.T_mid)
            assert hi.shape == (self.K, 7) and tm.shape == (self.K,)
            if lib().ora_mech_set_thermo2(self._h, _dp(hi), _dp(tm)) != 0:
                raise ValueError("ora_mech_set_thermo2 failed")

        # optional fall-off reactions (reading R31): fo_reaction [n], fo_low [n][3], fo_troe [n][4]
        if getattr(mech, "fo_reaction", None) is not None and len(mech.fo_reaction):
            fr, lo, tr = _i32(mech.fo_reaction), _f64(mech.fo_low), _f64(mech.fo_troe)
            assert lo.shape == (len(fr), 3) and tr.shape == (len(fr), 4)
            if lib().ora_mech_set_falloff(self._h, len(fr), _ip(fr), _dp(lo), _dp(tr)) != 0:
                raise ValueError("ora_mech_set_falloff failed")

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.ora_mech_free(self._h)
            self._h = None

    def rhs(self, y, p, cv=False):
        """f(y) at constant pressure p (dyn/cm^2), or with cv=True at constant volume, p = density (g/cm^3)."""
        y = _f64(y)
        out = np.empty_like(y)
        (lib().ora_rhs_cv if cv else lib().ora_rhs)(self._h, _dp(y), float(p), _dp(out))
        return out

    def equilibrium_constant(self, j, T):
        """K_c of reaction j at T (Chemkin form, reading R32)."""
        return lib().ora_equilibrium_constant(self._h, int(j), float(T))

    def reverse_parameters(self, j, T3):
        """Appendix A: (A_r, beta_r, E_r [cal/mol]) of the reverse of reaction j from k_f / K_c at the three temperatures."""
        T3, out = _f64(T3), np.zeros(3)
        lib().ora_reverse_parameters(self._h, int(j), _dp(T3), _dp(out))
        return out

    def integrate(self, states, p, dt, rtol, atol, method, t=0.0, nthreads=0, pressure=None, cv=False):
        """states: [(K+1)][N] SoA (copied).  Returns (new_states, status[N], stats[4][N]).
        cv=True: constant volume, p / pressure carry the density in g/cm^3 (reading R29)."""
        method = {"rkck": 0, "rkc": 1}.get(method, method)
        st = np.array(states, dtype=np.float64, order="C", copy=True)
        n, N = st.shape
        assert n == self.K + 1
        status = np.zeros(N, dtype=np.int32)
        stats = np.zeros((4, N), dtype=np.int32)
        pr = None if pressure is None else _f64(pressure)
        fn = lib().ora_integrate_cv if cv else lib().ora_integrate
        rc = fn(self._h, _dp(st), None if pr is None else _dp(pr), float(p), N, N,
                                 float(t), float(dt), float(rtol), float(atol), int(method),
                                 _ip(status), _ip(stats), int(nthreads))
        if rc != 0:
            raise ValueError(f"ora_integrate failed: {rc}")
        return st, status, stats


def rkck_tableau():
    out = np.zeros(48)
    lib().ora_rkck_tableau(_dp(out))
    return out[:6], out[6:36].reshape(6, 5), out[36:42], out[42:48]


def rkck_step(fn, t, y, h):
    y = _f64(y)
    n = len(y)
    ynew, delta = np.empty(n), np.empty(n)
    lib().ora_rkck_step(wrap_rhs(fn, n), None, n, float(t), _dp(y), float(h), _dp(ynew), _dp(delta))
    return ynew, delta


def rkc_step(fn, t, y, h, s, want_stages=False):
    y = _f64(y)
    n = len(y)
    ynew = np.empty(n)
    stages = np.empty((s, n)) if want_stages else None
    lib().ora_rkc_step(wrap_rhs(fn, n), None, n, float(t), _dp(y), float(h), int(s), _dp(ynew),
                       _dp(stages) if want_stages else None)
    return (ynew, stages) if want_stages else ynew


def rkc_coeffs(s):
    arrs = [np.zeros(s + 1) for _ in range(7)]
    w0, w1 = C.c_double(), C.c_double()
    rc = lib().ora_rkc_coeffs(int(s), C.byref(w0), C.byref(w1), *[_dp(a) for a in arrs])
    if rc != 0:
        raise ValueError("s must be >= 2")
    mu, nu, mut, gamt, c, a, b = arrs
    return dict(w0=w0.value, w1=w1.value, mu=mu, nu=nu, mut=mut, gamt=gamt, c=c, a=a, b=b)


def _generic(entry, fn, y, t0, t1, rtol, atol):
    y = np.array(y, dtype=np.float64, copy=True)
    n = len(y)
    stats = np.zeros(4, dtype=np.int32)
    status = entry(wrap_rhs(fn, n), None, n, _dp(y), float(t0), float(t1), float(rtol), float(atol), _ip(stats))
    return y, int(status), stats


def rkck_generic(fn, y, t0, t1, rtol, atol):
    return _generic(lib().ora_rkck_generic, fn, y, t0, t1, rtol, atol)


def rkc_generic(fn, y, t0, t1, rtol, atol):
    return _generic(lib().ora_rkc_generic, fn, y, t0, t1, rtol, atol)


TRACE_COLS = ("t", "h", "err", "accepted", "s", "sigma_refreshed", "sigma", "est0")


def _trace(entry, fn, y, t0, t1, rtol, atol, cap):
    y = np.array(y, dtype=np.float64, copy=True)
    n = len(y)
    stats = np.zeros(4, dtype=np.int32)
    rows = np.zeros((cap, len(TRACE_COLS)))
    nrows = C.c_int64()
    status = entry(wrap_rhs(fn, n), None, n, _dp(y), float(t0), float(t1), float(rtol), float(atol), _ip(stats),
                   _dp(rows), cap, C.byref(nrows))
    assert nrows.value <= cap, "trace buffer too small"
    tr = rows[: nrows.value]
    return y, int(status), stats, {k: tr[:, i] for i, k in enumerate(TRACE_COLS)}


def rkck_trace(fn, y, t0, t1, rtol, atol, cap=100000):
    """ora_rkck_generic with its step trace: one entry per attempt (t, h, errmax, accepted, ...)."""
    return _trace(lib().ora_rkck_trace, fn, y, t0, t1, rtol, atol, cap)


def rkc_trace(fn, y, t0, t1, rtol, atol, cap=100000):
    """ora_rkc_generic with its step trace: one entry per attempt (t, h, err, accepted, s, sigma_refreshed, sigma, est0)."""
    return _trace(lib().ora_rkc_trace, fn, y, t0, t1, rtol, atol, cap)


def spectral_radius(fn, t, y, v=None):
    y = _f64(y)
    n = len(y)
    have_v = v is not None
    vv = np.array(v, dtype=np.float64, copy=True) if have_v else np.zeros(n)
    nfe, flag = C.c_int32(), C.c_int32()
    s = lib().ora_spectral_radius(wrap_rhs(fn, n), None, n, float(t), _dp(y), _dp(vv), int(have_v),
                                  C.byref(nfe), C.byref(flag))
    return s, vv, nfe.value, flag.value


def fit_reverse(T3, kr3):
    """Eq. A.10-A.12: (A_r, beta_r, T_ar) through three (T, k_r) points."""
    T3, kr3, out = _f64(T3), _f64(kr3), np.zeros(3)
    lib().ora_fit_reverse(_dp(T3), _dp(kr3), _dp(out))
    return out


def num_threads():
    return lib().ora_num_threads()
