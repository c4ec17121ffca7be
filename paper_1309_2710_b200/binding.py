"""Thin ctypes binding over the C ABI of include/ckb.h (libckb.so).  Argument marshalling only: every
step of the path (source term, RKCK, RKC, spectral radius, controllers) runs in the CUDA kernels.

PyTorch is used for device memory and streams only.  There is no CPU fallback: if libckb.so is missing
the import of the entry points fails loudly (build it with ``python -m paper_1309_2710_b200.build``).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libckb.so")

OK, EINVAL, ENOMEM, ECUDA, EUNSUPPORTED, ECAPACITY = 0, -1, -2, -3, -4, -5
METHODS = {"rkck": 0, "rkc": 1}
VARIANTS = {"auto": 0, "thread": 1, "warp": 2, "sub8": 3, "sub16": 4, "sub2": 5, "sub4": 6}
ST_OK, ST_MAXSTEPS, ST_UNDERFLOW, ST_NONFINITE, ST_SIGMA = 0, 1, 2, 3, 4

# every symbol include/ckb.h declares
EXPORTS = ("ckb_mech_load", "ckb_mech_free", "ckb_mech_info", "ckb_integrate", "ckb_integrate_host",
           "ckb_rhs", "ckb_fp64_probe", "ckb_mech_pack_stats", "ckb_strerror", "ckb_last_cuda_error",
           "ckb_mech_specialize", "ckb_mech_precompile", "ckb_mech_codegen", "ckb_codegen_log",
           "ckb_integrate_cv", "ckb_integrate_host_cv", "ckb_rhs_cv", "ckb_mech_load2", "ckb_mech_load3",
           "ckb_mech_reserve", "ckb_chemkin_parse", "ckb_chemkin_free", "ckb_chemkin_desc", "ckb_chemkin_species",
           "ckb_chemkin_reaction_origin", "ckb_chemkin_error", "ckb_integrate_static")


class CkbError(RuntimeError):
    def __init__(self, code, where):
        L = lib()
        msg = L.ckb_strerror(code).decode()
        if code == ECUDA:
            msg += ": " + L.ckb_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} ({code})")
        self.code = code


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
    """Load libckb.so and declare the prototypes of include/ckb.h."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build the CUDA library with "
                          "`python -m paper_1309_2710_b200.build` (there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    L.ckb_mech_load.argtypes = [C.POINTER(_Desc), C.POINTER(vp)]
    L.ckb_mech_load.restype = C.c_int
    L.ckb_mech_load2.argtypes = [C.POINTER(_Desc), vp, vp, C.POINTER(vp)]
    L.ckb_mech_load2.restype = C.c_int
    L.ckb_mech_load3.argtypes = [C.POINTER(_Desc), vp, vp, i32, vp, vp, vp, C.POINTER(vp)]
    L.ckb_mech_load3.restype = C.c_int
    L.ckb_mech_free.argtypes = [vp]
    L.ckb_mech_free.restype = None
    L.ckb_mech_reserve.argtypes = [vp, i64]
    L.ckb_mech_reserve.restype = C.c_int
    L.ckb_chemkin_parse.argtypes = [C.c_char_p, C.c_char_p, vp, C.POINTER(vp)]
    L.ckb_chemkin_parse.restype = C.c_int
    L.ckb_chemkin_free.argtypes = [vp]
    L.ckb_chemkin_free.restype = None
    L.ckb_chemkin_desc.argtypes = [vp, C.POINTER(_Desc), C.POINTER(vp), C.POINTER(vp), C.POINTER(i32), C.POINTER(vp),
                                   C.POINTER(vp), C.POINTER(vp)]
    L.ckb_chemkin_desc.restype = C.c_int
    L.ckb_chemkin_species.argtypes = [vp, i32]
    L.ckb_chemkin_species.restype = C.c_char_p
    L.ckb_chemkin_reaction_origin.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(i32)]
    L.ckb_chemkin_reaction_origin.restype = C.c_int
    L.ckb_chemkin_error.argtypes = []
    L.ckb_chemkin_error.restype = C.c_char_p
    L.ckb_mech_info.argtypes = [vp, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32), C.POINTER(dbl)]
    L.ckb_mech_info.restype = C.c_int
    integ = [vp, vp, vp, dbl, i64, i64, dbl, dbl, dbl, dbl, i32, i32, vp, vp, vp]
    L.ckb_integrate.argtypes = integ
    L.ckb_integrate.restype = C.c_int
    L.ckb_integrate_host.argtypes = integ
    L.ckb_integrate_host.restype = C.c_int
    L.ckb_integrate_static.argtypes = integ
    L.ckb_integrate_static.restype = C.c_int
    L.ckb_rhs.argtypes = [vp, vp, vp, dbl, i64, i64, vp, i32, i32, vp]
    L.ckb_rhs.restype = C.c_int
    L.ckb_integrate_cv.argtypes = integ
    L.ckb_integrate_cv.restype = C.c_int
    L.ckb_integrate_host_cv.argtypes = integ
    L.ckb_integrate_host_cv.restype = C.c_int
    L.ckb_rhs_cv.argtypes = L.ckb_rhs.argtypes
    L.ckb_rhs_cv.restype = C.c_int
    L.ckb_fp64_probe.argtypes = [i32, i64, C.POINTER(dbl), vp]
    L.ckb_fp64_probe.restype = C.c_int
    L.ckb_mech_pack_stats.argtypes = [C.POINTER(_Desc), i32, C.POINTER(i32)]
    L.ckb_mech_pack_stats.restype = C.c_int
    L.ckb_mech_specialize.argtypes = [vp]
    L.ckb_mech_specialize.restype = C.c_int
    L.ckb_mech_precompile.argtypes = [C.POINTER(_Desc), C.c_char_p]
    L.ckb_mech_precompile.restype = C.c_int
    L.ckb_mech_codegen.argtypes = [C.POINTER(_Desc), C.c_char_p, i64, C.POINTER(i64)]
    L.ckb_mech_codegen.restype = C.c_int
    L.ckb_codegen_log.argtypes = []
    L.ckb_codegen_log.restype = C.c_char_p
    L.ckb_strerror.argtypes = [C.c_int]
    L.ckb_strerror.restype = C.c_char_p
    L.ckb_last_cuda_error.argtypes = []
    L.ckb_last_cuda_error.restype = C.c_char_p
    _lib = L
    return L


def _check(rc, where):
    if rc != OK:
        raise CkbError(rc, where)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _dev_ptr(t, dtype, where):
    import torch
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"{where}: expected a contiguous CUDA tensor of {dtype}")
    return C.c_void_p(t.data_ptr())


def _make_desc(mech):
    keep = dict(
        mol_weight=_f64(mech.mol_weight), nasa=_f64(mech.nasa), arr_A=_f64(mech.arr_A),
        arr_beta=_f64(mech.arr_beta), arr_E=_f64(mech.arr_E),
        reac_ptr=_i32(mech.reac_ptr), reac_species=_i32(mech.reac_species), reac_nu=_i32(mech.reac_nu),
        prod_ptr=_i32(mech.prod_ptr), prod_species=_i32(mech.prod_species), prod_nu=_i32(mech.prod_nu),
        tb_reaction=_i32(mech.tb_reaction), tb_ptr=_i32(mech.tb_ptr), tb_species=_i32(mech.tb_species),
        tb_eff=_f64(mech.tb_eff))
    d = _Desc()
    d.n_species = int(keep["mol_weight"].shape[0])
    d.n_reactions = int(keep["arr_A"].shape[0])
    d.n_third_body = int(keep["tb_reaction"].shape[0])
    for k, v in keep.items():
        setattr(d, k, v.ctypes.data)
    return d, keep


def pack_stats(mech, lanes=32):
    """ckb_mech_pack_stats (host only, no GPU needed): dict of the packing report for `lanes` lanes per system."""
    d, _keep = _make_desc(mech)
    out = (C.c_int32 * 8)()
    _check(lib().ckb_mech_pack_stats(C.byref(d), int(lanes), out), "ckb_mech_pack_stats")
    names = ("slots", "slot_rounds", "gather_steps", "gather_conflict_replays", "conc_conflict_replays",
             "table_words", "shared_doubles_per_system", "register_slots")
    return dict(zip(names, list(out)))


def codegen(mech) -> str:
    """ckb_mech_codegen (host only): the generated straight-line f(y) of the mechanism as CUDA text."""
    d, _keep = _make_desc(mech)
    need = C.c_int64()
    _check(lib().ckb_mech_codegen(C.byref(d), None, 0, C.byref(need)), "ckb_mech_codegen")
    buf = C.create_string_buffer(need.value)
    _check(lib().ckb_mech_codegen(C.byref(d), buf, need.value, C.byref(need)), "ckb_mech_codegen")
    return buf.value.decode()


def precompile(mech, arch="sm_100a") -> None:
    """ckb_mech_precompile (host only): generate + compile the specialised kernels into the on-disk cache."""
    d, _keep = _make_desc(mech)
    rc = lib().ckb_mech_precompile(C.byref(d), arch.encode())
    if rc != OK:
        raise CkbError(rc, "ckb_mech_precompile: " + lib().ckb_codegen_log().decode()[-2000:])


class ChemkinMechanism:
    """The arrays of ckb_mech_desc / ckb_mech_load3 as numpy attributes (copies), as ckb_chemkin_parse produced them."""


def chemkin_parse(mech_text, thermo_text=None, fit_T=None) -> ChemkinMechanism:
    """ckb_chemkin_parse + ckb_chemkin_desc (host only): read a Chemkin-format mechanism and convert every reversible
    reaction into two irreversible ones (Appendix A).  The result can be given to mech_load()."""
    L = lib()
    h = C.c_void_p()
    T3 = None if fit_T is None else _f64(fit_T)
    rc = L.ckb_chemkin_parse(mech_text.encode(), None if thermo_text is None else thermo_text.encode(),
                             None if T3 is None else C.c_void_p(T3.ctypes.data), C.byref(h))
    if rc != OK:
        raise CkbError(rc, "ckb_chemkin_parse: " + L.ckb_chemkin_error().decode())
    try:
        d = _Desc()
        hi, tm, fr, lo, tr, nfo = C.c_void_p(), C.c_void_p(), C.c_void_p(), C.c_void_p(), C.c_void_p(), C.c_int32()
        _check(L.ckb_chemkin_desc(h, C.byref(d), C.byref(hi), C.byref(tm), C.byref(nfo), C.byref(fr), C.byref(lo), C.byref(tr)),
               "ckb_chemkin_desc")
        K, R, R3, nf = d.n_species, d.n_reactions, d.n_third_body, nfo.value

        def arr(ptr, n, ct, dt):
            if n == 0 or not ptr:
                return np.zeros(0, dtype=dt)
            return np.ctypeslib.as_array(C.cast(ptr, C.POINTER(ct)), shape=(n,)).astype(dt, copy=True)

        m = ChemkinMechanism()
        m.name = "chemkin"
        m.n_species, m.n_reactions = K, R
        m.mol_weight = arr(d.mol_weight, K, C.c_double, np.float64)
        m.nasa = arr(d.nasa, 7 * K, C.c_double, np.float64).reshape(K, 7)
        m.nasa_high = arr(hi.value, 7 * K, C.c_double, np.float64).reshape(K, 7)
        m.T_mid = arr(tm.value, K, C.c_double, np.float64)
        m.arr_A, m.arr_beta, m.arr_E = (arr(p_, R, C.c_double, np.float64) for p_ in (d.arr_A, d.arr_beta, d.arr_E))
        m.reac_ptr = arr(d.reac_ptr, R + 1, C.c_int32, np.int32)
        m.prod_ptr = arr(d.prod_ptr, R + 1, C.c_int32, np.int32)
        m.reac_species = arr(d.reac_species, int(m.reac_ptr[-1]), C.c_int32, np.int32)
        m.reac_nu = arr(d.reac_nu, int(m.reac_ptr[-1]), C.c_int32, np.int32)
        m.prod_species = arr(d.prod_species, int(m.prod_ptr[-1]), C.c_int32, np.int32)
        m.prod_nu = arr(d.prod_nu, int(m.prod_ptr[-1]), C.c_int32, np.int32)
        m.tb_reaction = arr(d.tb_reaction, R3, C.c_int32, np.int32)
        m.tb_ptr = arr(d.tb_ptr, R3 + 1, C.c_int32, np.int32)
        m.tb_species = arr(d.tb_species, int(m.tb_ptr[-1]), C.c_int32, np.int32)
        m.tb_eff = arr(d.tb_eff, int(m.tb_ptr[-1]), C.c_double, np.float64)
        m.fo_reaction = arr(fr.value, nf, C.c_int32, np.int32)
        m.fo_low = arr(lo.value, 3 * nf, C.c_double, np.float64).reshape(nf, 3)
        m.fo_troe = arr(tr.value, 4 * nf, C.c_double, np.float64).reshape(nf, 4)
        m.species_names = [L.ckb_chemkin_species(h, k).decode() for k in range(K)]
        org, rev = C.c_int32(), C.c_int32()
        m.origin, m.is_reverse = np.zeros(R, dtype=np.int32), np.zeros(R, dtype=np.int32)
        for j in range(R):
            _check(L.ckb_chemkin_reaction_origin(h, j, C.byref(org), C.byref(rev)), "ckb_chemkin_reaction_origin")
            m.origin[j], m.is_reverse[j] = org.value, rev.value
        return m
    finally:
        L.ckb_chemkin_free(h)


class Mech:
    """ckb_mech handle.  `mech` is any object that carries the arrays of ckb_mech_desc as attributes."""

    def __init__(self, mech):
        d, keep = _make_desc(mech)      # `keep` holds the arrays the descriptor points at until the load returns
        self._h = C.c_void_p()
        if getattr(mech, "fo_reaction", None) is not None and len(mech.fo_reaction):   # fall-off reactions
            fr, lo, tr = _i32(mech.fo_reaction), _f64(mech.fo_low), _f64(mech.fo_troe)
            if lo.shape != (len(fr), 3) or tr.shape != (len(fr), 4):
                raise ValueError("fo_low must be [n][3] and fo_troe [n][4]")
            hi = tm = None
            if getattr(mech, "nasa_high", None) is not None:
                hi, tm = _f64(mech.nasa_high), _f64(mech.T_mid)
            p_ = lambda a: None if a is None else C.c_void_p(a.ctypes.data)
            _check(lib().ckb_mech_load3(C.byref(d), p_(hi), p_(tm), len(fr), p_(fr), p_(lo), p_(tr), C.byref(self._h)),
                   "ckb_mech_load3")
        elif getattr(mech, "nasa_high", None) is not None:    # two temperature ranges (ckb_mech_load2)
            hi, tm = _f64(mech.nasa_high), _f64(mech.T_mid)
            if hi.shape != (d.n_species, 7) or tm.shape != (d.n_species,):
                raise ValueError("nasa_high must be [K][7] and T_mid [K]")
            _check(lib().ckb_mech_load2(C.byref(d), C.c_void_p(hi.ctypes.data), C.c_void_p(tm.ctypes.data),
                                        C.byref(self._h)), "ckb_mech_load2")
        else:
            _check(lib().ckb_mech_load(C.byref(d), C.byref(self._h)), "ckb_mech_load")
        ks, rs, ns, fl = C.c_int32(), C.c_int32(), C.c_int32(), C.c_double()
        _check(lib().ckb_mech_info(self._h, C.byref(ks), C.byref(rs), C.byref(ns), C.byref(fl)), "ckb_mech_info")
        self.K, self.R, self.n_slots, self.flops_per_rhs = ks.value, rs.value, ns.value, fl.value

    def specialize(self):
        """ckb_mech_specialize: switch thread-per-ODE launches of this handle to mechanism-specialised kernels."""
        rc = lib().ckb_mech_specialize(self._h)
        if rc != OK:
            raise CkbError(rc, "ckb_mech_specialize: " + lib().ckb_codegen_log().decode()[-2000:])
        self.specialized = True
        return self

    def reserve(self, max_batch):
        """ckb_mech_reserve: size the handle's queue-order scratch for batches of up to max_batch systems."""
        _check(lib().ckb_mech_reserve(self._h, int(max_batch)), "ckb_mech_reserve")
        return self

    def close(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.ckb_mech_free(self._h)
            self._h = None

    __del__ = close


def mech_load(mech, specialize=False) -> Mech:
    m = Mech(mech)
    return m.specialize() if specialize else m


def integrate(m: Mech, states, dt, rtol, atol, method, *, N=None, t=0.0, p=None, pressure=None,
              variant="auto", status=None, stats=None, stream=None, cv=False):
    """ckb_integrate: advance states (CUDA float64 tensor [(K+1)][ld], in place) over one global step dt.

    p: uniform pressure (dyn/cm^2) or pressure: CUDA tensor [N].  status: int32 CUDA [N]; stats: int32 CUDA [4][N].
    cv=True calls ckb_integrate_cv: constant volume, p / pressure carry the density in g/cm^3.
    Asynchronous on the current (or given) torch stream.
    """
    import torch
    if states.dim() != 2 or states.shape[0] != m.K + 1:
        raise ValueError("states must be [(K+1)][ld]")
    ld = int(states.shape[1])
    N = ld if N is None else int(N)
    rc = (lib().ckb_integrate_cv if cv else lib().ckb_integrate)(
        m._h, _dev_ptr(states, torch.float64, "states"), _dev_ptr(pressure, torch.float64, "pressure"),
        float(0.0 if p is None else p), N, ld, float(t), float(dt), float(rtol), float(atol),
        int(METHODS.get(method, method)), int(VARIANTS.get(variant, variant)),
        _dev_ptr(status, torch.int32, "status"), _dev_ptr(stats, torch.int32, "stats"), _stream_ptr(stream))
    _check(rc, "ckb_integrate")
    return states


STATIC_MAX_BATCH = 524288
DEFAULT_MAX_BATCH = 1 << 20   # CKB_DEFAULT_MAX_BATCH: what ckb_mech_load reserves for ckb_integrate


def integrate_static(m: Mech, states, dt, rtol, atol, method, *, N=None, t=0.0, p=None, pressure=None,
                     variant="auto", status=None, stats=None, stream=None):
    """ckb_integrate_static: ckb_integrate with its scratch in the library's static device array -- no device allocation on
    the call path; N <= STATIC_MAX_BATCH; calls that overlap on the GPU race on that array."""
    import torch
    if states.dim() != 2 or states.shape[0] != m.K + 1:
        raise ValueError("states must be [(K+1)][ld]")
    ld = int(states.shape[1])
    N = ld if N is None else int(N)
    rc = lib().ckb_integrate_static(
        m._h, _dev_ptr(states, torch.float64, "states"), _dev_ptr(pressure, torch.float64, "pressure"),
        float(0.0 if p is None else p), N, ld, float(t), float(dt), float(rtol), float(atol),
        int(METHODS.get(method, method)), int(VARIANTS.get(variant, variant)),
        _dev_ptr(status, torch.int32, "status"), _dev_ptr(stats, torch.int32, "stats"), _stream_ptr(stream))
    _check(rc, "ckb_integrate_static")
    return states


def integrate_host(m: Mech, states, dt, rtol, atol, method, *, t=0.0, p=None, pressure=None, variant="auto",
                   status=None, stats=None, stream=None, cv=False):
    """ckb_integrate_host (cv=True: ckb_integrate_host_cv): the same call on HOST buffers (numpy float64 [(K+1)][N] C-contiguous, or a pinned
    CPU torch tensor), host<->device copies inside the call; returns after the stream has been synchronised."""
    def hp(a, dtype):
        if a is None:
            return None
        if hasattr(a, "data_ptr"):
            return C.c_void_p(a.data_ptr())
        assert a.dtype == dtype and a.flags["C_CONTIGUOUS"]
        return C.c_void_p(a.ctypes.data)
    n, N = int(states.shape[0]), int(states.shape[1])
    if n != m.K + 1:
        raise ValueError("states must be [(K+1)][N]")
    rc = (lib().ckb_integrate_host_cv if cv else lib().ckb_integrate_host)(
        m._h, hp(states, np.float64), hp(pressure, np.float64), float(0.0 if p is None else p), N, N, float(t),
        float(dt), float(rtol), float(atol), int(METHODS.get(method, method)), int(VARIANTS.get(variant, variant)),
        hp(status, np.int32), hp(stats, np.int32), _stream_ptr(stream))
    _check(rc, "ckb_integrate_host")
    return states


def rhs(m: Mech, states, *, p=None, pressure=None, variant="auto", repeat=1, out=None, N=None, stream=None,
        cv=False):
    """ckb_rhs (cv=True: ckb_rhs_cv, p / pressure carry the density): f(y) for every system; returns dydt
    [(K+1)][ld] (CUDA float64)."""
    import torch
    ld = int(states.shape[1])
    N = ld if N is None else int(N)
    if out is None:
        out = torch.empty_like(states)
    rc = (lib().ckb_rhs_cv if cv else lib().ckb_rhs)(m._h, _dev_ptr(states, torch.float64, "states"), _dev_ptr(pressure, torch.float64, "pressure"),
                       float(0.0 if p is None else p), N, ld, _dev_ptr(out, torch.float64, "out"),
                       int(VARIANTS.get(variant, variant)), int(repeat), _stream_ptr(stream))
    _check(rc, "ckb_rhs")
    return out


def integrate_cv(m: Mech, states, dt, rtol, atol, method, **kw):
    """ckb_integrate_cv: constant-volume closure (R29); p= / pressure= carry the density in g/cm^3."""
    return integrate(m, states, dt, rtol, atol, method, cv=True, **kw)


def integrate_host_cv(m: Mech, states, dt, rtol, atol, method, **kw):
    """ckb_integrate_host_cv."""
    return integrate_host(m, states, dt, rtol, atol, method, cv=True, **kw)


def rhs_cv(m: Mech, states, **kw):
    """ckb_rhs_cv."""
    return rhs(m, states, cv=True, **kw)


def fp64_probe(kind="dfma", iters=1 << 16, stream=None) -> float:
    """ckb_fp64_probe: measured FP64 FLOP/s (kind='dfma') or exp(double)/s (kind='exp') of this device."""
    v = C.c_double()
    _check(lib().ckb_fp64_probe({"dfma": 0, "exp": 1}[kind], int(iters), C.byref(v), _stream_ptr(stream)),
           "ckb_fp64_probe")
    return v.value
