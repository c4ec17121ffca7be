"""The C-ABI library builds, loads and exports every symbol include/ckb.h declares; argument checks that
need no GPU.  (No compute calls here: those are the -m gpu parity tests.)"""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1309_2710_b200 import binding, build, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    build.build()
    return binding.lib()


def test_header_symbols_exported(L):
    hdr = open(os.path.join(ROOT, "include", "ckb.h")).read()
    declared = set(re.findall(r"\b(ckb_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert getattr(L, name) is not None


def test_strerror(L):
    assert L.ckb_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4):
        assert len(L.ckb_strerror(code)) > 3
    assert b"unknown" in L.ckb_strerror(-99)


def test_instantiation_list_consistent():
    inst = build.instantiations()
    assert (1, 10) in inst and (1, 14) in inst and (32, 2) in inst and (32, 4) in inst
    assert {l for l, _ in inst} == {1, 2, 4, 8, 16, 32}             # one packing per lanes-per-system value


def _load(mech):
    d = binding._Desc()
    keep = {}
    for k in ("mol_weight", "nasa", "arr_A", "arr_beta", "arr_E", "tb_eff"):
        keep[k] = np.ascontiguousarray(getattr(mech, k), dtype=np.float64)
    for k in ("reac_ptr", "reac_species", "reac_nu", "prod_ptr", "prod_species", "prod_nu", "tb_reaction",
              "tb_ptr", "tb_species"):
        keep[k] = np.ascontiguousarray(getattr(mech, k), dtype=np.int32)
    d.n_species, d.n_reactions, d.n_third_body = len(keep["mol_weight"]), len(keep["arr_A"]), len(keep["tb_reaction"])
    for k, v in keep.items():
        setattr(d, k, v.ctypes.data)
    h = C.c_void_p()
    rc = binding.lib().ckb_mech_load(C.byref(d), C.byref(h))
    return rc, h, keep


def test_mech_load_rejects_bad_input(L):
    """Validation happens before any CUDA call, so these return codes are the same with or without a GPU."""
    assert L.ckb_mech_load(None, None) == binding.EINVAL
    m = synth.toy_mechanism(2, [({0: 1}, {1: 1}, 1.0, 0.0, 0.0)])
    m.reac_species = np.array([5], dtype=np.int32)             # species index out of range
    assert _load(m)[0] == binding.EINVAL
    m = synth.toy_mechanism(2, [({0: 1}, {1: 1}, -1.0, 0.0, 0.0)])   # negative A
    assert _load(m)[0] == binding.EINVAL
    m = synth.toy_mechanism(2, [({0: 4}, {1: 4}, 1.0, 0.0, 0.0)])    # 4 molecules on a side
    assert _load(m)[0] == binding.EUNSUPPORTED
    m = synth.toy_mechanism(2, [({0: 1}, {1: 1}, 1.0, 0.0, 0.0)], W=[1.0, -2.0])
    assert _load(m)[0] == binding.EINVAL
    m = synth.toy_mechanism(2, [({0: 1}, {1: 1}, 1.0, 0.0, 0.0)], third_body={3: {0: 2.0}})  # bad reaction index
    assert _load(m)[0] == binding.EINVAL


def test_integrate_argument_errors_without_handle(L):
    assert L.ckb_integrate(None, None, None, 1e6, 0, 0, 0.0, 1e-6, 1e-8, 1e-12, 0, 0, None, None, None) == binding.EINVAL
    assert L.ckb_rhs(None, None, None, 1e6, 0, 0, None, 0, 1, None) == binding.EINVAL
    v = C.c_double()
    assert L.ckb_fp64_probe(7, 10, C.byref(v), None) == binding.EINVAL


@pytest.mark.parametrize("cfg", [0, 2, 3, 4])
def test_packing_report(cfg, L):
    """Host-only packing (ckb_mech_pack_stats): forward/reverse pairs are fused, the gather schedule of the
    warp-per-ODE packing is as short as its longest (split) row with few shared-memory bank conflicts left, thread-per-ODE
    tables fit the parameter block."""
    mech = synth.make_mechanism(cfg)
    spec = synth.CONFIGS[cfg]
    warp = binding.pack_stats(mech, 32)
    assert warp["slots"] == spec.R // 2                       # every synthetic reaction has its reverse
    assert warp["slot_rounds"] == -(-warp["slots"] // 32)
    assert warp["gather_conflict_replays"] <= 0.5 * warp["gather_steps"]   # least-used-bank schedule: < 1 replay per 2 steps
    assert warp["register_slots"] == -(-(spec.K + 1) // 32) or warp["register_slots"] in (1, 2, 4)
    nnz = sum(len(set(mech.reac_species[mech.reac_ptr[j]:mech.reac_ptr[j + 1]]) |
                  set(mech.prod_species[mech.prod_ptr[j]:mech.prod_ptr[j + 1]])) for j in range(0, spec.R, 2))
    assert warp["gather_steps"] * 32 >= nnz                   # every entry is scheduled
    assert warp["gather_steps"] <= 2.5 * nnz / 32 + 8         # and the padding stays bounded
    if spec.K + 1 <= 16:
        thr = binding.pack_stats(mech, 1)
        assert thr["table_words"] <= 3072 and thr["register_slots"] >= spec.K + 1
        assert thr["gather_steps"] == nnz                     # thread-per-ODE walks the rows as they are
    else:
        with pytest.raises(binding.CkbError):
            binding.pack_stats(mech, 1)
    for lanes in (8, 16):
        st = binding.pack_stats(mech, lanes)
        assert st["slots"] == warp["slots"] and st["register_slots"] * lanes >= spec.K + 1
    for lanes in (2, 4):                                      # few lanes per system: small mechanisms only
        if spec.K + 1 <= 16:
            st = binding.pack_stats(mech, lanes)
            assert st["slots"] == warp["slots"] and st["register_slots"] * lanes >= spec.K + 1
        else:
            with pytest.raises(binding.CkbError):
                binding.pack_stats(mech, lanes)


def test_unpaired_and_duplicate_reactions_pack(L):
    """An irreversible reaction without reverse keeps its own slot; duplicates of the same pair are kept apart."""
    m = synth.toy_mechanism(3, [({0: 1}, {1: 1}, 1.0, 0.0, 0.0), ({1: 1}, {0: 1}, 2.0, 0.0, 0.0),
                                ({0: 1}, {1: 1}, 3.0, 0.0, 0.0), ({1: 2}, {2: 1}, 4.0, 0.0, 0.0)])
    assert binding.pack_stats(m, 32)["slots"] == 3
    assert binding.pack_stats(m, 1)["slots"] == 3


def test_product_path_does_not_import_oracle():
    """The binding, the generator and bench's product arm never touch oracle/ (no CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_1309_2710_b200")
    for fn in os.listdir(pkg):
        if fn.endswith(".py"):
            src = open(os.path.join(pkg, fn)).read()
            assert not re.search(r"^\s*(import|from)\s+oracle", src, re.M), fn
    for fn in os.listdir(os.path.join(pkg, "csrc")):
        src = open(os.path.join(pkg, "csrc", fn)).read()
        assert not re.search(r"#include[^\n]*oracle|ora_[a-z]+\s*\(|libckoracle", src), fn


def test_codegen_text(L):
    """ckb_mech_codegen (host only): the straight-line f(y) of a mechanism -- one exp per irreversible reaction
    with A > 0, every species' thermodynamic polynomials, no table reads; too many unknowns are refused."""
    mech = synth.make_mechanism(1)
    src = binding.codegen(mech)
    assert src.count("ckb_exp(") == mech.n_reactions
    assert src.count("double cp =") == mech.n_species and src.count("double h =") == mech.n_species
    assert "f[0][0] =" in src and "tab" not in src and "sR" not in src
    n_sets = len({tuple(sorted((int(mech.tb_species[e]), float(mech.tb_eff[e]))
                               for e in range(mech.tb_ptr[r], mech.tb_ptr[r + 1])))
                  for r in range(len(mech.tb_reaction))})
    assert src.count("= ctot;") == n_sets + 0
    toy = synth.toy_mechanism(2, [({0: 2}, {1: 1}, 5.0, 0.0, 300.0), ({1: 1}, {0: 2}, 0.0, 0.0, 0.0)])
    s2 = binding.codegen(toy)
    assert s2.count("ckb_exp(") == 1 and "fma(-0x1p+1, q, om" in s2      # A = 0: no rate; nu' = 2 on the reactant
    assert "lnT, " not in s2                                             # beta = 0: the term is not emitted
    toy = synth.toy_mechanism(2, [({0: 1}, {1: 1}, 5.0, 0.0, 0.0)])
    s3 = binding.codegen(toy)
    assert "ckb_exp(" not in s3 and "double rf = 0x1.4p+2;" in s3        # no temperature dependence: a literal
    with pytest.raises(binding.CkbError):
        binding.codegen(synth.make_mechanism(3))


def test_precompile_fills_cache(L, tmp_path, monkeypatch):
    """ckb_mech_precompile (host only): NVRTC compiles the generated kernels for sm_100a without a GPU and the
    second call is served from the on-disk cache."""
    import ctypes.util
    import time
    if not (ctypes.util.find_library("nvrtc") or os.path.exists("/usr/local/cuda/lib64/libnvrtc.so.12")):
        pytest.skip("NVRTC not installed")
    monkeypatch.setenv("CKB_JIT_CACHE", str(tmp_path / "jit"))
    mech = synth.make_mechanism(0)
    t0 = time.time()
    binding.precompile(mech)
    t1 = time.time()
    files = list((tmp_path / "jit").iterdir())
    assert len(files) == 1 and files[0].stat().st_size > 10000
    binding.precompile(mech)
    assert time.time() - t1 < 0.5 * (t1 - t0) + 0.05
    assert len(list((tmp_path / "jit").iterdir())) == 1


def test_mech_load2_rejects_bad_input(L):
    """ckb_mech_load2 validates the second temperature range before any CUDA call (same codes with or without a GPU)."""
    mech = synth.with_two_range_thermo(synth.make_mechanism(0), synth.CONFIGS[0].T_range)
    d, keep = binding._make_desc(mech)
    h = C.c_void_p()
    hi = np.ascontiguousarray(mech.nasa_high)
    tm = np.ascontiguousarray(mech.T_mid)
    vp = lambda a: C.c_void_p(a.ctypes.data)
    assert L.ckb_mech_load2(C.byref(d), vp(hi), None, C.byref(h)) == binding.EINVAL      # one array without the other
    assert L.ckb_mech_load2(C.byref(d), None, vp(tm), C.byref(h)) == binding.EINVAL
    bad = tm.copy()
    bad[2] = np.inf
    assert L.ckb_mech_load2(C.byref(d), vp(hi), vp(bad), C.byref(h)) == binding.EINVAL
    bad_hi = hi.copy()
    bad_hi[1, 3] = np.nan
    assert L.ckb_mech_load2(C.byref(d), vp(bad_hi), vp(tm), C.byref(h)) == binding.EINVAL
    assert L.ckb_mech_load2(None, vp(hi), vp(tm), C.byref(h)) == binding.EINVAL
