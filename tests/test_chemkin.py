"""Chemkin-format reader + Appendix-A converter of the product (csrc/ckb_chemkin.cu; P:84, P:243,
P:459-528).  Host-side: everything but the last test runs without a GPU.

The fixture tests/golden/synthetic_hon.inp is synthetic (tests/golden/make_chemkin_fixture.py wrote it together with
synthetic_hon.json, the arrays a reader must get out of it).  The reverse parameters the product fits are compared with
the oracle's own Appendix-A routine (oracle/ckoracle.c: ora_reverse_parameters, an independent implementation pinned in
tests/test_oracle_convert.py).
"""
import json
import os

import numpy as np
import pytest

import oracle
from paper_1309_2710_b200 import binding

HERE = os.path.dirname(os.path.abspath(__file__))
INP = open(os.path.join(HERE, "golden", "synthetic_hon.inp")).read()
EXP = json.load(open(os.path.join(HERE, "golden", "synthetic_hon.json")))
NAMES = [s["name"] for s in EXP["species"]]


def _side(m, ptr, sp, nu, j):
    return {NAMES[sp[e]]: int(nu[e]) for e in range(ptr[j], ptr[j + 1])}


def test_reader_recovers_species_thermo_and_forward_reactions():
    m = binding.chemkin_parse(INP)
    assert m.species_names == NAMES
    for k, s in enumerate(EXP["species"]):
        assert abs(m.mol_weight[k] / s["W"] - 1) < 1e-12
        assert m.T_mid[k] == s["T_mid"]
        assert np.array_equal(m.nasa[k], s["nasa_low"]) and np.array_equal(m.nasa_high[k], s["nasa_high"])
    rx = EXP["reactions"]
    assert m.n_reactions == sum(2 if r["reversible"] else 1 for r in rx)
    tb = {int(j): i for i, j in enumerate(m.tb_reaction)}
    fo = {int(j): i for i, j in enumerate(m.fo_reaction)}
    j = 0
    for i, r in enumerate(rx):
        for rev in ([0, 1] if r["reversible"] else [0]):
            assert m.origin[j] == i and m.is_reverse[j] == rev
            lhs, rhs = (r["prod"], r["reac"]) if rev else (r["reac"], r["prod"])
            assert _side(m, m.reac_ptr, m.reac_species, m.reac_nu, j) == lhs
            assert _side(m, m.prod_ptr, m.prod_species, m.prod_nu, j) == rhs
            if not rev:
                assert m.arr_A[j] == r["A"] and m.arr_beta[j] == r["beta"] and abs(m.arr_E[j] / max(r["E_cal"], 1e-300) - 1) < 1e-14
            # third body / efficiencies on both directions
            has_set = r["third_body"] or (r["falloff"] and r["eff"])
            assert (j in tb) == bool(has_set)
            if has_set:
                t = tb[j]
                got = {NAMES[m.tb_species[e]]: m.tb_eff[e] for e in range(m.tb_ptr[t], m.tb_ptr[t + 1])}
                assert got == r["eff"]
            assert (j in fo) == r["falloff"]
            if r["falloff"] and not rev:
                f = fo[j]
                assert np.allclose(m.fo_low[f], r["low"], rtol=1e-14)
                tr = r.get("troe")
                if tr is None:
                    assert np.isnan(m.fo_troe[f, 0])
                else:
                    assert np.array_equal(m.fo_troe[f, :len(tr)], tr)
                    assert len(tr) == 4 or np.isinf(m.fo_troe[f, 3])
            j += 1


@pytest.mark.parametrize("fit_T", [None, [800.0, 1400.0, 2400.0]])
def test_reverse_parameters_are_appendix_a_of_the_oracle(fit_T):
    m = binding.chemkin_parse(INP, fit_T=fit_T)
    om = oracle.OracleMech(m)          # the irreversible mechanism, two-range thermo and fall-off included
    T3 = [1000.0, 1500.0, 2000.0] if fit_T is None else fit_T
    rx = EXP["reactions"]
    fo = {int(j): i for i, j in enumerate(m.fo_reaction)}
    checked = 0
    for j in range(m.n_reactions):
        if not m.is_reverse[j]:
            continue
        r = rx[m.origin[j]]
        if "rev" in r:                              # explicit REV parameters are taken as they are
            assert m.arr_A[j] == r["rev"][0] and m.arr_beta[j] == r["rev"][1] and abs(m.arr_E[j] / r["rev"][2] - 1) < 1e-14
            continue
        A_r, b_r, E_r = om.reverse_parameters(j - 1, T3)     # the forward reaction sits just before its reverse
        assert abs(m.arr_A[j] / A_r - 1) < 1e-8 and abs(m.arr_beta[j] - b_r) < 1e-9 and abs(m.arr_E[j] - E_r) < 1e-5 * max(1.0, abs(E_r))
        # at the three temperatures k_f / k_r reproduces K_c (Eq. A.1-A.3)
        for T in T3:
            kf = m.arr_A[j - 1] * T ** m.arr_beta[j - 1] * np.exp(-m.arr_E[j - 1] / (1.98720425864 * T))
            kr = m.arr_A[j] * T ** m.arr_beta[j] * np.exp(-m.arr_E[j] / (1.98720425864 * T))
            assert abs(kf / kr / om.equilibrium_constant(j - 1, T) - 1) < 1e-8
        if j in fo:     # a fall-off reaction: the low-pressure limit of the reverse is k_0 / K_c fitted the same way
            f, ff = fo[j], fo[j - 1]
            for T in T3:
                k0f = m.fo_low[ff, 0] * T ** m.fo_low[ff, 1] * np.exp(-m.fo_low[ff, 2] / (1.98720425864 * T))
                k0r = m.fo_low[f, 0] * T ** m.fo_low[f, 1] * np.exp(-m.fo_low[f, 2] / (1.98720425864 * T))
                assert abs(k0f / k0r / om.equilibrium_constant(j - 1, T) - 1) < 1e-8
            assert np.array_equal(m.fo_troe[f], m.fo_troe[ff], equal_nan=True)
        checked += 1
    assert checked >= 8


def test_units_and_separate_thermo_file():
    head, rest = INP.split("THERMO ALL")
    thermo_body, reactions = rest.split("END", 1)
    mech_only = head + reactions
    thermo_only = "THERMO ALL" + thermo_body + "END\n"
    base = binding.chemkin_parse(INP)
    split = binding.chemkin_parse(mech_only, thermo_text=thermo_only)
    for k in ("arr_A", "arr_beta", "arr_E", "nasa", "nasa_high", "mol_weight", "fo_low"):
        assert np.array_equal(getattr(base, k), getattr(split, k)), k
    # the same energies given in cal/mol and in kelvin
    fwd = base.is_reverse == 0

    def reunit(text, unit, f):
        out = []
        for ln in text.splitlines():
            if ln.startswith("REACTIONS"):
                ln = "REACTIONS " + unit
            elif "! E in kJ/mol" in ln:
                eq, A, b, E = ln.split("!")[0].rsplit(None, 3)
                ln = "%s %s %s %.10E" % (eq, A, b, f(float(E)))
            elif ln.strip().startswith(("LOW", "REV")):
                kw, vals = ln.split("/")[0], ln.split("/")[1].split()
                ln = "%s/ %s %s %.10E /" % (kw, vals[0], vals[1], f(float(vals[2])))
            out.append(ln)
        return "\n".join(out) + "\n"

    cal = binding.chemkin_parse(reunit(INP, "CAL/MOLE", lambda e: e * 1000.0 / 4.184))
    kel = binding.chemkin_parse(reunit(INP, "KELVINS", lambda e: e * 1000.0 / 4.184 / 1.98720425864))
    for other in (cal, kel):
        assert np.allclose(other.arr_E[fwd], base.arr_E[fwd], rtol=1e-9, atol=1e-9)
        assert np.allclose(other.arr_A, base.arr_A, rtol=1e-7) and np.allclose(other.fo_low, base.fo_low, rtol=1e-7)


def _without_last_low(text):
    lines = text.splitlines()
    last = max(i for i, l in enumerate(lines) if l.strip().startswith("LOW"))
    return "\n".join(lines[:last] + lines[last + 1:]) + "\n"


def test_syntax_errors_are_reported():
    cases = [
        (INP.replace("H+O2=O+OH ", "H+O2=O+XYZ "), binding.EINVAL, "unknown species"),
        (INP.replace("2OH=O+H2O", "2OH=O+H2O2"), binding.EINVAL, "not balanced"),
        (_without_last_low(INP), binding.EINVAL, "without LOW"),
        (INP.replace("   N2/1.40/", "   SRI / 0.5 100. 200. /"), binding.EUNSUPPORTED, "SRI"),
        (INP.replace("H+H+M=H2+M", "H+H+M=H2"), binding.EINVAL, "third body"),
        (INP.replace("HO2  H2O2  N2  AR  NO  N", "HO2  H2O2  N2  AR  NO  N  HE"), binding.EINVAL, "no thermodynamic data"),
    ]
    for text, code, what in cases:
        with pytest.raises(binding.CkbError) as e:
            binding.chemkin_parse(text)
        assert e.value.code == code and what.lower() in str(e.value).lower(), (what, str(e.value))


@pytest.mark.gpu
def test_parsed_mechanism_runs_on_the_gpu_and_matches_the_oracle():
    """The converted mechanism through ckb_mech_load3 on every mapping: f(y) and an integration against the oracle."""
    import torch
    from test_gpu_parity import _compare, _oracle, _run_gpu
    m = binding.chemkin_parse(INP)
    om = oracle.OracleMech(m)
    rng = np.random.default_rng(1)
    N, K = 96, m.n_species
    # 900-1500 K, dt = 1e-6 s: sigma up to ~1e9 1/s, RKC with 2-3 stages, RKCK with a few rejections per system; the oracle
    # perturbed by one ulp takes the same decisions on all 96 systems there (hotter states reach s > 100: DESIGN.md 4.6)
    states = np.ascontiguousarray(np.vstack([rng.uniform(900, 1500, N)[None, :], rng.dirichlet(np.ones(K), size=N).T]))
    p = 1.01325e6
    ref = np.stack([om.rhs(states[:, i].copy(), p) for i in range(N)], axis=1)
    h = binding.mech_load(m)
    for v in ("thread", "warp", "sub4", "sub8"):
        out = binding.rhs(h, torch.from_numpy(states).cuda(), p=p, variant=v).cpu().numpy()
        scale = np.abs(ref).max(axis=1, keepdims=True)
        assert (np.abs(out - ref) <= 1e-11 * scale + 1e-13 * np.abs(ref)).all(), v
    h.close()
    for method, variant in (("rkck", "thread"), ("rkc", "warp"), ("rkc", "gen")):
        _compare(_run_gpu(m, states, p, 1e-6, method, variant=variant), _oracle(m, states, p, 1e-6, method), max_flip_frac=0.03)
