"""Writes tests/golden/synthetic_hon.inp (a mechanism in the Chemkin text format) and synthetic_hon.json (what a
reader must get out of it).  Everything in the file is synthetic: the species are the usual names of the H/O/N system,
every number (NASA coefficients, Arrhenius parameters, efficiencies, Troe parameters) is drawn here from a seeded
generator -- no data of any published mechanism.  Calls nothing of the CUDA path and nothing of oracle/.

    python tests/golden/make_chemkin_fixture.py
"""
import json
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
AW = {"H": 1.008, "O": 15.999, "N": 14.007, "AR": 39.948}
SPECIES = [("H2", {"H": 2}), ("O2", {"O": 2}), ("H", {"H": 1}), ("O", {"O": 1}), ("OH", {"O": 1, "H": 1}),
           ("H2O", {"H": 2, "O": 1}), ("HO2", {"H": 1, "O": 2}), ("H2O2", {"H": 2, "O": 2}), ("N2", {"N": 2}),
           ("AR", {"AR": 1}), ("NO", {"N": 1, "O": 1}), ("N", {"N": 1})]
# (equation as written, reactants {name: nu}, products, arrow, kind, extras)
REACTIONS = [
    ("H+O2=O+OH", {"H": 1, "O2": 1}, {"O": 1, "OH": 1}, "=", "plain", {}),
    ("O+H2<=>H+OH", {"O": 1, "H2": 1}, {"H": 1, "OH": 1}, "<=>", "plain", {}),
    ("2OH=O+H2O", {"OH": 2}, {"O": 1, "H2O": 1}, "=", "plain", {}),
    ("H+H+M=H2+M", {"H": 2}, {"H2": 1}, "=", "tb", {"eff": {"H2": 2.5, "H2O": 12.0, "AR": 0.7}}),
    ("H+O2(+M)=HO2(+M)", {"H": 1, "O2": 1}, {"HO2": 1}, "=", "fo", {"eff": {"H2O": 11.0, "O2": 0.8}, "troe": 4}),
    ("H2O2(+M)<=>OH+OH(+M)", {"H2O2": 1}, {"OH": 2}, "<=>", "fo", {"eff": {"N2": 1.4}, "troe": 3}),
    ("HO2+HO2=>H2O2+O2", {"HO2": 2}, {"H2O2": 1, "O2": 1}, "=>", "plain", {"dup": True}),
    ("HO2+HO2=>H2O2+O2", {"HO2": 2}, {"H2O2": 1, "O2": 1}, "=>", "plain", {"dup": True}),
    ("N+O2=NO+O", {"N": 1, "O2": 1}, {"NO": 1, "O": 1}, "=", "plain", {"rev": True}),
    ("N+NO<=>N2+O", {"N": 1, "NO": 1}, {"N2": 1, "O": 1}, "<=>", "plain", {}),
    ("H+OH+M=H2O+M", {"H": 1, "OH": 1}, {"H2O": 1}, "=", "tb", {"eff": {}}),
    ("O + O + M = O2 + M", {"O": 2}, {"O2": 1}, "=", "tb", {"eff": {"AR": 0.5}}),
    ("N+N(+M)=N2(+M)", {"N": 2}, {"N2": 1}, "=", "fo", {"eff": {}, "troe": 0}),
    ("H2O2+H=>H2O+OH", {"H2O2": 1, "H": 1}, {"H2O": 1, "OH": 1}, "=>", "plain", {}),
]
KJ = 4.184  # the file gives energies in KJOULES/MOLE


def e15(x):
    return "%15.8E" % x


def main(seed=20131309):
    rng = np.random.default_rng(seed)
    lines = ["! synthetic test mechanism: every number below comes from tests/golden/make_chemkin_fixture.py",
             "ELEMENTS", "H O N AR", "END", "SPECIES"]
    lines += ["  ".join(n for n, _ in SPECIES[:6]), "  ".join(n for n, _ in SPECIES[6:]) + "   ! second line", "END"]
    lines += ["THERMO ALL", "   300.000  1000.000  5000.000"]
    spec_out = []
    for name, comp in SPECIES:
        tmid = float(rng.choice([900.0, 1000.0, 1200.0]))
        # cp/R stays in 3..8 over 300..5000 K (a positive heat capacity: the mechanism must be integrable)
        lo = np.array([rng.uniform(3.5, 5.0), rng.uniform(0.0, 8e-4), rng.uniform(-4e-8, 4e-8), rng.uniform(-4e-12, 4e-12),
                       rng.uniform(-2e-16, 2e-16), -25000.0 * (sum(comp.values()) - 1) + rng.uniform(-2e3, 2e3), rng.uniform(3.0, 5.0)])
        # (a6: about 50 kcal/mol per bond, so that an association is exothermic enough to offset its entropy loss and the
        # equilibrium constants -- hence the fitted reverse rates -- have physical magnitudes)
        hi = lo * rng.uniform(0.7, 1.0, 7)
        # the two ranges meet at T_mid: a1, a6, a7 of the high range from the continuity of cp, h and s (as real fits do)
        T = tmid
        pw = np.array([T, T ** 2, T ** 3, T ** 4])
        hi[0] = lo[0] + np.dot(lo[1:5] - hi[1:5], pw)
        hcoef = pw / np.array([2.0, 3.0, 4.0, 5.0])
        hi[5] = lo[5] + T * ((lo[0] - hi[0]) + np.dot(lo[1:5] - hi[1:5], hcoef))
        scoef = pw / np.array([1.0, 2.0, 3.0, 4.0])
        hi[6] = lo[6] + (lo[0] - hi[0]) * np.log(T) + np.dot(lo[1:5] - hi[1:5], scoef)
        lo = np.array([float(e15(x)) for x in lo])
        hi = np.array([float(e15(x)) for x in hi])
        compf = "".join("%-2s%3d" % (e, c) for e, c in comp.items()).ljust(20)
        l1 = ("%-18s%-6s%sG%10.3f%10.3f%8.2f" % (name, "SYNTH", compf, 300.0, 5000.0, tmid)).ljust(79) + "1"
        c = list(hi) + list(lo)
        l2 = "".join(e15(x) for x in c[0:5]).ljust(79) + "2"
        l3 = "".join(e15(x) for x in c[5:10]).ljust(79) + "3"
        l4 = "".join(e15(x) for x in c[10:14]).ljust(79) + "4"
        lines += [l1, l2, l3, l4]
        spec_out.append(dict(name=name, W=sum(AW[e] * c_ for e, c_ in comp.items()), T_mid=tmid, nasa_low=list(lo), nasa_high=list(hi)))
    lines += ["END", "REACTIONS   KJOULES/MOLE   MOLES"]
    rx_out = []

    def num(x):
        return float("%.6E" % x)

    for eq, reac, prod, arrow, kind, ex in REACTIONS:
        A, b, E = num(10 ** rng.uniform(4, 8)), num(rng.uniform(-1.0, 1.0)), num(rng.uniform(0, 80.0))
        lines.append("%-40s %12.6E %13.6E %12.6E   ! E in kJ/mol" % (eq, A, b, E))
        r = dict(equation=eq, reac=reac, prod=prod, reversible=arrow != "=>", A=A, beta=b, E_cal=E * 1000.0 / KJ,
                 third_body=kind == "tb", falloff=kind == "fo", eff=ex.get("eff", {}))
        if kind == "fo":
            low = [num(A * 10 ** rng.uniform(4.0, 6.5)), num(b + rng.uniform(-1.0, 0.0)), num(rng.uniform(0, 20.0))]
            lines.append("   LOW / %.6E %.6E %.6E /" % tuple(low))
            r["low"] = [low[0], low[1], low[2] * 1000.0 / KJ]
            if ex["troe"]:
                tr = [num(rng.uniform(0.3, 0.9)), num(rng.uniform(50, 500)), num(rng.uniform(800, 3000)), num(rng.uniform(3000, 9000))][:ex["troe"]]
                lines.append("   TROE / " + " ".join("%.6E" % x for x in tr) + " /")
                r["troe"] = tr
        if ex.get("eff"):
            lines.append("   " + " ".join("%s/%.2f/" % (k, v) for k, v in ex["eff"].items()))
        if ex.get("rev"):
            rev = [num(10 ** rng.uniform(4, 8)), num(rng.uniform(-1, 1)), num(rng.uniform(0, 150.0))]
            lines.append("   REV / %.6E %.6E %.6E /" % tuple(rev))
            r["rev"] = [rev[0], rev[1], rev[2] * 1000.0 / KJ]
        if ex.get("dup"):
            lines.append("   DUPLICATE")
        rx_out.append(r)
    lines.append("END")
    with open(os.path.join(HERE, "synthetic_hon.inp"), "w") as fh:
        fh.write("\n".join(lines) + "\n")
    with open(os.path.join(HERE, "synthetic_hon.json"), "w") as fh:
        json.dump(dict(species=spec_out, reactions=rx_out, source="tests/golden/make_chemkin_fixture.py, seed %d" % seed), fh, indent=1)
        fh.write("\n")


if __name__ == "__main__":
    main()
