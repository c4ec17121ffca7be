"""Seeded synthetic inputs: mechanisms and initial states shaped like the paper's workloads.

This module is the ONE piece shared by the CUDA path (tests, bench) and the CPU oracle's tests.
It holds none of the method's arithmetic: no rate law, no thermodynamic evaluation, no integrator.
It only draws tables (species, stoichiometry, Arrhenius parameters, polynomial coefficients) and
states (T, Y) from seeded numpy generators.  Recipe: SURVEY.md section 8(d) D1/D2, restated in
DESIGN.md section 5.  The paper's own mechanisms (9/38, 13/54, 53/634, 111/1566
species / irreversible reactions) are third-party data that is not reproduced; these inputs stand in
for them with the same shapes.

The single global rate factor ``g`` per mechanism (stiffness calibration) is
NOT computed here: it is read from ``synth_calibration.json`` beside this file, which is written by
``oracle/calibrate_sigma.py`` (a committed script that evaluates only the oracle).
"""
from __future__ import annotations

import itertools
import json
import os
from dataclasses import dataclass, field

import numpy as np

ATOMIC_WEIGHT = {"H": 1.008, "C": 12.011, "N": 14.007, "O": 15.999}
P_ATM = 1.01325e6            # dyn/cm^2
_RU = 8.314462618e7          # erg/(mol K) -- used only to form the reference concentration C_ref
_CALIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "synth_calibration.json")


@dataclass
class Mechanism:
    """Plain arrays describing one mechanism (the argument of mech_load on both libraries)."""
    name: str
    elements: tuple
    elem_counts: np.ndarray      # [K][E] int32, atoms of element e in species k
    mol_weight: np.ndarray       # [K] g/mol
    nasa: np.ndarray             # [K][7] a1..a7, one temperature range
    arr_A: np.ndarray            # [R] cgs
    arr_beta: np.ndarray         # [R]
    arr_E: np.ndarray            # [R] cal/mol
    reac_ptr: np.ndarray         # [R+1] int32 CSR over reactant entries
    reac_species: np.ndarray     # [nnz_r] int32
    reac_nu: np.ndarray          # [nnz_r] int32 >= 1
    prod_ptr: np.ndarray         # [R+1]
    prod_species: np.ndarray
    prod_nu: np.ndarray
    tb_reaction: np.ndarray      # [R3] int32 indices of third-body reactions
    tb_ptr: np.ndarray           # [R3+1] CSR over listed (non-unity) efficiencies
    tb_species: np.ndarray       # [nnz_tb] int32
    tb_eff: np.ndarray           # [nnz_tb] alpha_jk
    rate_factor: float = 1.0     # calibration factor already folded into arr_A
    meta: dict = field(default_factory=dict)
    nasa_high: np.ndarray = None # [K][7] optional second (high) temperature range, used where T > T_mid[k]
    T_mid: np.ndarray = None     # [K] K
    fo_reaction: np.ndarray = None  # [n_fo] int32: fall-off reactions (arr_A/beta/E are then the high-pressure limit)
    fo_low: np.ndarray = None       # [n_fo][3] A_0, beta_0, E_0 of the low-pressure limit
    fo_troe: np.ndarray = None      # [n_fo][4] a, T***, T*, T** (a = NaN: Lindemann; T** = inf: three-parameter form)

    @property
    def n_species(self) -> int:
        return int(self.mol_weight.shape[0])

    @property
    def n_reactions(self) -> int:
        return int(self.arr_A.shape[0])

    @property
    def n_third_body(self) -> int:
        return int(self.tb_reaction.shape[0])


@dataclass(frozen=True)
class ConfigSpec:
    """One entry of BASELINE.json `configs` (shape + state recipe)."""
    cfg: int
    mech_id: int                 # mechanisms are shared between cfg0 and cfg1
    name: str
    elements: tuple
    K: int
    R: int
    max_side: int                # max molecules per reaction side (2 or 3)
    A_range: tuple               # nominal log-uniform range of the bimolecular-equivalent A'
    n_tb_pairs: int
    class_mix: tuple             # ((n_reac, n_prod) unordered class, fraction) ...
    method: str                  # "rkck" | "rkc"
    T_range: tuple
    dirichlet_alpha: float
    dt: tuple                    # global step(s)
    N_list: tuple
    sigma_span: tuple            # target spectral-radius span at t=0 (calibration target)


_MIX_SMALL = ((frozenset({(2, 2)}), 0.75), (frozenset({(1, 2), (2, 1)}), 0.25))
_MIX_LARGE = ((frozenset({(2, 2)}), 0.70), (frozenset({(1, 2), (2, 1)}), 0.15),
              (frozenset({(2, 3), (3, 2)}), 0.10), (frozenset({(1, 3), (3, 1), (3, 3)}), 0.05))

CONFIGS = (
    ConfigSpec(0, 0, "h2-like 9/38", ("H", "O"), 9, 38, 2, (1e6, 1e14), 4, _MIX_SMALL, "rkck",
               (1000.0, 1500.0), 1.0, (1e-6,), (1024,), (1e4, 1e6)),
    ConfigSpec(1, 0, "h2-like 9/38", ("H", "O"), 9, 38, 2, (1e6, 1e14), 4, _MIX_SMALL, "rkck",
               (800.0, 2000.0), 1.0, (1e-6,), tuple(2 ** e for e in (6, 8, 10, 12, 14, 16, 18, 19)),
               (1e4, 1e6)),
    ConfigSpec(2, 2, "h2co-like 13/54", ("C", "H", "O"), 13, 54, 2, (1e8, 1e16), 4, _MIX_SMALL, "rkc",
               (1000.0, 1800.0), 0.5, (1e-6,), tuple(2 ** e for e in range(6, 19, 2)), (1e5, 1e7)),
    ConfigSpec(3, 3, "ch4-like 53/634", ("C", "H", "O", "N"), 53, 634, 3, (1e8, 1e16), 48, _MIX_LARGE,
               "rkc", (1000.0, 2200.0), 0.3, (1e-6,), tuple(2 ** e for e in range(6, 18)) + (2 ** 17,),
               (1e6, 1e8)),
    ConfigSpec(4, 4, "c2h4-like 111/1566", ("C", "H", "O", "N"), 111, 1566, 3, (1e8, 1e16), 117,
               _MIX_LARGE, "rkc", (900.0, 2400.0), 0.2, (1e-6, 1e-5),
               tuple(2 ** e for e in range(13, 17)), (1e7, 1e9)),
)


def _rng(seed: int, ident: int, stream: int) -> np.random.Generator:
    return np.random.default_rng([int(seed), int(ident), int(stream)])


def _draw_species(rng, n_elem: int, K: int) -> np.ndarray:
    """K distinct non-zero element-count vectors from {0..4}^E, drawn without replacement with
    probability proportional to 2^-(number of atoms): small molecules are favoured, as in a real
    mechanism, which is what makes element-balanced reactions between the species plentiful (a
    uniform draw of 13 vectors out of 124 yields ~8 balanced pairs; 27 are needed)."""
    every = [v for v in itertools.product(range(5), repeat=n_elem) if any(v)]
    w = np.array([2.0 ** (-sum(v)) for v in every])
    pick = rng.choice(len(every), size=K, replace=False, p=w / w.sum())
    return np.array([every[i] for i in sorted(pick)], dtype=np.int32)


class _PairSampler:
    """Element-balanced reversible pairs (left, right) of DISJOINT species multisets with
    1..max_side molecules per side, grouped by class (n_left <= n_right).

    Sides with equal summed element vector are bucketed with numpy; a class whose bucket-pair count
    is small (<= 2e5) is enumerated exactly and shuffled, a large one (e.g. 7.4e6 (3,3) candidates
    for 111 species) is sampled uniformly by rejection: bucket ~ number of side pairs, then one side
    of each size, rejected when the sides share a species or the pair was already taken.
    """

    def __init__(self, counts: np.ndarray, max_side: int):
        K, E = counts.shape
        self.sides, self.keys, self.groups = {}, {}, {}
        radix = 1 + 4 * max_side
        for m in range(1, max_side + 1):
            ms = np.array(list(itertools.combinations_with_replacement(range(K), m)), dtype=np.int32)
            tot = counts[ms].sum(axis=1).astype(np.int64)          # [n][E]
            key = np.zeros(len(ms), dtype=np.int64)
            for e in range(E):
                key = key * radix + tot[:, e]
            o = np.argsort(key, kind="stable")
            self.sides[m], self.keys[m] = ms[o], key[o]
            uk, start, cnt = np.unique(self.keys[m], return_index=True, return_counts=True)
            self.groups[m] = (uk, start, cnt)
        self.taken = set()

    def _disjoint(self, a, b):
        return not (set(a.tolist()) & set(b.tolist()))

    def draw(self, rng, na: int, nb: int, n: int):
        """Up to n not-yet-taken pairs of class (na, nb), na <= nb, uniformly without replacement."""
        if n <= 0 or na not in self.sides or nb not in self.sides:
            return []
        uka, sa, ca = self.groups[na]
        ukb, sb, cb = self.groups[nb]
        common, ia, ib = np.intersect1d(uka, ukb, return_indices=True)
        if len(common) == 0:
            return []
        sa, ca, sb, cb = sa[ia], ca[ia], sb[ib], cb[ib]
        w = (ca * (ca - 1) // 2) if na == nb else ca * cb
        total = int(w.sum())
        out = []
        A, B = self.sides[na], self.sides[nb]
        if total <= 200_000:
            cand = []
            for g in range(len(common)):
                for i in range(sa[g], sa[g] + ca[g]):
                    j0 = i + 1 if na == nb else sb[g]
                    for j in range(j0, sb[g] + cb[g]):
                        if self._disjoint(A[i], B[j]):
                            pair = (tuple(A[i].tolist()), tuple(B[j].tolist()))
                            if pair not in self.taken:
                                cand.append(pair)
            for i in rng.permutation(len(cand))[:n]:
                out.append(cand[i])
        else:
            p = w / w.sum()
            tries = 0
            while len(out) < n and tries < 1000 * n + 10000:
                tries += 1
                g = int(rng.choice(len(common), p=p))
                i = sa[g] + int(rng.integers(ca[g]))
                j = sb[g] + int(rng.integers(cb[g]))
                if na == nb and i == j:
                    continue
                if na == nb and j < i:
                    i, j = j, i
                if not self._disjoint(A[i], B[j]):
                    continue
                pair = (tuple(A[i].tolist()), tuple(B[j].tolist()))
                if pair in self.taken or pair in out:
                    continue
                out.append(pair)
        self.taken.update(out)
        return out


def _sample_pairs(rng, sampler: "_PairSampler", n_pairs: int, class_mix, max_side: int):
    """Stratified draw of n_pairs reversible pairs; a class short of candidates spills into (2,2),
    and what (2,2) cannot supply is taken from the remaining classes in order."""
    def norm(c):
        return (min(c), max(c))
    chosen = []
    remaining = n_pairs
    short = 0
    for i, (classes, frac) in enumerate(class_mix):
        n = int(round(frac * n_pairs)) if i < len(class_mix) - 1 else remaining
        n = min(n, remaining)
        remaining -= n
        cls = sorted({norm(c) for c in classes})
        for ci, c in enumerate(cls):                   # split n evenly over the class's shapes
            n_c = n // len(cls) + (1 if ci < n % len(cls) else 0)
            got = sampler.draw(rng, c[0], c[1], n_c)
            chosen.extend(got)
            short += n_c - len(got)
    spill = [(2, 2)] + [(a, b) for a in range(1, max_side + 1) for b in range(a, max_side + 1)
                        if (a, b) != (2, 2)]
    for c in spill:
        if short <= 0:
            break
        got = sampler.draw(rng, c[0], c[1], short)
        chosen.extend(got)
        short -= len(got)
    return chosen if short <= 0 else None


def _side_to_entries(side):
    sp = sorted(set(side))
    return sp, [side.count(k) for k in sp]


def load_calibration() -> dict:
    if os.path.exists(_CALIB_PATH):
        with open(_CALIB_PATH) as fh:
            return json.load(fh)
    return {}


def make_mechanism(cfg: int, seed: int = 0, calibrated: bool = True) -> Mechanism:
    """Build the synthetic mechanism of BASELINE.json configs[cfg]."""
    spec = CONFIGS[cfg]
    E = len(spec.elements)
    n_pairs = spec.R // 2
    attempt = 0
    while True:
        rng = _rng(seed, spec.mech_id, 0 + 16 * attempt)
        counts = _draw_species(rng, E, spec.K)
        pairs = _sample_pairs(rng, _PairSampler(counts, spec.max_side), n_pairs, spec.class_mix,
                              spec.max_side)
        if pairs is not None:
            break
        attempt += 1                      # too few balanced candidates: redraw the species set
        if attempt > 256:
            raise RuntimeError("could not draw a species set with enough balanced reactions")
    aw = np.array([ATOMIC_WEIGHT[e] for e in spec.elements])
    W = counts @ aw

    # third-body pairs: prefer (1,2) classes, never a 3-molecule side
    idx_12 = [i for i, (l, r) in enumerate(pairs) if (len(l), len(r)) == (1, 2)]
    idx_22 = [i for i, (l, r) in enumerate(pairs) if (len(l), len(r)) == (2, 2)]
    order = [idx_12[i] for i in rng.permutation(len(idx_12))] + [idx_22[i] for i in rng.permutation(len(idx_22))]
    tb_pairs = sorted(order[: spec.n_tb_pairs])
    n_listed = min(3, spec.K)

    reac_ptr, reac_sp, reac_nu = [0], [], []
    prod_ptr, prod_sp, prod_nu = [0], [], []
    order_j = []
    tb_reaction, tb_ptr, tb_sp, tb_eff = [], [0], [], []
    for i, (left, right) in enumerate(pairs):
        is_tb = i in set(tb_pairs)
        if is_tb:
            listed = sorted(int(k) for k in rng.choice(spec.K, size=n_listed, replace=False))
            eff = rng.uniform(0.5, 3.0, size=n_listed)
        for (a, b) in ((left, right), (right, left)):       # forward, then reverse
            sp, nu = _side_to_entries(a)
            reac_sp += sp
            reac_nu += nu
            reac_ptr.append(len(reac_sp))
            sp, nu = _side_to_entries(b)
            prod_sp += sp
            prod_nu += nu
            prod_ptr.append(len(prod_sp))
            order_j.append(len(a) + (1 if is_tb else 0))
            if is_tb:
                tb_reaction.append(len(order_j) - 1)
                tb_sp += listed
                tb_eff += list(eff)
                tb_ptr.append(len(tb_sp))
    R = len(order_j)
    assert R == spec.R
    order_j = np.array(order_j, dtype=np.float64)

    # Arrhenius parameters: forward and reverse drawn independently (no equilibrium consistency)
    lo, hi = spec.A_range
    A_prime = 10.0 ** rng.uniform(np.log10(lo), np.log10(hi), size=R)
    beta = rng.uniform(-1.0, 2.0, size=R)
    E_act = rng.uniform(0.0, 30000.0, size=R)                # cal/mol
    C_ref = P_ATM / (_RU * 1500.0)
    A = A_prime * C_ref ** (2.0 - order_j) / 1000.0 ** beta   # nominal range = bimolecular k at 1000 K

    nasa = np.zeros((spec.K, 7))
    nasa[:, 0] = rng.uniform(3.5, 5.0, size=spec.K)
    nasa[:, 1] = rng.uniform(0.0, 8e-4, size=spec.K)
    nasa[:, 2] = rng.uniform(-5e-8, 5e-8, size=spec.K)
    nasa[:, 3] = rng.uniform(-5e-12, 5e-12, size=spec.K)
    nasa[:, 4] = rng.uniform(-5e-16, 5e-16, size=spec.K)
    nasa[:, 5] = rng.uniform(-3000.0, 3000.0, size=spec.K)

    g = 1.0
    if calibrated:
        cal = load_calibration().get(f"mech{spec.mech_id}_seed{seed}")
        if cal is not None:
            g = float(cal["g"])
    i32 = lambda x: np.ascontiguousarray(np.array(x, dtype=np.int32))
    return Mechanism(
        name=spec.name, elements=spec.elements, elem_counts=counts,
        mol_weight=np.ascontiguousarray(W, dtype=np.float64), nasa=np.ascontiguousarray(nasa),
        arr_A=np.ascontiguousarray(A * g), arr_beta=np.ascontiguousarray(beta),
        arr_E=np.ascontiguousarray(E_act),
        reac_ptr=i32(reac_ptr), reac_species=i32(reac_sp), reac_nu=i32(reac_nu),
        prod_ptr=i32(prod_ptr), prod_species=i32(prod_sp), prod_nu=i32(prod_nu),
        tb_reaction=i32(tb_reaction), tb_ptr=i32(tb_ptr), tb_species=i32(tb_sp),
        tb_eff=np.ascontiguousarray(np.array(tb_eff, dtype=np.float64)),
        rate_factor=g,
        meta={"cfg": cfg, "seed": seed, "species_redraws": attempt, "n_pairs": n_pairs,
              "tb_pairs": len(tb_pairs)},
    )


def make_states(cfg: int, N: int, seed: int = 0, stream: int = 1, ordering: str = "shuffled"):
    """States for configs[cfg]: SoA array [(K+1)][N] (row 0 = T in K, rows 1..K = Y) and P (dyn/cm^2).

    One array per config is drawn at the config's largest N and smaller N are prefixes, so sweeps
    nest.  ordering = "shuffled" (i.i.d. order, the default for every headline
    number) or "similar" (the same N states sorted by T; stands in for the paper's neighbouring
    grid points).
    """
    spec = CONFIGS[cfg]
    n_max = max(max(spec.N_list), N)
    rng = _rng(seed, 100 + cfg, stream)
    T = rng.uniform(spec.T_range[0], spec.T_range[1], size=n_max)
    Y = rng.dirichlet(np.full(spec.K, spec.dirichlet_alpha), size=n_max)
    T, Y = T[:N], Y[:N]
    if ordering == "similar":
        o = np.argsort(T, kind="stable")
        T, Y = T[o], Y[o]
    elif ordering != "shuffled":
        raise ValueError(ordering)
    states = np.empty((spec.K + 1, N), dtype=np.float64)
    states[0] = T
    states[1:] = Y.T
    return np.ascontiguousarray(states), P_ATM


def make_densities(mech: "Mechanism", states: np.ndarray, p: float = P_ATM) -> np.ndarray:
    """Densities (g/cm^3) for the constant-volume inputs: the density each system of `states` has at pressure p
    (ideal gas, rho = p / (Ru T sum_k Y_k/W_k)) -- i.e. the same 1 atm initial conditions as the constant-pressure
    workload, then held at their own volume.  Input recipe only; no method arithmetic."""
    w = np.asarray(mech.mol_weight, dtype=np.float64)
    return p / (_RU * states[0] * (states[1:] / w[:, None]).sum(axis=0))


def with_two_range_thermo(mech: "Mechanism", T_range, seed: int = 0) -> "Mechanism":
    """The same mechanism with two-range NASA fits: `mech.nasa` stays the low range, a high range is
    drawn beside it, and each species switches at its own T_mid drawn inside `T_range` (so that a batch of states
    straddles the switch and systems cross it while they react).  Like real fits, c_p and h are continuous at T_mid:
    a2..a5 of the high range are drawn (a flatter polynomial), a1 and a6 follow from the two continuity conditions.
    Input recipe only; the source term itself is in neither library's interest here."""
    import copy
    rng = _rng(seed, 900, int(mech.n_species))
    K = mech.n_species
    lo = np.asarray(mech.nasa, dtype=np.float64)
    Tm = rng.uniform(T_range[0] + 0.25 * (T_range[1] - T_range[0]), T_range[1] - 0.25 * (T_range[1] - T_range[0]), size=K)
    hi = np.zeros_like(lo)
    hi[:, 1] = lo[:, 1] * rng.uniform(0.3, 0.8, size=K)
    hi[:, 2] = lo[:, 2] * rng.uniform(0.3, 0.8, size=K)
    hi[:, 3] = lo[:, 3] * rng.uniform(0.3, 0.8, size=K)
    hi[:, 4] = lo[:, 4] * rng.uniform(0.3, 0.8, size=K)
    pw = np.stack([Tm ** i for i in range(5)], axis=1)                       # [K][5]: 1, T, T^2, T^3, T^4
    hi[:, 0] = (lo[:, :5] * pw).sum(1) - (hi[:, 1:5] * pw[:, 1:]).sum(1)    # c_p/R continuous
    H = lambda a: (a[:, :5] * pw * Tm[:, None] / np.arange(1, 6)).sum(1)     # T (a1 + a2 T/2 + ... + a5 T^4/5)
    hi[:, 5] = lo[:, 5] + H(lo) - H(hi)                                       # h/R continuous
    hi[:, 6] = lo[:, 6]
    out = copy.copy(mech)
    out.nasa_high, out.T_mid = np.ascontiguousarray(hi), np.ascontiguousarray(Tm)
    out.name = mech.name + "+2range"
    return out


def with_falloff(mech: "Mechanism", seed: int = 0) -> "Mechanism":
    """The same mechanism with some reactions turned into pressure-dependent (fall-off) reactions:
    every second third-body reaction (they keep their efficiencies for [M]) and three reactions without a third body.
    The listed Arrhenius parameters become the high-pressure limit; the low-pressure limit is drawn so that the reduced
    pressure P_r = k_0 [M]/k_inf spans about 1e-2..1e2 at 1 atm (A_0 = A_inf 10^U(-1.5, 1.5) / C_ref with C_ref the molar
    density at 1 atm and 1200 K, beta_0 = beta_inf - U(0, 1), E_0 = E_inf + U(-3, 3) kcal/mol) -- the fall-off regime, as
    for the real mechanisms' (+M) reactions at atmospheric pressure.  One half Lindemann, one quarter Troe with four and
    one quarter with three parameters (a ~ U(0.3, 0.8), T*** ~ U(50, 500), T* ~ U(800, 3000), T** ~ U(2000, 6000) K)."""
    import copy
    rng = _rng(seed, 901, int(mech.n_reactions))
    tb = [int(j) for j in mech.tb_reaction[::2]]
    plain = [j for j in range(mech.n_reactions) if j not in set(int(x) for x in mech.tb_reaction)][:3]
    pick = np.array(sorted(tb + plain), dtype=np.int32)
    n = len(pick)
    c_ref = P_ATM / (_RU * 1200.0)
    low = np.stack([mech.arr_A[pick] * 10.0 ** rng.uniform(-1.5, 1.5, size=n) / c_ref,
                    mech.arr_beta[pick] - rng.uniform(0.0, 1.0, size=n),
                    mech.arr_E[pick] + rng.uniform(-3000.0, 3000.0, size=n)], axis=1)
    troe = np.full((n, 4), np.nan)
    for i in range(n):
        if i % 2 == 1:
            troe[i] = (rng.uniform(0.3, 0.8), rng.uniform(50.0, 500.0), rng.uniform(800.0, 3000.0),
                       rng.uniform(2000.0, 6000.0) if i % 4 == 1 else np.inf)
    out = copy.copy(mech)
    out.fo_reaction, out.fo_low, out.fo_troe = pick, np.ascontiguousarray(low), np.ascontiguousarray(troe)
    out.name = mech.name + "+falloff"
    return out


def toy_mechanism(K, reactions, W=None, nasa=None, third_body=None, name="toy") -> Mechanism:
    """Hand-built mechanism for closed-form tests.

    reactions: list of (reactants {k: nu}, products {k: nu}, A, beta, E_cal_per_mol)
    third_body: dict reaction_index -> {k: alpha}
    """
    W = np.ones(K) * 10.0 if W is None else np.asarray(W, dtype=np.float64)
    if nasa is None:
        nasa = np.zeros((K, 7))
        nasa[:, 0] = 3.5
    reac_ptr, reac_sp, reac_nu, prod_ptr, prod_sp, prod_nu = [0], [], [], [0], [], []
    A, b, E = [], [], []
    for (re, pr, a_, b_, e_) in reactions:
        for k in sorted(re):
            reac_sp.append(k)
            reac_nu.append(re[k])
        reac_ptr.append(len(reac_sp))
        for k in sorted(pr):
            prod_sp.append(k)
            prod_nu.append(pr[k])
        prod_ptr.append(len(prod_sp))
        A.append(a_)
        b.append(b_)
        E.append(e_)
    tb_reaction, tb_ptr, tb_sp, tb_eff = [], [0], [], []
    for j in sorted(third_body or {}):
        tb_reaction.append(j)
        for k in sorted(third_body[j]):
            tb_sp.append(k)
            tb_eff.append(third_body[j][k])
        tb_ptr.append(len(tb_sp))
    i32 = lambda x: np.ascontiguousarray(np.array(x, dtype=np.int32))
    f64 = lambda x: np.ascontiguousarray(np.array(x, dtype=np.float64))
    return Mechanism(name=name, elements=(), elem_counts=np.zeros((K, 0), dtype=np.int32),
                     mol_weight=f64(W), nasa=f64(nasa), arr_A=f64(A), arr_beta=f64(b), arr_E=f64(E),
                     reac_ptr=i32(reac_ptr), reac_species=i32(reac_sp), reac_nu=i32(reac_nu),
                     prod_ptr=i32(prod_ptr), prod_species=i32(prod_sp), prod_nu=i32(prod_nu),
                     tb_reaction=i32(tb_reaction), tb_ptr=i32(tb_ptr), tb_species=i32(tb_sp),
                     tb_eff=f64(tb_eff))
