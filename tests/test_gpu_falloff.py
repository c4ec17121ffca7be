"""Fall-off reactions (reading R31) on the GPU: mechanisms loaded with ckb_mech_load3 against
the oracle with ora_mech_set_falloff on the same seeded inputs, to the bar of tests/test_gpu_parity.py; plus the
Lindemann closed form through ckb_rhs (no oracle involved).

Inputs: the configs' synthetic mechanisms with every second third-body reaction and three plain reactions turned into
fall-off reactions in the fall-off regime at 1 atm (synth.with_falloff: half Lindemann, half Troe)."""
import numpy as np
import pytest

from paper_1309_2710_b200 import synth
from test_gpu_parity import _compare, _compare_tight, _oracle, _run_gpu

pytestmark = pytest.mark.gpu

RU, RC = 8.314462618e7, 1.98720425864


def test_recipe_is_in_the_falloff_regime():
    import oracle
    mech = synth.with_falloff(synth.make_mechanism(2))
    assert len(mech.fo_reaction) >= 5 and np.isnan(mech.fo_troe[:, 0]).any() and np.isfinite(mech.fo_troe[:, 0]).any()
    assert np.isinf(mech.fo_troe[:, 3]).any()
    states, p = synth.make_states(2, 8)
    a, b = oracle.OracleMech(mech), oracle.OracleMech(synth.make_mechanism(2))
    fa = np.stack([a.rhs(states[:, i].copy(), p) for i in range(8)])
    fb = np.stack([b.rhs(states[:, i].copy(), p) for i in range(8)])
    assert not np.allclose(fa, fb, rtol=1e-2)


def test_lindemann_closed_form_on_gpu():
    """A (+M) -> B, all efficiencies 1: at [M] = k_inf/k_0 the effective coefficient is k_inf/2, at any [M] it is
    k_inf k_0 [M] / (k_inf + k_0 [M]) -- checked through ckb_rhs on every mapping that holds 3 species."""
    import torch
    from paper_1309_2710_b200 import binding
    A_INF, B_INF, E_INF, A_0, B_0, E_0 = 3.0e10, 0.5, 9000.0, 4.0e16, -1.2, 3000.0
    W = [20.0, 20.0, 30.0]
    mech = synth.toy_mechanism(3, [({0: 1}, {1: 1}, A_INF, B_INF, E_INF)], W=W)
    mech.fo_reaction = np.array([0], dtype=np.int32)
    mech.fo_low = np.array([[A_0, B_0, E_0]])
    mech.fo_troe = np.full((1, 4), np.nan)
    k = lambda A, b, E, T: A * T ** b * np.exp(-E / (RC * T))
    N = 40
    T = np.linspace(800.0, 1600.0, N)
    kinf, k0 = k(A_INF, B_INF, E_INF, T), k(A_0, B_0, E_0, T)
    M = (kinf / k0) * np.where(np.arange(N) % 2 == 0, 1.0, 10.0 ** np.linspace(-3, 3, N))
    states = np.stack([T, np.full(N, 0.3), np.full(N, 0.2), np.full(N, 0.5)])
    pressure = M * RU * T
    want = kinf * k0 * M / (kinf + k0 * M)
    assert np.allclose(want[::2], kinf[::2] / 2.0, rtol=1e-14)
    m = binding.mech_load(mech)
    st, pr = torch.from_numpy(states).cuda(), torch.from_numpy(pressure).cuda()
    for v in ("thread", "warp", "sub8", "sub4", "sub2", "gen"):
        if v == "gen":
            m.specialize()
            v = "thread"
        f = binding.rhs(m, st, pressure=pr, variant=v).cpu().numpy()
        assert np.allclose(-f[1] / 0.3, want, rtol=1e-12, atol=0), v
        assert np.allclose(f[2], -f[1], rtol=1e-13, atol=0)
    m.close()


def test_source_term_parity_falloff():
    import torch
    import oracle
    from paper_1309_2710_b200 import binding
    for cfg, variants in ((0, ("thread", "warp", "sub8", "sub2", "sub4", "gen")), (2, ("thread", "sub16", "sub4", "gen")),
                          (3, ("warp", "sub8", "sub16")), (4, ("warp", "sub8"))):
        mech = synth.with_falloff(synth.make_mechanism(cfg))
        om = oracle.OracleMech(mech)
        states, p = synth.make_states(cfg, 70)
        pressure = p * 10.0 ** np.linspace(-2.0, 2.0, 70)                       # across the fall-off curve
        ref = np.stack([om.rhs(states[:, i].copy(), pressure[i]) for i in range(70)], axis=1)
        m = binding.mech_load(mech)
        st, pr = torch.from_numpy(states).cuda(), torch.from_numpy(pressure).cuda()
        for v in variants:
            if v == "gen":
                m.specialize()
                v = "thread"
            out = binding.rhs(m, st, pressure=pr, variant=v).cpu().numpy()
            scale = np.abs(ref).max(axis=1, keepdims=True)
            assert (np.abs(out - ref) <= 1e-11 * scale + 1e-13 * np.abs(ref)).all(), (cfg, v)
        m.close()


@pytest.mark.parametrize("cfg,N,method,variant", [
    (0, 1024, "rkck", "auto"), (1, 1500, "rkck", "thread"), (1, 1500, "rkck", "gen"), (0, 700, "rkck", "sub4"),
    (2, 1024, "rkc", "thread"), (2, 1024, "rkc", "gen"), (2, 500, "rkc", "sub4"), (2, 300, "rkc", "warp"),
    (3, 192, "rkc", "warp"), (3, 96, "rkc", "sub16"), (4, 64, "rkc", "warp"),
])
def test_parity_falloff(cfg, N, method, variant):
    mech = synth.with_falloff(synth.make_mechanism(cfg))
    states, p = synth.make_states(cfg, N)
    ora = _oracle(mech, states, p, 1e-6, method)
    gpu = _run_gpu(mech, states, p, 1e-6, method, variant=variant, ld=N + 5)
    # The fall-off mechanisms make the RKC controller reject steps (0.9 rejections per system on 13/54, 3.4 on 111/1566,
    # against none without fall-off): accept/reject and stage-count decisions near their thresholds are round-off
    # sensitive (R28: where decision parity stops being defined).  The yardstick is the ORACLE ITSELF on
    # inputs perturbed by one ulp: it takes different decisions on 14 of 1024 (13/54) and 7 of 64 (111/1566) systems; the
    # CUDA path differs from it on 17 and 7.  So the CUDA path may flip on at most twice as many systems as the oracle
    # does against itself (+2) -- each still held to the flipped-system bound, every other system to the north_star
    # bound with identical decisions.
    flips = 2e-3
    if method == "rkc":
        pert = states.copy()
        pert[1:] = np.nextafter(pert[1:], 2.0)
        ora2 = _oracle(mech, pert, p, 1e-6, method)
        self_flips = int((~((ora2[2] == ora[2]).all(axis=0) & (ora2[1] == ora[1]))).sum())
        flips = (2 * self_flips + 2) / N
    if flips > 0.01:
        # more than 1 % of the systems may flip (111/1566: the oracle flips on 7 of 64 against itself): the flip count is
        # then no assertion at all -- instead every system of a sample must end as close to the truth (an oracle run at
        # rtol 1e-11) as the oracle's own result does, whatever its decisions; systems with identical
        # decisions still meet the north_star bound
        rep = _compare(gpu, ora, max_flip_frac=1.0)
        idx = np.arange(N) if cfg < 4 else np.arange(0, N, 8)   # the truth run of 111/1566 costs ~12 s per system
        rep["against_truth"] = _compare_tight(mech, states, p, 1e-6, method, gpu, ora, idx=idx)
    else:
        rep = _compare(gpu, ora, max_flip_frac=flips)
    print(f"fall-off cfg{cfg} {method} {variant} N={N}: {rep}")
    assert np.isin(ora[1], (0, 4)).all()


def test_falloff_with_two_ranges_at_size_tensor_memory_kernel():
    """Everything at once at size: fall-off + two-range thermo on the 53-species class, N = 4096 (tensor-memory kernel),
    sampled against the oracle."""
    import torch
    from paper_1309_2710_b200 import binding
    mech = synth.with_falloff(synth.with_two_range_thermo(synth.make_mechanism(3), synth.CONFIGS[3].T_range))
    N = 4096
    states, p = synth.make_states(3, N)
    m = binding.mech_load(mech)
    dev = torch.from_numpy(states).cuda()
    stats = torch.zeros((4, N), dtype=torch.int32, device="cuda")
    status = torch.full((N,), -1, dtype=torch.int32, device="cuda")
    binding.integrate(m, dev, 1e-6, 1e-8, 1e-12, "rkc", p=p, status=status, stats=stats)
    torch.cuda.synchronize()
    y, st, stt = dev.cpu().numpy(), status.cpu().numpy(), stats.cpu().numpy()
    m.close()
    assert np.isin(st, (0, 4)).all() and np.abs(y[1:].sum(0) - 1.0).max() < 1e-11
    pick = np.random.default_rng(5).choice(N, size=48, replace=False)
    sub_states = np.ascontiguousarray(states[:, pick])
    ora = _oracle(mech, sub_states, p, 1e-6, "rkc")
    sub = (y[:, pick], st[pick], stt[:, pick])
    _compare(sub, ora, max_flip_frac=1.0)            # identical decisions: north_star bound; flips: judged against the truth
    print("against the truth:", _compare_tight(mech, sub_states, p, 1e-6, "rkc", sub, ora, idx=np.arange(0, 48, 3)))
