"""Two-range NASA thermodynamics (reading R30) on the GPU: mechanisms loaded with
ckb_mech_load2 against the oracle with ora_mech_set_thermo2, on the same seeded inputs, to the bar of
tests/test_gpu_parity.py; plus enthalpy conservation at size (holds at any batch size, no oracle involved).

Inputs: the configs' synthetic mechanisms with a high range drawn beside the low one and every species' T_mid inside the
config's temperature range (synth.with_two_range_thermo), so that batches straddle the switch and systems cross it."""
import numpy as np
import pytest

from paper_1309_2710_b200 import synth
from test_gpu_parity import ATOL, RTOL, _compare, _oracle, _run_gpu

pytestmark = pytest.mark.gpu

RU = 8.314462618e7


def _two(cfg):
    return synth.with_two_range_thermo(synth.make_mechanism(cfg), synth.CONFIGS[cfg].T_range)


def test_source_term_parity_two_ranges():
    """ckb_rhs / ckb_rhs_cv on every mapping, states on both sides of (and between) the species' T_mid."""
    import torch
    import oracle
    from paper_1309_2710_b200 import binding
    for cfg, variants in ((0, ("thread", "warp", "sub8", "sub2", "sub4", "gen")), (2, ("thread", "sub16", "sub4", "gen")),
                          (3, ("warp", "sub8", "sub16")), (4, ("warp", "sub8"))):
        mech = _two(cfg)
        om = oracle.OracleMech(mech)
        states, p = synth.make_states(cfg, 70)
        frac_hi = (states[0][None, :] > mech.T_mid[:, None]).mean()
        assert 0.15 < frac_hi < 0.85
        ref = np.stack([om.rhs(states[:, i].copy(), p) for i in range(70)], axis=1)
        one = oracle.OracleMech(synth.make_mechanism(cfg))
        ref_one = np.stack([one.rhs(states[:, i].copy(), p) for i in range(70)], axis=1)
        assert not np.allclose(ref[0], ref_one[0], rtol=1e-3)                  # the second range matters here
        rho = synth.make_densities(mech, states, p)
        ref_cv = np.stack([om.rhs(states[:, i].copy(), rho[i], cv=True) for i in range(70)], axis=1)
        m = binding.mech_load(mech)
        st, dn = torch.from_numpy(states).cuda(), torch.from_numpy(rho).cuda()
        for v in variants:
            if v == "gen":
                m.specialize()
                v = "thread"
            for got, want in ((binding.rhs(m, st, p=p, variant=v), ref), (binding.rhs_cv(m, st, pressure=dn, variant=v), ref_cv)):
                got = got.cpu().numpy()
                scale = np.abs(want).max(axis=1, keepdims=True)
                assert (np.abs(got - want) <= 1e-11 * scale + 1e-13 * np.abs(want)).all(), (cfg, v)
        m.close()


@pytest.mark.parametrize("cfg,N,method,variant", [
    (0, 1024, "rkck", "auto"), (1, 1500, "rkck", "thread"), (1, 1500, "rkck", "gen"), (0, 700, "rkck", "sub4"),
    (2, 1024, "rkc", "thread"), (2, 1024, "rkc", "gen"), (2, 500, "rkc", "sub4"), (2, 300, "rkc", "warp"),
    (3, 192, "rkc", "warp"), (3, 96, "rkc", "sub16"), (3, 96, "rkck", "warp"), (4, 64, "rkc", "warp"),
])
def test_parity_two_ranges(cfg, N, method, variant):
    mech = _two(cfg)
    states, p = synth.make_states(cfg, N)
    ora = _oracle(mech, states, p, 1e-6, method)
    gpu = _run_gpu(mech, states, p, 1e-6, method, variant=variant, ld=N + 11)
    rep = _compare(gpu, ora)
    print(f"two-range cfg{cfg} {method} {variant} N={N}: {rep}")
    one = _oracle(synth.make_mechanism(cfg), states, p, 1e-6, method)
    assert np.abs(one[0][0] - ora[0][0]).max() > 1e-6 * np.abs(ora[0][0]).max()    # not the one-range result


@pytest.mark.parametrize("cfg,N,method", [(1, 1 << 17, "rkck"), (3, 4096, "rkc")])
def test_enthalpy_conserved_across_the_switch_at_size(cfg, N, method):
    """Adiabatic constant-pressure reactor: specific enthalpy (two-range fits evaluated in numpy) is conserved to the
    accumulated local tolerance although systems cross their species' T_mid; AUTO mapping at this batch size (the
    specialised kernels for cfg 1, the tensor-memory warp-per-ODE kernel for cfg 3)."""
    import torch
    from paper_1309_2710_b200 import binding
    mech = _two(cfg)
    states, p = synth.make_states(cfg, N)
    m = binding.mech_load(mech, specialize=mech.n_species + 1 <= 16)
    dev = torch.from_numpy(states).cuda()
    stats = torch.zeros((4, N), dtype=torch.int32, device="cuda")
    status = torch.full((N,), -1, dtype=torch.int32, device="cuda")
    binding.integrate(m, dev, 1e-6, RTOL, ATOL, method, p=p, status=status, stats=stats)
    torch.cuda.synchronize()
    y, st, stt = dev.cpu().numpy(), status.cpu().numpy(), stats.cpu().numpy()
    m.close()
    assert np.isin(st, (0, 4)).all()

    def h_mass(s_):
        T = s_[0][None, :]
        hi = T > mech.T_mid[:, None]
        a = np.where(hi[:, :, None], mech.nasa_high[:, None, :], mech.nasa[:, None, :])     # [K][N][7]
        h_rt = (a[..., 0] + a[..., 1] * T / 2 + a[..., 2] * T ** 2 / 3 + a[..., 3] * T ** 3 / 4 + a[..., 4] * T ** 4 / 5
                + a[..., 5] / T)
        cp_r = a[..., 0] + a[..., 1] * T + a[..., 2] * T ** 2 + a[..., 3] * T ** 3 + a[..., 4] * T ** 4
        w = mech.mol_weight[:, None]
        return (s_[1:] * RU * T * h_rt / w).sum(0), (s_[1:] * RU * cp_r / w).sum(0)

    (h0, cp0), (h1, _) = h_mass(states), h_mass(y)
    assert (np.abs(h1 - h0) <= 3.0 * RTOL * (stt[1] + 5) * cp0 * states[0]).all()
    crossed = ((states[0][None, :] > mech.T_mid[:, None]) != (y[0][None, :] > mech.T_mid[:, None])).any(axis=0)
    print(f"cfg{cfg}: {int(crossed.sum())} of {N} systems crossed a T_mid")
    assert crossed.sum() >= 1
    pick = np.random.default_rng(7).choice(N, size=48 if cfg == 3 else 1500, replace=False)
    ora = _oracle(mech, np.ascontiguousarray(states[:, pick]), p, 1e-6, method)
    _compare((y[:, pick], st[pick], stt[:, pick]), ora, max_flip_frac=5e-3)


def test_load2_argument_checks():
    import ctypes as C
    from paper_1309_2710_b200 import binding
    mech = _two(0)
    bad = synth.with_two_range_thermo(synth.make_mechanism(0), (1000.0, 1500.0))
    bad.T_mid = bad.T_mid.copy()
    bad.T_mid[3] = np.nan
    with pytest.raises(binding.CkbError):
        binding.mech_load(bad)
    d, keep = binding._make_desc(mech)
    h = C.c_void_p()
    hi = np.ascontiguousarray(mech.nasa_high)
    assert binding.lib().ckb_mech_load2(C.byref(d), C.c_void_p(hi.ctypes.data), None, C.byref(h)) == binding.EINVAL
