"""Thread-per-ODE for mechanisms with more than 16 unknowns (csrc/ckb_thread.cuh; BASELINE.json configs[3]:
"run with the warp-per-ODE and thread-per-ODE variants"; the paper's own mapping).

The element-wise parity cases on configs[3] / configs[4] sit in tests/test_gpu_parity.py (variant "thread"); here: the
lane-refill queue with more systems than resident lanes, agreement with the warp-per-ODE kernels system by system, both
closures, two-range thermo and fall-off, irregular reaction slots (a species twice on one side / on both sides).
"""
import numpy as np
import pytest

from paper_1309_2710_b200 import synth
from test_gpu_parity import ATOL, RTOL, _compare, _oracle, _run_gpu

pytestmark = pytest.mark.gpu


def test_thread_large_queue_refill_matches_warp_and_oracle():
    """More systems than the 148 x 256 resident lanes: refill from the queue, cost-proxy order; every system agrees with the
    warp-per-ODE result (same decisions, round-off only), a sample with the oracle one by one."""
    import torch
    from paper_1309_2710_b200 import binding
    cfg, N = 3, 45000
    mech = synth.make_mechanism(cfg)
    states, p = synth.make_states(cfg, N)
    m = binding.mech_load(mech)
    outs = {}
    for variant in ("thread", "warp"):
        dev = torch.from_numpy(states).cuda()
        stats = torch.zeros((4, N), dtype=torch.int32, device="cuda")
        status = torch.full((N,), -1, dtype=torch.int32, device="cuda")
        binding.integrate(m, dev, 1e-6, RTOL, ATOL, "rkc", p=p, variant=variant, status=status, stats=stats)
        torch.cuda.synchronize()
        outs[variant] = (dev.cpu().numpy(), status.cpu().numpy(), stats.cpu().numpy())
        assert np.isin(outs[variant][1], (0, 4)).all()
    m.close()
    a, b = outs["thread"], outs["warp"]
    same = (a[2] == b[2]).all(axis=0) & (a[1] == b[1])
    assert same.mean() > 0.998, same.mean()
    assert (np.abs(a[0][0] - b[0][0])[same] <= 1e-8 * np.abs(b[0][0])[same]).all()
    pick = np.random.default_rng(11).choice(N, size=96, replace=False)
    ora = _oracle(mech, np.ascontiguousarray(states[:, pick]), p, 1e-6, "rkc")
    _compare((a[0][:, pick], a[1][pick], a[2][:, pick]), ora, max_flip_frac=0.03)


@pytest.mark.parametrize("method", ["rkck", "rkc"])
def test_thread_large_constant_volume(method):
    import torch
    import oracle
    from paper_1309_2710_b200 import binding
    cfg, N = 3, 200
    mech = synth.make_mechanism(cfg)
    states, p = synth.make_states(cfg, N)
    rho = synth.make_densities(mech, states, p)
    om = oracle.OracleMech(mech)
    ora = om.integrate(states, 0.0, 1e-6, RTOL, ATOL, method, pressure=rho, cv=True)
    m = binding.mech_load(mech)
    dev = torch.from_numpy(states).cuda()
    stats = torch.zeros((4, N), dtype=torch.int32, device="cuda")
    status = torch.full((N,), -1, dtype=torch.int32, device="cuda")
    binding.integrate_cv(m, dev, 1e-6, RTOL, ATOL, method, pressure=torch.from_numpy(rho).cuda(), variant="thread",
                         status=status, stats=stats)
    torch.cuda.synchronize()
    _compare((dev.cpu().numpy(), status.cpu().numpy(), stats.cpu().numpy()), ora)
    # f(y) at constant volume
    ref = np.stack([om.rhs(states[:, i].copy(), rho[i], cv=True) for i in range(64)], axis=1)
    out = binding.rhs_cv(m, torch.from_numpy(states[:, :64].copy()).cuda(), pressure=torch.from_numpy(rho[:64].copy()).cuda(),
                         variant="thread").cpu().numpy()
    scale = np.abs(ref).max(axis=1, keepdims=True)
    assert (np.abs(out - ref) <= 1e-11 * scale + 1e-13 * np.abs(ref)).all()
    m.close()


def test_thread_large_two_range_thermo_and_falloff():
    """R30 / R31 on the thread-per-ODE path: f(y) over four decades of pressure and an integration."""
    import torch
    import oracle
    from paper_1309_2710_b200 import binding
    cfg, N = 3, 160
    spec = synth.CONFIGS[cfg]
    mech = synth.with_falloff(synth.with_two_range_thermo(synth.make_mechanism(cfg), spec.T_range))
    states, p = synth.make_states(cfg, N)
    om = oracle.OracleMech(mech)
    m = binding.mech_load(mech)
    for pf in (0.01, 1.0, 100.0):
        ref = np.stack([om.rhs(states[:, i].copy(), p * pf) for i in range(64)], axis=1)
        out = binding.rhs(m, torch.from_numpy(states[:, :64].copy()).cuda(), p=p * pf, variant="thread").cpu().numpy()
        scale = np.abs(ref).max(axis=1, keepdims=True)
        assert (np.abs(out - ref) <= 1e-11 * scale + 1e-13 * np.abs(ref)).all(), pf
    m.close()
    ora = _oracle(mech, states, p, 1e-6, "rkc")
    gpu = _run_gpu(mech, states, p, 1e-6, "rkc", variant="thread")
    _compare(gpu, ora, max_flip_frac=0.05)


def test_thread_large_irregular_slots():
    """A mechanism of 20 species whose reactions repeat a species on one side (2A -> B + C, A + B -> 2C, 3A -> ...), carry
    a species on both sides (A + B -> A + C) or have an empty product... : the irregular class of the slot stream."""
    import torch
    import oracle
    from paper_1309_2710_b200 import binding
    K = 20
    rng = np.random.default_rng(3)
    rx = []
    for i in range(30):
        a, b, c, d = rng.choice(K, size=4, replace=False)
        kind = i % 5
        a, b, c, d = int(a), int(b), int(c), int(d)
        if kind == 0:
            reac, prod = {a: 2}, {b: 1, c: 1}
        elif kind == 1:
            reac, prod = {a: 1, b: 1}, {c: 2}
        elif kind == 2:
            reac, prod = {a: 1, b: 1}, {a: 1, c: 1}
        elif kind == 3:
            reac, prod = {a: 3}, {b: 1, c: 2}
        else:
            reac, prod = {a: 1, b: 1}, {c: 1, d: 1}
        A = 10.0 ** rng.uniform(3, 7)
        rx.append((reac, prod, A, rng.uniform(-1, 1), rng.uniform(0, 2e4)))
        rx.append((prod, reac, A * 10.0 ** rng.uniform(-2, 0), rng.uniform(-1, 1), rng.uniform(0, 2e4)))
    tb = {4: {0: 2.5, 3: 0.4}, 5: {0: 2.5, 3: 0.4}, 18: {7: 1.7}}
    nasa = np.zeros((K, 7))
    nasa[:, 0] = rng.uniform(3.0, 5.0, K)
    nasa[:, 1] = rng.uniform(0.0, 1e-3, K)
    nasa[:, 5] = rng.uniform(-3e3, 3e3, K)          # distinct enthalpies: dT/dt is not a cancellation residue
    mech = synth.toy_mechanism(K, rx, W=rng.uniform(2.0, 40.0, K), nasa=nasa, third_body=tb, name="irregular20")
    N = 128
    T = rng.uniform(900, 1800, N)
    Y = rng.dirichlet(np.ones(K), size=N).T
    states = np.ascontiguousarray(np.vstack([T[None, :], Y]))
    p = 1.01325e6
    om = oracle.OracleMech(mech)
    m = binding.mech_load(mech)
    ref = np.stack([om.rhs(states[:, i].copy(), p) for i in range(N)], axis=1)
    for v in ("thread", "warp"):
        out = binding.rhs(m, torch.from_numpy(states).cuda(), p=p, variant=v).cpu().numpy()
        scale = np.abs(ref).max(axis=1, keepdims=True)
        assert (np.abs(out - ref) <= 1e-11 * scale + 1e-13 * np.abs(ref)).all(), v
    m.close()
    for method in ("rkck", "rkc"):
        _compare(_run_gpu(mech, states, p, 1e-5, method, variant="thread"), _oracle(mech, states, p, 1e-5, method),
                 max_flip_frac=0.02)
