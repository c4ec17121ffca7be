"""Constant-volume closure (reading R29) on the GPU: ckb_rhs_cv / ckb_integrate_cv /
ckb_integrate_host_cv against the oracle's ora_rhs_cv / ora_integrate_cv on the same seeded inputs, to the same bar
as the constant-pressure path (tests/test_gpu_parity.py), plus the conservation law the closure exists for (specific
internal energy of an adiabatic constant-volume reactor), which holds at any batch size.

Inputs: the configs' 1 atm initial states, each held at the density it has at 1 atm (synth.make_densities)."""
import numpy as np
import pytest

from paper_1309_2710_b200 import synth
from test_gpu_parity import ATOL, RTOL, _compare

pytestmark = pytest.mark.gpu

RU = 8.314462618e7


def _u_mass(mech, y):
    """u = sum_k Y_k (h_k - Ru T)/W_k from the NASA fits, in numpy (not the oracle's code)."""
    T, Y = y[0], y[1:]
    a = mech.nasa[:, :, None] if y.ndim == 2 else mech.nasa
    h_rt = a[:, 0] + a[:, 1] * T / 2 + a[:, 2] * T ** 2 / 3 + a[:, 3] * T ** 3 / 4 + a[:, 4] * T ** 4 / 5 + a[:, 5] / T
    w = mech.mol_weight[:, None] if y.ndim == 2 else mech.mol_weight
    return (Y * RU * T * (h_rt - 1.0) / w).sum(axis=0)


def _run_gpu_cv(mech, states, rho, dt, method, variant="auto", density=None, rtol=RTOL, atol=ATOL, host=False):
    import torch
    from paper_1309_2710_b200 import binding
    m = binding.mech_load(mech)
    if variant == "gen":
        m.specialize()
        variant = "thread"
    n, N = states.shape
    if host:
        buf = states.copy()
        status = np.full(N, -7, dtype=np.int32)
        stats = np.full((4, N), -7, dtype=np.int32)
        binding.integrate_host_cv(m, buf, dt, rtol, atol, method, p=rho, pressure=density, variant=variant,
                                  status=status, stats=stats)
        m.close()
        return buf, status, stats
    ld = N + 19
    buf = torch.full((n, ld), float("nan"), dtype=torch.float64, device="cuda")
    buf[:, :N] = torch.from_numpy(states).cuda()
    status = torch.full((N,), -7, dtype=torch.int32, device="cuda")
    stats = torch.full((4, N), -7, dtype=torch.int32, device="cuda")
    dn = None if density is None else torch.from_numpy(density).cuda()
    binding.integrate_cv(m, buf, dt, rtol, atol, method, N=N, p=rho, pressure=dn, variant=variant, status=status,
                         stats=stats)
    torch.cuda.synchronize()
    out = buf.cpu().numpy()
    assert np.isnan(out[:, N:]).all()
    m.close()
    return out[:, :N].copy(), status.cpu().numpy(), stats.cpu().numpy()


def _oracle_cv(mech, states, rho, dt, method, density=None, rtol=RTOL, atol=ATOL):
    import oracle
    return oracle.OracleMech(mech).integrate(states, rho, dt, rtol, atol, method, pressure=density, cv=True)


def test_source_term_parity_cv():
    """ckb_rhs_cv against ora_rhs_cv: every mapping variant, every mechanism, per-system densities."""
    import torch
    import oracle
    from paper_1309_2710_b200 import binding
    for cfg, variants in ((0, ("thread", "warp", "sub8", "sub2", "sub4", "gen")), (2, ("thread", "sub16", "sub4", "gen")),
                          (3, ("warp", "sub8", "sub16")), (4, ("warp", "sub8"))):
        mech = synth.make_mechanism(cfg)
        om = oracle.OracleMech(mech)
        states, p = synth.make_states(cfg, 70)
        rho = synth.make_densities(mech, states, p) * np.linspace(0.5, 2.0, 70)
        ref = np.stack([om.rhs(states[:, i].copy(), rho[i], cv=True) for i in range(70)], axis=1)
        ref_p = np.stack([om.rhs(states[:, i].copy(), p) for i in range(70)], axis=1)
        assert not np.allclose(ref[0], ref_p[0], rtol=1e-3)          # the closure matters on these inputs
        m = binding.mech_load(mech)
        st, dn = torch.from_numpy(states).cuda(), torch.from_numpy(rho).cuda()
        for v in variants:
            if v == "gen":
                m.specialize()
                v = "thread"
            out = binding.rhs_cv(m, st, pressure=dn, variant=v).cpu().numpy()
            scale = np.abs(ref).max(axis=1, keepdims=True)
            assert (np.abs(out - ref) <= 1e-11 * scale + 1e-13 * np.abs(ref)).all(), (cfg, v)
            # the constant-pressure entry on the same handle is unaffected by the closure flag of the last launch
            out_p = binding.rhs(m, st, p=p, variant=v).cpu().numpy()
            scale_p = np.abs(ref_p).max(axis=1, keepdims=True)
            assert (np.abs(out_p - ref_p) <= 1e-11 * scale_p + 1e-13 * np.abs(ref_p)).all(), (cfg, v)
        m.close()


@pytest.mark.parametrize("cfg,N,method,variant", [
    (0, 1024, "rkck", "auto"), (1, 1500, "rkck", "thread"), (1, 1500, "rkck", "gen"), (0, 700, "rkck", "sub4"),
    (0, 512, "rkc", "gen"), (2, 1024, "rkc", "thread"), (2, 1024, "rkc", "gen"), (2, 500, "rkc", "sub4"),
    (2, 300, "rkc", "warp"), (2, 512, "rkck", "sub2"), (3, 192, "rkc", "warp"), (3, 96, "rkc", "sub16"),
    (3, 96, "rkck", "warp"), (4, 64, "rkc", "warp"), (4, 40, "rkc", "sub8"),
])
def test_parity_cv(cfg, N, method, variant):
    mech = synth.make_mechanism(cfg)
    states, p = synth.make_states(cfg, N)
    rho = synth.make_densities(mech, states, p)
    ora = _oracle_cv(mech, states, 0.0, 1e-6, method, density=rho)
    gpu = _run_gpu_cv(mech, states, 0.0, 1e-6, method, variant=variant, density=rho)
    rep = _compare(gpu, ora)
    print(f"cv cfg{cfg} {method} {variant} N={N}: {rep}")
    assert np.isin(ora[1], (0, 4)).all()
    # not the constant-pressure result: the two closures differ by far more than the parity bar on these inputs
    import oracle
    yp = oracle.OracleMech(mech).integrate(states, p, 1e-6, RTOL, ATOL, method)[0]
    assert np.abs(yp[0] - ora[0][0]).max() > 1e-6 * np.abs(yp[0]).max()


def test_uniform_density_and_host_entry():
    mech = synth.make_mechanism(1)
    states, p = synth.make_states(1, 3000)
    rho_u = float(np.median(synth.make_densities(mech, states, p)))
    ora = _oracle_cv(mech, states, rho_u, 1e-6, "rkck")
    _compare(_run_gpu_cv(mech, states, rho_u, 1e-6, "rkck"), ora)
    _compare(_run_gpu_cv(mech, states, rho_u, 1e-6, "rkck", host=True), ora)
    rho = synth.make_densities(mech, states, p)
    ora = _oracle_cv(mech, states, 0.0, 1e-6, "rkck", density=rho)
    _compare(_run_gpu_cv(mech, states, 0.0, 1e-6, "rkck", density=rho, host=True), ora)


def test_host_entry_cv_pipelined_chunks():
    """N >= 65536 RKCK goes through ckb_integrate_host_cv in chunks on internal streams; sampled against the oracle."""
    mech = synth.make_mechanism(1)
    N = 70001
    states, p = synth.make_states(1, N)
    rho = synth.make_densities(mech, states, p)
    got, st, stats = _run_gpu_cv(mech, states, 0.0, 1e-6, "rkck", density=rho, host=True)
    assert (st == 0).all() and (stats[0] > 0).all()
    idx = np.random.default_rng(5).choice(N, 1200, replace=False)
    ora = _oracle_cv(mech, states[:, idx].copy(), 0.0, 1e-6, "rkck", density=rho[idx].copy())
    _compare((got[:, idx], st[idx], stats[:, idx]), ora)


@pytest.mark.parametrize("cfg,N,method", [(1, 1 << 17, "rkck"), (2, 1 << 15, "rkc"), (3, 2048, "rkc")])
def test_internal_energy_conserved_at_size(cfg, N, method):
    """Property that holds at any size (no oracle involved): an adiabatic constant-volume reactor keeps its specific
    internal energy; the integrators keep this nonlinear invariant to the accumulated local tolerance (accepted
    steps x rtol, relative to c_v T).  Also sum Y = 1 (linear: to round-off).  AUTO mapping, i.e. the launch configuration a user gets at this batch size."""
    mech = synth.make_mechanism(cfg)
    states, p = synth.make_states(cfg, N)
    rho = synth.make_densities(mech, states, p)
    got, st, stats = _run_gpu_cv(mech, states, 0.0, 1e-6, method, density=rho)
    assert np.isin(st, (0, 4)).all()
    u0, u1 = _u_mass(mech, states), _u_mass(mech, got)
    a = mech.nasa[:, :, None]
    T = states[0]
    cv_mass = (states[1:] * RU * (a[:, 0] + a[:, 1] * T + a[:, 2] * T ** 2 + a[:, 3] * T ** 3 + a[:, 4] * T ** 4 - 1.0)
               / mech.mol_weight[:, None]).sum(axis=0)
    assert (np.abs(u1 - u0) <= 3.0 * RTOL * (stats[1] + 5) * cv_mass * T).all()
    assert np.abs(got[1:].sum(axis=0) - 1.0).max() < 1e-11
    assert np.abs(got[0] - states[0]).max() > 0.05            # the batch does react


def test_cv_argument_checks():
    import torch
    from paper_1309_2710_b200 import binding
    mech = synth.make_mechanism(0)
    m = binding.mech_load(mech)
    st = torch.from_numpy(synth.make_states(0, 8)[0]).cuda()
    with pytest.raises(binding.CkbError):
        binding.integrate_cv(m, st, 1e-6, 1e-8, 1e-12, "rkck", p=0.0)          # no density given
    with pytest.raises(binding.CkbError):
        binding.rhs_cv(m, st, p=-1.0)
    m.close()


@pytest.mark.parametrize("cfg,N,n_sample,specialize", [(2, 40000, 400, False), (2, 120000, 400, True), (1, 1 << 19, 2000, True),
                                                       (3, 4096, 64, False)])
def test_cv_at_size_sampled(cfg, N, n_sample, specialize):
    """Constant volume in the launch configurations a user gets at size (AUTO: 4 lanes per system with the cost-proxy
    queue order of the cv kernels at mid sizes, the specialised thread-per-ODE kernels at full size, the tensor-memory
    warp-per-ODE kernel on the 53-species class): sampled systems against the oracle one by one."""
    import torch
    from paper_1309_2710_b200 import binding
    spec = synth.CONFIGS[cfg]
    mech = synth.make_mechanism(cfg)
    states, p = synth.make_states(cfg, N)
    rho = synth.make_densities(mech, states, p)
    m = binding.mech_load(mech, specialize=specialize)
    dev = torch.from_numpy(states).cuda()
    stats = torch.zeros((4, N), dtype=torch.int32, device="cuda")
    status = torch.full((N,), -1, dtype=torch.int32, device="cuda")
    binding.integrate_cv(m, dev, 1e-6, RTOL, ATOL, spec.method, pressure=torch.from_numpy(rho).cuda(), status=status,
                         stats=stats)
    torch.cuda.synchronize()
    y, st, stt = dev.cpu().numpy(), status.cpu().numpy(), stats.cpu().numpy()
    m.close()
    assert np.isin(st, (0, 4)).all() and np.isfinite(y).all() and (stt[0] > 0).all()
    pick = np.random.default_rng(23 + cfg).choice(N, size=n_sample, replace=False)
    ora = _oracle_cv(mech, np.ascontiguousarray(states[:, pick]), 0.0, 1e-6, spec.method, density=rho[pick].copy())
    rep = _compare((y[:, pick], st[pick], stt[:, pick]), ora, max_flip_frac=5e-3)
    print(f"cv at size cfg{cfg} N={N}: {rep}")


@pytest.mark.parametrize("cfg,N,dt,rtol,atol", [(1, 2048, 1e-8, 1e-10, 1e-40), (2, 1024, 1e-6, 1e-6, 1e-10),
                                               (3, 128, 1e-6, 1e-6, 1e-10)])
def test_parity_cv_paper_settings(cfg, N, dt, rtol, atol):
    """The paper's own tolerances and global steps at constant volume."""
    spec = synth.CONFIGS[cfg]
    mech = synth.make_mechanism(cfg)
    states, p = synth.make_states(cfg, N)
    rho = synth.make_densities(mech, states, p)
    ora = _oracle_cv(mech, states, 0.0, dt, spec.method, density=rho, rtol=rtol, atol=atol)
    gpu = _run_gpu_cv(mech, states, 0.0, dt, spec.method, density=rho, rtol=rtol, atol=atol)
    _compare(gpu, ora, max_flip_frac=5e-3, rtol=rtol, atol=atol)
