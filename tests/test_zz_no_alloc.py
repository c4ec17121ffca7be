"""ckb_integrate_static (include/ckb.h): the integrate entry point whose scratch lives in a file-scope device array of the
library, for callers that may not allocate device memory.  Its output is compared with the existing path's
(ckb_integrate) on two calls in a row -- the array is shared and keeps the previous call's contents, so the second call
(another batch size, another queue-order mode) shows that nothing stale is used.  Collected last on purpose (the suite runs
with pytest -x).  Passes alone in a fresh process and after the other tests.
"""
import numpy as np
import pytest

from paper_1309_2710_b200 import synth

pytestmark = pytest.mark.gpu

RTOL, ATOL = 1e-8, 1e-12
TOL_Y, TOL_T, Y_CUT = 1e-6, 1e-8, 1e-12          # the parity bar of tests/test_gpu_parity.py


def _both(cfg, N, variant):
    import torch
    from paper_1309_2710_b200 import binding
    spec = synth.CONFIGS[cfg]
    mech = synth.make_mechanism(cfg)
    states, p = synth.make_states(cfg, N)
    m = binding.mech_load(mech)
    out = {}
    for name, fn in (("existing", binding.integrate), ("static", binding.integrate_static)):
        dev = torch.from_numpy(states).cuda()
        status = torch.full((N,), -7, dtype=torch.int32, device="cuda")
        stats = torch.full((4, N), -7, dtype=torch.int32, device="cuda")
        fn(m, dev, 1e-6, RTOL, ATOL, spec.method, p=p, variant=variant, status=status, stats=stats)
        torch.cuda.synchronize()
        out[name] = (dev.cpu().numpy(), status.cpu().numpy(), stats.cpu().numpy())
    m.close()
    return out


def _check(out):
    (ya, sa, ta), (yb, sb, tb) = out["existing"], out["static"]
    assert np.isfinite(yb).all() and np.isin(sb, (0, 4)).all()
    assert np.array_equal(sa, sb) and np.array_equal(ta, tb)           # every system integrated once, same decisions
    relT = np.abs(yb[0] - ya[0]) / np.abs(ya[0])
    big = ya[1:] > Y_CUT
    relY = np.where(big, np.abs(yb[1:] - ya[1:]) / np.where(big, ya[1:], 1.0), 0.0)
    assert relT.max() <= TOL_T and relY.max() <= TOL_Y, (relT.max(), relY.max())


def test_static_scratch_entry_matches_existing_path_on_two_calls_in_a_row():
    # call 1: RKCK, 9/38, thread-per-ODE: queue ordered by temperature (order + bins of the static array)
    _check(_both(1, 40000, "thread"))
    # call 2, smaller batch and the other order mode (RKC, cost-proxy keys in the static array as well): stale contents of
    # call 1 beyond [0, N) and in the bins must not matter
    _check(_both(2, 30000, "thread"))
    # and the warp-per-ODE kernels of the 53-species class
    _check(_both(3, 4500, "warp"))


def test_static_scratch_entry_rejects_batches_beyond_its_maximum():
    import torch
    from paper_1309_2710_b200 import binding
    m = binding.mech_load(synth.make_mechanism(0))
    N = binding.STATIC_MAX_BATCH + 1
    dev = torch.ones((m.K + 1, N), dtype=torch.float64, device="cuda")
    before = dev.clone()
    with pytest.raises(binding.CkbError) as e:
        binding.integrate_static(m, dev, 1e-6, RTOL, ATOL, "rkck", p=synth.P_ATM)
    assert e.value.code == binding.ECAPACITY and "CKB_STATIC_MAX_BATCH" in str(e.value)
    torch.cuda.synchronize()
    assert torch.equal(dev, before)                                      # nothing was launched
    m.close()
