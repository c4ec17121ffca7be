"""The N > 1 protocol of bench.py on CPU: two gloo ranks shard independent systems (no data-path collective); the only
exchange is the barrier and the max-over-ranks of the per-rank time.  What integrates here is the ORACLE
(there is no GPU on the CPU box and the product has no CPU path): the test covers the sharding, the barrier and the
reduction of the timing, not the CUDA kernels -- those have no inter-rank step at all ("replicas only")."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys, json
    import numpy as np
    import torch, torch.distributed as dist
    sys.path.insert(0, %r)
    import oracle
    from paper_1309_2710_b200 import synth
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    N = 64                                   # systems per rank: weak scaling, every rank its own batch
    mech = synth.make_mechanism(0)
    states, p = synth.make_states(0, N * world)
    mine = states[:, rank * N:(rank + 1) * N]
    out, status, stats = oracle.OracleMech(mech).integrate(mine, p, 1e-6, 1e-8, 1e-12, "rkck", nthreads=1)
    t = torch.tensor([1.0 + rank], dtype=torch.float64)     # stand-in for the per-rank device time
    dist.barrier()
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    gathered = [torch.zeros(out.shape, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(gathered, torch.from_numpy(out))        # test-only: to compare with the unsharded run
    if rank == 0:
        full, _, _ = oracle.OracleMech(mech).integrate(states, p, 1e-6, 1e-8, 1e-12, "rkck", nthreads=1)
        same = all(np.array_equal(g.numpy(), full[:, r * N:(r + 1) * N]) for r, g in enumerate(gathered))
        print(json.dumps({"max_time": t.item(), "world": world, "sharded_equals_full": bool(same),
                          "value": N * world / t.item()}))
    dist.destroy_process_group()
""")


def test_two_gloo_ranks_shard_independent_systems(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", str(port), str(script)],
                       capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    import json
    line = [l for l in r.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["world"] == 2 and d["max_time"] == 2.0 and d["sharded_equals_full"]
    assert d["value"] == 64.0                 # (N * world) / max-over-ranks time


def test_bench_reference_arm_only_rank0_prints():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                        "--warmup", "0"], capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0 and r.stdout.strip() == ""
