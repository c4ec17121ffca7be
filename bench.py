#!/usr/bin/env python
"""bench.py -- ODE systems integrated per second for one global step dt (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C] [--n N] [--no-extra]

A "step" is one pass of the whole hot path over one batch: ckb_integrate() advances all N systems of the
workload from their (seeded, synthetic) initial states over one global step dt -- load state, adaptive
sub-stepping (RKCK or RKC with its spectral-radius estimate), source term f(y) fused in, store state.
Headline workload = BASELINE.json configs[1] (9/38 synthetic mechanism, RKCK, N = 2^19, dt = 1e-6 s,
rtol 1e-8, atol 1e-12); the other configs are measured too and reported under "configs" (configs[3] at
N = 2^17 is the one north_star's roofline target is stated on).

Timing: every step restarts from the same initial states (device-to-device copy, not timed), L2 is flushed
(256 MiB write, not timed), then CUDA events on the launching stream bracket the ckb_integrate launch;
`value` = N * K / sum of the K event durations (max over ranks).  `e2e` is the same step through
ckb_integrate_host with pinned HOST buffers (H2D + kernel + D2H inside the timed region).
`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1309_2710_b200 import synth  # noqa: E402

RTOL, ATOL = 1e-8, 1e-12
METRIC = "ODE systems integrated/sec per global dt"
UNIT = "ODEs/s"
# nominal FP64 FMA peak of a B200: 148 SMs x 64 FP64 FMA lanes/clk x 2 flop x 1.965 GHz
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
HEADLINE_N = {0: 1024, 1: 2 ** 19, 2: 2 ** 18, 3: 2 ** 17, 4: 2 ** 16}


def parse():
    global RTOL, ATOL
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--n", type=int, default=0, help="override the batch size N")
    ap.add_argument("--dt", type=float, default=0.0)
    ap.add_argument("--rtol", type=float, default=RTOL, help="relative tolerance (default: BASELINE.json's 1e-8)")
    ap.add_argument("--atol", type=float, default=ATOL, help="absolute tolerance (default: BASELINE.json's 1e-12)")
    ap.add_argument("--variant", default="auto")
    ap.add_argument("--ordering", default="shuffled", choices=["shuffled", "similar"])
    ap.add_argument("--no-specialize", action="store_true",
                    help="keep the table-driven thread-per-ODE kernels (no runtime-generated mechanism code)")
    ap.add_argument("--no-extra", action="store_true", help="skip the other configs, e2e and cpu_baseline")
    ap.add_argument("--f1", action="store_true", help="the config's mechanism with two-range thermo and fall-off reactions (SURVEY 8(f)-f1)")
    ap.add_argument("--cv", action="store_true", help="constant-volume closure (SURVEY 8(f)-f3)")
    ap.add_argument("--sweep", action="store_true", help="also sweep N over the config's N_list")
    args = ap.parse_args()
    RTOL, ATOL = args.rtol, args.atol   # every leg (ours, e2e, oracle) uses the same tolerances
    return args


def workload(cfg, n_override=0, dt=0.0):
    spec = synth.CONFIGS[cfg]
    N = n_override or HEADLINE_N[cfg]
    return spec, N, (dt or spec.dt[0])


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        self.samples, self.reasons, self._stop = [], set(), threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv, self.h = pynvml, pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:  # pragma: no cover
            self.nv = None
            self.max = None
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:  # pragma: no cover
                pass
            time.sleep(0.0005)

    def __enter__(self):
        if self.nv:
            self.t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self.nv:
            self.t.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


class GpuCase:
    """One (config, N, dt, variant) workload resident on the GPU."""

    specialize = True   # class-wide switch (--no-specialize)

    def __init__(self, cfg, N, dt, variant="auto", ordering="shuffled", device=0, cv=False, f1=False):
        import torch
        from paper_1309_2710_b200 import binding
        self.torch, self.binding = torch, binding
        self.spec = synth.CONFIGS[cfg]
        self.cfg, self.N, self.dt, self.variant = cfg, N, dt, variant
        self.mech = synth.make_mechanism(cfg)
        if f1:   # two-range NASA fits and fall-off reactions on the same mechanism (ckb_mech_load3)
            self.mech = synth.with_falloff(synth.with_two_range_thermo(self.mech, self.spec.T_range))
        self.m = binding.mech_load(self.mech)
        # mechanism-specialised thread-per-ODE kernels (ckb_mech_specialize) where the mapping applies; if the
        # runtime compiler is missing the table-driven kernels stay in place and the bench line says so
        self.specialized, self.specialize_error = False, None
        if GpuCase.specialize and self.mech.n_species + 1 <= 16:
            try:
                self.m.specialize()
                self.specialized = True
            except binding.CkbError as e:
                self.specialize_error = str(e)[:200]
        st, self.p = synth.make_states(cfg, N, ordering=ordering)
        # constant-volume closure: the same states, each held at the density it has at 1 atm
        self.cv = cv
        self.density = torch.from_numpy(synth.make_densities(self.mech, st, self.p)).cuda() if cv else None
        self.host0 = st
        self.states0 = torch.from_numpy(st).cuda()
        self.states = torch.empty_like(self.states0)
        self.status = torch.zeros((N,), dtype=torch.int32, device="cuda")
        self.stats = torch.zeros((4, N), dtype=torch.int32, device="cuda")
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def step(self, want_stats=False):
        self.binding.integrate(self.m, self.states, self.dt, RTOL, ATOL, self.spec.method,
                               p=0.0 if self.cv else self.p, pressure=self.density, cv=self.cv,
                               variant=self.variant, status=self.status if want_stats else None,
                               stats=self.stats if want_stats else None)

    def timed_steps(self, K, W):
        """Returns the K per-step kernel durations in ms (CUDA events on the launching stream)."""
        torch = self.torch
        for _ in range(W):
            self.states.copy_(self.states0)
            self.step()
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
        for a, b in ev:
            self.states.copy_(self.states0)
            self.flush.fill_(1)
            a.record()
            self.step()
            b.record()
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in ev]

    def work(self):
        """Per-step work counters (same every step: same inputs): one untimed step with stats on."""
        torch = self.torch
        self.states.copy_(self.states0)
        self.step(want_stats=True)
        torch.cuda.synchronize()
        st = self.stats.cpu().numpy().astype(np.int64)
        status = self.status.cpu().numpy()
        d = st[0].reshape(-1, 32) if self.N % 32 == 0 else None
        out = {"rhs_calls": int(st[0].sum()), "rhs_per_ode_mean": float(st[0].mean()), "rhs_per_ode_max": int(st[0].max()),
               "accepted_mean": float(st[1].mean()), "rejected_mean": float(st[2].mean()),
               "stages_max": int(st[3].max()), "status_nonzero": int((status != 0).sum()),
               "status_sigma": int((status == 4).sum())}
        if d is not None:   # Eq. 40: D = sum d_i / (32 max d_i) per 32 consecutive systems
            D = d.sum(1) / (32.0 * d.max(1))
            out["divergence_D_mean"] = float(D.mean())
            out["divergence_D_hist10"] = [int(x) for x in np.histogram(D, bins=10, range=(0.0, 1.0))[0]]
        return out

    def e2e(self, K, W):
        """ckb_integrate_host on pinned host buffers: H2D + kernel + D2H inside the timed region."""
        torch = self.torch
        n = self.mech.n_species + 1
        host = torch.empty((n, self.N), dtype=torch.float64).pin_memory()
        status = torch.zeros((self.N,), dtype=torch.int32).pin_memory()
        src = torch.from_numpy(self.host0)
        times = []
        for i in range(W + K):
            host.copy_(src)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            self.binding.integrate_host(self.m, host, self.dt, RTOL, ATOL, self.spec.method, p=self.p,
                                        variant=self.variant, status=status)
            t1 = time.perf_counter()
            if i >= W:
                times.append(t1 - t0)
        return times, n * self.N * 8, n * self.N * 8 + 4 * self.N

    def close(self):
        self.m.close()


def measured_traffic(cfg, N, specialised=False):
    """dram__bytes_read.sum + dram__bytes_write.sum of the integrate kernel for this workload, from the committed
    ncu --set full capture (profiles/traffic.json, written from the capture named there), per launch; else None."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(path):
        with open(path) as fh:
            for e in json.load(fh).get("captures", []):
                if e["config"] == cfg and e["N"] == N and bool(e.get("specialised", False)) == bool(specialised):
                    return e["dram_bytes_read"] + e["dram_bytes_write"]
    return None


def north_star_counters():
    """branch uniformity / active lanes of the configs[3] kernels from the committed ncu captures (profiles/north_star.json)"""
    path = os.path.join(ROOT, "profiles", "north_star.json")
    if os.path.exists(path):
        with open(path) as fh:
            return {"ncu": json.load(fh)}
    return {"ncu": None}


def roofline(case, ms, work, peak_tflops, peak_src):
    flops = case.m.flops_per_rhs * work["rhs_calls"]
    ach = flops / (ms * 1e-3) / 1e12
    return {"bound": "alu", "achieved": ach, "peak": peak_tflops, "unit": "TFLOP/s", "frac": ach / peak_tflops,
            "traffic": None if getattr(case, "cv", False) else measured_traffic(case.cfg, case.N, case.specialized), "peak_source": peak_src, "frac_of_nominal": ach / FP64_NOMINAL_TFLOPS,
            "flops_per_rhs": case.m.flops_per_rhs, "rhs_calls_per_launch": work["rhs_calls"],
            "kernel_ms": ms, "hbm_algorithmic_GBps": 2 * 8 * (case.mech.n_species + 1) * case.N / (ms * 1e-3) / 1e9}


def oracle_time(cfg, N, dt, budget_s=15.0, nthreads=0):
    """The oracle as it stands on a bounded sample (first n systems of the same workload)."""
    import oracle
    spec = synth.CONFIGS[cfg]
    mech = synth.make_mechanism(cfg)
    om = oracle.OracleMech(mech)
    states, p = synth.make_states(cfg, N)
    probe = min(N, 256)
    t0 = time.perf_counter()
    om.integrate(states[:, :probe], p, dt, RTOL, ATOL, spec.method, nthreads=nthreads)
    t_probe = time.perf_counter() - t0
    n = int(min(N, max(probe, probe * budget_s / max(t_probe, 1e-6))))
    t0 = time.perf_counter()
    om.integrate(states[:, :n], p, dt, RTOL, ATOL, spec.method, nthreads=nthreads)
    t = time.perf_counter() - t0
    cores = oracle.num_threads() if nthreads <= 0 else nthreads
    return n / t, n, cores, t


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, bounded sample per step (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    spec, N, dt = workload(args.config, args.n, args.dt)
    budget = max(2.0, min(15.0, 120.0 / max(1, args.steps + args.warmup)))
    rates, n_used, cores = [], 0, 0
    for i in range(args.warmup + args.steps):
        r, n_used, cores, _ = oracle_time(args.config, N, dt, budget_s=budget)
        if i >= args.warmup:
            rates.append(r)
    value = float(len(rates) / sum(1.0 / r for r in rates))
    sample = f"first {n_used} of {N} systems of the workload per step, OpenMP over systems"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * N / value, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config}]: {spec.name} species/reactions, {spec.method.upper()}, "
                               f"N={N} per GPU, dt={dt:g} s, rtol={RTOL:g}, atol={ATOL:g}", "N_per_gpu": N, "sample_n": n_used},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_ours(args):
    GpuCase.specialize = not args.no_specialize
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    spec, N, dt = workload(args.config, args.n, args.dt)
    K, W = args.steps, max(args.warmup, 3)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    from paper_1309_2710_b200 import binding
    # roofline denominator: sustained DFMA rate of this GPU (>= 1 s per run, SM clock sampled under that load;
    # 3 runs of ~1.2 s after a warm-up run, the fastest counts)
    with ClockSampler(local) as pclk:
        t_probe = time.perf_counter()
        peak_flops = binding.fp64_probe("dfma", 1 << 23)
        t_probe = time.perf_counter() - t_probe
    probe_info = {"tflops": peak_flops / 1e12, "runs": 4, "seconds_per_run": t_probe / 4.0,
                  "sm_mhz_under_probe": pclk.summary()["sm_mhz"], "reasons": pclk.summary()["reasons"],
                  "frac_of_nominal": peak_flops / 1e12 / FP64_NOMINAL_TFLOPS}
    exp_rate = binding.fp64_probe("exp", 1 << 12)
    # every rank integrates its own N systems (independent problems, no data-path collective): weak scaling
    case = GpuCase(args.config, N, dt, args.variant, args.ordering, local, cv=args.cv, f1=args.f1)
    work = case.work()
    barrier()
    with ClockSampler(local) as clk:
        ms = case.timed_steps(K, W)
    barrier()
    total_ms = float(sum(ms))
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    value = N * world * K / (total_ms * 1e-3)
    ms_step = total_ms / K
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config}]: {spec.name} species/reactions, {spec.method.upper()}, "
                               f"N={N} per GPU, dt={dt:g} s, rtol={RTOL:g}, atol={ATOL:g}",
                   "N_per_gpu": N, "variant": args.variant, "ordering": args.ordering, "f1": args.f1, "cv": args.cv,
                   "specialised": case.specialized, **({"specialise_error": case.specialize_error} if case.specialize_error else {}),
                   "l2": "flushed between timed steps (256 MiB write, untimed)",
                   "restart": "every step restarts from the same initial states (device copy, untimed)"},
        "clocks": clk.summary(),
        # our kernels per ckb_integrate call: integrate_kernel, and for N >= 4096 the queue order (hist, scan, scatter;
        # plus the cost-proxy kernel for thread-per-ODE RKC)
        "gpu_launches": K * (1 + (3 if N >= 4096 else 0) + (1 if (N >= 24576 and spec.method == "rkc" and spec.K + 1 <= 16 and args.variant in ("auto", "thread", "sub4", "sub2")) else 0)
                             + (1 if (N >= 4096 and spec.method == "rkc" and spec.K + 1 > 16 and args.variant == "thread") else 0)),
        "work_per_step": work,
        "roofline": roofline(case, float(np.mean(ms)), work, peak_flops / 1e12,
                             "measured: ckb_fp64_probe, sustained DFMA chains on this GPU, >= 1 s per run (MEASURED_PEAKS.json has no FP64 figure)"),
        "exp_per_s": {"achieved": 2.0 * case.m.n_slots * work["rhs_calls"] / (np.mean(ms) * 1e-3), "peak_measured": exp_rate},
        "fp64_probe": probe_info,
        "ms_min_max": [float(min(ms)), float(max(ms))],
    }
    if not args.no_extra:  # every rank at the same time (they share the host's PCIe complex), max over ranks
        barrier()
        tt, h2d, d2h = case.e2e(min(K, 5), 2)
        t_e2e = float(np.mean(tt))
        if world > 1:
            te = torch.tensor([t_e2e], dtype=torch.float64, device="cuda")
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
            t_e2e = float(te.item())
        out["e2e"] = {"value": N * world / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                      "note": "ckb_integrate_host on pinned host buffers (H2D + kernels + D2H in the timed region), "
                              "all ranks at once, max over ranks"}
    if rank == 0 and not args.no_extra and world == 1:
        r, n_used, cores, t = oracle_time(args.config, N, dt, budget_s=12.0)
        out["cpu_baseline"] = {"value": r, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": f"first {n_used} of {N} systems of the workload, {t:.1f} s, OpenMP over systems"}
        r1, n1, _, t1 = oracle_time(args.config, N, dt, budget_s=6.0, nthreads=1)
        out["cpu_baseline"]["single_core"] = {"value": r1, "sample_n": n1, "seconds": t1}
        extra = {}

        def measure(key, c, N2, dt2, var, K2=3, W2=3, cpu=False, **kw):
            """one more workload: ODEs/s, work counters, roofline; optionally the oracle on a bounded sample of it"""
            try:
                s2 = synth.CONFIGS[c]
                cs = GpuCase(c, N2, dt2, var, **kw)
                wk = cs.work()
                m2 = cs.timed_steps(K2, W2)
                rf = roofline(cs, float(np.mean(m2)), wk, peak_flops / 1e12, "measured DFMA probe")
                if kw.get("f1"):
                    rf["traffic"] = None
                e = {"odes_per_s": N2 / (np.mean(m2) * 1e-3), "ms": float(np.mean(m2)), "N": N2, "dt": dt2,
                     "method": s2.method, "variant": var, "work": wk, "roofline": rf}
                if kw.get("f1"):
                    e["n_falloff"] = int(len(cs.mech.fo_reaction))
                cs.close()
                del cs
                if cpu:   # the oracle on all cores and on one core, bounded sample of the same workload
                    r, n_used, cores, t = oracle_time(c, N2, dt2, budget_s=5.0)
                    r1, n1, _, t1 = oracle_time(c, N2, dt2, budget_s=3.0, nthreads=1)
                    e["cpu_baseline"] = {"value": r, "unit": UNIT, "cores": cores, "kind": "oracle",
                                         "sample": f"first {n_used} of {N2} systems, {t:.1f} s",
                                         "single_core": {"value": r1, "sample_n": n1, "seconds": t1}}
                extra[key] = e
            except Exception as ex:  # pragma: no cover
                extra[key] = {"error": str(ex)[:300]}

        # BASELINE.json configs[2..4] at their full sizes; configs[3] with the warp-per-ODE AND the thread-per-ODE variant
        # (B:configs[3]); configs[4] at both global steps (B:configs[4])
        if args.config != 2:
            measure(f"cfg2_rkc_auto_N{HEADLINE_N[2]}", 2, HEADLINE_N[2], 1e-6, "auto", cpu=True)
        if args.config != 3:
            measure(f"cfg3_rkc_warp_N{HEADLINE_N[3]}", 3, HEADLINE_N[3], 1e-6, "warp", cpu=True)
            measure(f"cfg3_rkc_thread_N{HEADLINE_N[3]}", 3, HEADLINE_N[3], 1e-6, "thread")
        if args.config != 4:
            measure(f"cfg4_rkc_auto_N{HEADLINE_N[4]}_dt1e-6", 4, HEADLINE_N[4], 1e-6, "auto", cpu=True)
            measure(f"cfg4_rkc_auto_N{HEADLINE_N[4] // 4}_dt1e-5", 4, HEADLINE_N[4] // 4, 1e-5, "auto", K2=2, W2=1, cpu=True)
        if args.config != 1:
            measure(f"cfg1_rkck_auto_N{HEADLINE_N[1]}", 1, HEADLINE_N[1], 1e-6, "auto", cpu=True)
        # constant-volume closure and two-range thermo + fall-off (8(f)-f1) on the 53-species class
        measure(f"cv_cfg3_rkc_auto_N{HEADLINE_N[3] // 4}", 3, HEADLINE_N[3] // 4, 1e-6, "auto", K2=2, W2=1, cv=True)
        measure(f"f1_cfg3_rkc_auto_N{HEADLINE_N[3] // 8}", 3, HEADLINE_N[3] // 8, 1e-6, "auto", K2=2, W2=1, f1=True)
        # the paper's "similar neighbours" experiment: the same systems sorted by T
        try:
            cs = GpuCase(args.config, N, dt, args.variant, "similar")
            m2 = cs.timed_steps(3, 3)
            wk = cs.work()
            extra["headline_similar_ordering"] = {"odes_per_s": N / (np.mean(m2) * 1e-3), "ms": float(np.mean(m2)),
                                                  "divergence_D_mean": wk.get("divergence_D_mean"),
                                                  "divergence_D_hist10": wk.get("divergence_D_hist10")}
            cs.close()
        except Exception as ex:  # pragma: no cover
            extra["headline_similar_ordering"] = {"error": str(ex)}
        # ODEs/s versus N for the other configs (BASELINE.json metric; a few sizes of each N_list)
        for c, sizes in ((2, (2 ** 10, 2 ** 14, 2 ** 16)), (3, (2 ** 10, 2 ** 13, 2 ** 15)), (4, (2 ** 13, 2 ** 14))):
            if c == args.config:
                continue
            sw = {}
            for n2 in sizes:
                try:
                    cs = GpuCase(c, n2, 1e-6, "auto")
                    m2 = cs.timed_steps(2, 3)
                    sw[str(n2)] = {"odes_per_s": n2 / (np.mean(m2) * 1e-3), "ms": float(np.mean(m2))}
                    cs.close()
                    del cs
                except Exception as ex:  # pragma: no cover
                    sw[str(n2)] = {"error": str(ex)[:200]}
            extra[f"sweep_cfg{c}_auto"] = sw
        # the figure BASELINE.json's north_star target is stated on: configs[3] (53/634, RKC) at N = 2^17
        ns = [extra.get(k) for k in (f"cfg3_rkc_warp_N{HEADLINE_N[3]}", f"cfg3_rkc_thread_N{HEADLINE_N[3]}")]
        ns = [e for e in ns if e and "roofline" in e]
        if ns:
            best = max(ns, key=lambda e: e["odes_per_s"])
            out["north_star"] = {"config": 3, "N": HEADLINE_N[3], "method": "rkc", "variant": best["variant"],
                                 "odes_per_s": best["odes_per_s"], "frac": best["roofline"]["frac"],
                                 "frac_of_nominal": best["roofline"]["frac_of_nominal"], "target_frac": 0.40,
                                 "by_variant": {e["variant"]: {"odes_per_s": e["odes_per_s"], "frac": e["roofline"]["frac"]} for e in ns},
                                 **north_star_counters()}
        out["configs"] = extra
    if (args.sweep or not args.no_extra) and rank == 0 and world == 1:  # ODEs/s versus N (BASELINE.json metric)
        sw = {}
        for n in spec.N_list:
            cs = GpuCase(args.config, n, dt, args.variant, args.ordering)
            m2 = cs.timed_steps(5, 3)
            sw[str(n)] = {"odes_per_s": n / (np.mean(m2) * 1e-3), "ms": float(np.mean(m2))}
            cs.close()
        out["sweep"] = sw
    if "e2e" not in out:
        out["e2e"] = None
    case.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(out))


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
