"""Stiffness calibration of the synthetic mechanisms.  Run once; output committed.

BASELINE.json's configs state both parameter ranges for the Arrhenius constants and a spectral-radius
span at t=0.  The literal ranges do not give those spans (they give sigma 8-10 decades larger), so
the spans are treated as binding: f is linear in a common factor g on every A_j, hence sigma scales
exactly with g.  This script measures sigma_i = max |eig(df/dy)| on 256 calibration states per
mechanism -- central-difference Jacobian of the ORACLE's source term (oracle/ckoracle.c, ora_rhs),
dense eigenvalues by numpy (harness code) -- and sets

    g = sqrt(lo * hi) / geomean_i(sigma_i)

It calls only oracle/ and the input generator, never the CUDA path.  It writes
paper_1309_2710_b200/synth_calibration.json, which synth.make_mechanism() applies to arr_A.

    python -m oracle.calibrate_sigma
"""
from __future__ import annotations

import json
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import oracle  # noqa: E402
from paper_1309_2710_b200 import synth  # noqa: E402

N_CAL = 256
# mechanism id -> config whose state distribution it is calibrated on (cfg0 and cfg1 share mech 0)
CAL_CFG = {0: 1, 2: 2, 3: 3, 4: 4}


def sigma_fd(om, y0, p):
    n = len(y0)
    J = np.empty((n, n))
    for c in range(n):
        h = 1e-6 * max(abs(y0[c]), 1e-3)
        yp, ym = y0.copy(), y0.copy()
        yp[c] += h
        ym[c] -= h
        J[:, c] = (om.rhs(yp, p) - om.rhs(ym, p)) / (2.0 * h)
    return float(np.abs(np.linalg.eigvals(J)).max())


def main(seed=0):
    out = {}
    for mech_id, cfg in CAL_CFG.items():
        spec = synth.CONFIGS[cfg]
        mech = synth.make_mechanism(cfg, seed=seed, calibrated=False)
        om = oracle.OracleMech(mech)
        states, p = synth.make_states(cfg, N_CAL, seed=seed, stream=2)
        sig = np.array([sigma_fd(om, states[:, i].copy(), p) for i in range(N_CAL)])
        lo, hi = spec.sigma_span
        g = float(np.sqrt(lo * hi) / np.exp(np.mean(np.log(sig))))
        # re-measure on the calibrated mechanism (sigma is exactly linear in g; this is a check)
        mech.arr_A = mech.arr_A * g
        om2 = oracle.OracleMech(mech)
        sig2 = np.array([sigma_fd(om2, states[:, i].copy(), p) for i in range(0, N_CAL, 8)])
        pct = np.percentile(sig * g, [0, 5, 50, 95, 100])
        out[f"mech{mech_id}_seed{seed}"] = {
            "g": g, "target_span": [lo, hi], "calibrated_on_cfg": cfg, "n_states": N_CAL,
            "sigma_uncalibrated_geomean": float(np.exp(np.mean(np.log(sig)))),
            "sigma_min_p5_p50_p95_max": [float(x) for x in pct],
            "recheck_max_rel_dev": float(np.max(np.abs(sig2 / (sig[::8] * g) - 1.0))),
        }
        print(mech_id, json.dumps(out[f"mech{mech_id}_seed{seed}"]))
    path = os.path.join(os.path.dirname(os.path.abspath(synth.__file__)), "synth_calibration.json")
    with open(path, "w") as fh:
        json.dump(out, fh, indent=1, sort_keys=True)
        fh.write("\n")


if __name__ == "__main__":
    main()
