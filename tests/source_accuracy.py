#!/usr/bin/env python
"""Measured comparison of the three deposit profiles (not collected by pytest; needs a B200, ~1 min).

  python tests/source_accuracy.py [--levels 4] [--out gpurun_out/source_accuracy.json]

PAPER.md:114 says the "discrete delta" gives "an order-of-magnitude improvement in accuracy and efficiency"
over the smeared Gaussian.  With the model source of DESIGN.md reading A7 all three profiles approximate the
same distribution A' delta(x - x_p) delta(theta - theta_p), so their waveforms must converge to the SAME
limit, and the speed of that convergence can be measured: config 3's physics (a = 0.9, m = 2, circular
r0 = 10) on a small domain, resolutions h, h/2, h/4, ... through the replica driver's Richardson levels, the
steady-state waveform at r* = 50 over t in [100, 150] M.  Reported per profile: the relative distance of
every level to the common reference (Richardson extrapolation of the two finest four-point-delta levels)."""
import argparse
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1206_0270_b200 import replicas, workloads as wl  # noqa: E402

KINDS = {0: "gaussian_sigma_4_cells", 1: "two_point_delta", 2: "four_point_delta"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--levels", type=int, default=4)
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "source_accuracy.json"))
    a = ap.parse_args()
    base = wl.CONFIGS[3].scaled(name="source_accuracy", rs_min=-60.0, rs_max=140.0, n_r=1601, n_theta=32,
                                dt_over_dx=0.05, steps=24000, observers=(50.0,))
    factors = tuple(2 ** k for k in range(a.levels))
    runs = {}
    for kind in KINDS:
        t, levels, ext = replicas.run_richardson(base, 50.0, factors=factors, source_kind=kind)
        runs[kind] = (t, levels, ext)
    t = runs[0][0]
    sel = (t >= 100.0) & (t <= 150.0)
    ref = runs[2][2][-1][sel]
    nrm = float(np.linalg.norm(ref))
    res = {"grid_base": [base.n_r, base.n_theta], "dx_base": base.dx, "dt_base": base.dt, "factors": list(factors),
           "window_t": [100.0, 150.0], "x_obs": 50.0, "norm_ref": nrm, "profiles": {}}
    for kind, name in KINDS.items():
        _, levels, ext = runs[kind]
        res["profiles"][name] = {
            "level_error": [float(np.linalg.norm(l[sel] - ref)) / nrm for l in levels],
            "richardson_error": [float(np.linalg.norm(e[sel] - ref)) / nrm for e in ext],
            "amplitude": [float(np.sqrt(np.mean(np.abs(l[sel]) ** 2))) for l in levels],
        }
    os.makedirs(os.path.dirname(a.out), exist_ok=True)
    with open(a.out, "w") as f:
        json.dump(res, f, indent=1)
    print(json.dumps(res))


if __name__ == "__main__":
    main()
