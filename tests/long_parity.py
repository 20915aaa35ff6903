#!/usr/bin/env python
"""Full-length parity runs (not collected by pytest: minutes to hours of host-core time).

  python tests/long_parity.py --config 3 [--steps N] [--out gpurun_out/long_parity.jsonl]

Runs the CUDA path (through the C ABI) and the CPU oracle on the same seeded inputs for the config's
step count (or --steps), then reports relative L2 errors of Phi, Pi and every observer's waveform
(protocol of SURVEY.md 8(d) / DESIGN.md section 6) and both throughputs.  Appends one JSON line."""
import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from oracle import oracle as orc  # noqa: E402
from paper_1206_0270_b200 import Solver, workloads as wl  # noqa: E402


def rel(got, ref):
    den = np.linalg.norm(ref)
    return float(np.linalg.norm(got - ref) / den) if den > 0 else float(np.linalg.norm(got))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True)
    ap.add_argument("--steps", type=int, default=0)
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "long_parity.jsonl"))
    ap.add_argument("--no-oracle", action="store_true", help="GPU only: report the rounding sensitivity")
    ap.add_argument("--no-sensitivity", action="store_true")
    a = ap.parse_args()
    cfg = wl.CONFIGS[a.config]
    steps = a.steps or cfg.steps
    ini = wl.initial_data(cfg)
    orbit = wl.orbit_table(cfg, n_steps=steps)
    W = wl.observer_weights(cfg)
    g = Solver.from_config(cfg)
    g.set_initial(*ini)
    g.set_source(orbit)
    for x in cfg.observers:
        g.add_observer(x, W)
    g.sync()
    kernel = g.stat("kernel")     # 2 = resident kernel (state on chip), 0 = marching kernel
    t0 = time.perf_counter()
    g.step(steps)
    g.sync()
    t_gpu = time.perf_counter() - t0
    sg = g.get_state()
    wg = [g.extract(x) for x in cfg.observers]
    g.close()
    # rounding sensitivity: the same CUDA path with differently rounded coefficients (streamed planes
    # instead of per-point rebuilds); any two non-bit-identical implementations differ at least this much
    sens = None
    if cfg.n_theta <= 128 and not a.no_sensitivity:
        g2 = Solver.from_config(cfg)
        g2.set_option("coef_mode", 1)
        g2.set_initial(*ini)
        g2.set_source(orbit)
        g2.step(steps)
        s2 = g2.get_state()
        g2.close()
        sens = {"rel_l2_phi": rel(s2[0] + 1j * s2[1], sg[0] + 1j * sg[1]),
                "rel_l2_pi": rel(s2[2] + 1j * s2[3], sg[2] + 1j * sg[3])}
    if a.no_oracle:
        print(json.dumps({"config": cfg.cid, "steps": steps, "gpu_gpts": cfg.n_pts * steps / t_gpu / 1e9,
                          "sensitivity_coef_mode_0_vs_1": sens}))
        return
    o = orc.OracleSolver.from_config(cfg)
    o.set_initial(*ini)
    o.set_source(orbit)
    for x in cfg.observers:
        o.add_observer(x, W)
    t0 = time.perf_counter()
    o.step(steps)
    t_cpu = time.perf_counter() - t0
    so = o.get_state()
    wo = [o.waveform(k) for k in range(len(cfg.observers))]
    o.close()
    phi_g, phi_o = sg[0] + 1j * sg[1], so[0] + 1j * so[1]
    pi_g, pi_o = sg[2] + 1j * sg[3], so[2] + 1j * so[3]
    res = {
        "config": cfg.cid, "workload": cfg.name, "steps": steps, "full_length": steps == cfg.steps, "kernel": int(kernel),
        "rel_l2_phi": rel(phi_g, phi_o), "rel_l2_pi": rel(pi_g, pi_o),
        "norm_phi": float(np.linalg.norm(phi_o)), "norm_pi": float(np.linalg.norm(pi_o)),
        "waveforms": [{"x_obs": x, "rel_l2": (rel(g_[1], o_[1]) if np.linalg.norm(o_[1]) >= 1e-200 else "silent"),
                       "norm": float(np.linalg.norm(o_[1])), "samples": int(len(o_[0]))}
                      for x, g_, o_ in zip(cfg.observers, wg, wo)],
        "gpu_gpts": cfg.n_pts * steps / t_gpu / 1e9, "oracle_mpts": cfg.n_pts * steps / t_cpu / 1e6,
        "oracle_threads": int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1)),
        "oracle_seconds": t_cpu,
        "sensitivity_coef_mode_0_vs_1": sens,
    }
    os.makedirs(os.path.dirname(a.out), exist_ok=True)
    with open(a.out, "a") as f:
        f.write(json.dumps(res) + "\n")
    print(json.dumps(res))


if __name__ == "__main__":
    main()
