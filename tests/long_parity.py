#!/usr/bin/env python
"""Full-length parity runs (not collected by pytest: minutes to hours of host-core time).

  python tests/long_parity.py --config 3 [--steps N] [--arm gpu|oracle2] [--checkpoints 8] [--out FILE]

Protocol of SURVEY.md 8(d) / DESIGN.md section 6: relative L2 distances of Phi, of Pi and of every observer's
waveform after the config's step count (or --steps), on the seeded inputs of paper_1206_0270_b200/workloads.py.
Two arms, each appending ONE JSON line to profiles/r2_long_parity.jsonl (or --out):

  --arm gpu      (needs the GPU) the CUDA path through the C ABI against the CPU oracle ("gpu_vs_oracle"), and the
                 CUDA path against itself with differently ROUNDED coefficients, coef_mode 1 ("gpu_vs_gpu2");
  --arm oracle2  (CPU only) the oracle against a second build of the same source with FMA contraction allowed
                 ("oracle_vs_oracle2": oracle/oracle.py build_fma) -- the distance two correct implementations of
                 the iteration reach through rounding alone, whatever the hardware.

All solvers advance in lockstep and are compared at --checkpoints evenly spaced iteration counts, so a record
also shows up to which iteration the 1e-10 bar of BASELINE.json holds ("bar_holds_until").  The waveform distances
are over the samples recorded up to each checkpoint."""
import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from oracle import oracle as orc  # noqa: E402
from paper_1206_0270_b200 import workloads as wl  # noqa: E402

BAR = 1e-10


def rel(got, ref):
    den = np.linalg.norm(ref)
    return float(np.linalg.norm(got - ref) / den) if den > 0 else float(np.linalg.norm(got))


def state_distance(sa, sb):
    """(rel-L2 Phi, rel-L2 Pi, ||Phi||, ||Pi||) of state sa against the reference sb."""
    phi_a, phi_b = sa[0] + 1j * sa[1], sb[0] + 1j * sb[1]
    pi_a, pi_b = sa[2] + 1j * sa[3], sb[2] + 1j * sb[3]
    return rel(phi_a, phi_b), rel(pi_a, pi_b), float(np.linalg.norm(phi_b)), float(np.linalg.norm(pi_b))


def wave_distance(wa, wb):
    n = float(np.linalg.norm(wb))
    return "silent" if n < 1e-200 else rel(wa, wb)


class Series:
    """Accumulates the waveform of one observer across extract() calls (the CUDA binding hands out increments)."""

    def __init__(self):
        self.w = []

    def add(self, w):
        self.w.append(np.asarray(w))

    def all(self):
        return np.concatenate(self.w) if self.w else np.empty((0, 1), dtype=complex)


def print_tables(path):
    """Markdown tables of the last record per (config, arm) in the jsonl file: final distances, the iteration count
    up to which the 1e-10 bar holds, and the three pairs side by side."""
    recs = {}
    for line in open(path):
        if line.strip():
            d = json.loads(line)
            recs[(d["config"], d["arm"], d["steps"])] = d

    def fmt(v):
        return v if isinstance(v, str) else "%.1e" % v

    def wv(f):
        ws = [w for w in f["waveforms"] if w != "silent"]
        return fmt(max(ws)) if ws else "silent"

    print("| config | iterations | pair | Phi | Pi | waveform (audible observers, worst) | 1e-10 holds up to iteration |")
    print("|---|---|---|---|---|---|---|")
    for key in sorted(recs):
        d = recs[key]
        for pair in ("gpu_vs_oracle", "gpu_vs_gpu2", "oracle_vs_oracle2"):
            if pair in d:
                f = d[pair]["final"]
                full = "full length" if d["full_length"] else "%d of %d" % (d["steps"], wl.CONFIGS[d["config"]].steps)
                hold = d[pair]["bar_holds_until"]
                print("| %d | %d (%s) | %s | %s | %s | %s | %s |" % (
                    d["config"], d["steps"], full, pair.replace("_", " "), fmt(f["rel_l2_phi"]), fmt(f["rel_l2_pi"]), wv(f),
                    ("the end" if hold == d["steps"] else str(hold))))
    print()
    print("History (relative L2 of Pi, the most sensitive field, per checkpoint):")
    print()
    for key in sorted(recs):
        d = recs[key]
        for pair in ("gpu_vs_oracle", "gpu_vs_gpu2", "oracle_vs_oracle2"):
            if pair in d:
                print("- config %d, %s: " % (d["config"], pair.replace("_", " ")) +
                      ", ".join("%d: %.1e" % (c["n"], c["rel_l2_pi"]) for c in d[pair]["history"]))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=0)
    ap.add_argument("--table", action="store_true", help="print BASELINE.md's parity tables (markdown) from the records in --out and exit")
    ap.add_argument("--steps", type=int, default=0)
    ap.add_argument("--arm", default="gpu", choices=["gpu", "oracle2"])
    ap.add_argument("--checkpoints", type=int, default=8)
    ap.add_argument("--out", default=os.path.join(ROOT, "profiles", "r2_long_parity.jsonl"))
    ap.add_argument("--resume-dir", default=None, help="directory for the states between segments (see --segment)")
    ap.add_argument("--segment", type=int, default=0)
    ap.add_argument("--segments", type=int, default=1,
                    help="run iterations [k S, (k+1) S), S = steps / segments, of the run in this call: every "
                         "solver restarts from the state ITS OWN previous segment saved in --resume-dir, with a trajectory table "
                         "that starts at t0 = k S dt (one call on the GPU box is limited to an hour; config 5 needs three)")
    ap.add_argument("--no-oracle", action="store_true", help="--arm gpu without the oracle: gpu_vs_gpu2 only")
    ap.add_argument("--no-sensitivity", action="store_true", help="--arm gpu without the coef_mode 1 run")
    a = ap.parse_args()
    if a.table:
        print_tables(a.out)
        return
    if a.config not in wl.CONFIGS:
        ap.error("--config 1..6 is required")
    cfg = wl.CONFIGS[a.config]
    steps = a.steps or cfg.steps
    ini = wl.initial_data(cfg)
    W = wl.observer_weights(cfg)
    seg = None
    if a.segments > 1:
        assert a.resume_dir and steps % a.segments == 0 and 0 <= a.segment < a.segments
        S = steps // a.segments
        seg = {"k": a.segment, "S": S, "dir": a.resume_dir, "first": a.segment * S}
        os.makedirs(a.resume_dir, exist_ok=True)
        orbit = wl.orbit_table(cfg, n_steps=S, t0=seg["first"] * cfg.dt)     # both sides get the same table
        total_steps, steps = steps, S
    else:
        orbit = wl.orbit_table(cfg, n_steps=steps)
    ncp = max(1, min(a.checkpoints, steps))
    marks = sorted(set(round(steps * (k + 1) / ncp) for k in range(ncp)))

    def make_oracle(library=None):
        o = orc.OracleSolver.from_config(cfg, library=library)
        o.set_initial(*ini)
        o.set_source(orbit)
        for x in cfg.observers:
            o.add_observer(x, W)
        return o

    res = {"config": cfg.cid, "workload": cfg.name, "steps": steps, "full_length": steps == cfg.steps,
           "arm": a.arm, "observers": list(cfg.observers), "checkpoints": marks,
           "threads": int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))}
    pairs = {}          # name -> list of per-checkpoint dicts
    t_cpu = t_gpu = 0.0
    if a.arm == "oracle2":
        o1, o2 = make_oracle(), make_oracle(orc.lib_fma())
        w_prev = [[np.empty((0, cfg.n_modes), dtype=complex)] * 2 for _ in cfg.observers]
        hist_prev = {}
        if seg is not None and seg["k"] > 0:
            for name, oo in (("o1", o1), ("o2", o2)):
                z = np.load(os.path.join(seg["dir"], "%s_seg%d.npy" % (name, seg["k"] - 1)))
                oo.set_initial(*[np.ascontiguousarray(z[c]) for c in range(4)])
            z = np.load(os.path.join(seg["dir"], "owaves_seg%d.npz" % (seg["k"] - 1)))
            w_prev = [[z["a%d" % k], z["b%d" % k]] for k in range(len(cfg.observers))]
            hist_prev = json.load(open(os.path.join(seg["dir"], "ohistory_seg%d.json" % (seg["k"] - 1))))
        off = seg["first"] if seg is not None else 0
        done = 0
        for mk in marks:
            t0 = time.perf_counter()
            o1.step(mk - done)
            t_cpu += time.perf_counter() - t0
            o2.step(mk - done)
            done = mk
            dphi, dpi, nphi, npi = state_distance(o2.get_state(), o1.get_state())
            waves = [wave_distance(np.concatenate([w_prev[k][1], o2.waveform(k)[1]]),
                                   np.concatenate([w_prev[k][0], o1.waveform(k)[1]])) for k in range(len(cfg.observers))]
            pairs.setdefault("oracle_vs_oracle2", []).append(
                {"n": mk + off, "rel_l2_phi": dphi, "rel_l2_pi": dpi, "norm_phi": nphi, "norm_pi": npi, "waveforms": waves})
            print("n=%d oracle_vs_oracle2 phi %.2e pi %.2e w %s" % (mk, dphi, dpi, waves), flush=True)
        res["oracle2_build"] = " ".join(orc.CXXFLAGS_FMA)
        if seg is not None:
            for name, oo in (("o1", o1), ("o2", o2)):
                np.save(os.path.join(seg["dir"], "%s_seg%d.npy" % (name, seg["k"])), np.stack(oo.get_state()))
                old = os.path.join(seg["dir"], "%s_seg%d.npy" % (name, seg["k"] - 1))
                if os.path.exists(old):
                    os.remove(old)
            wz = {}
            for k in range(len(cfg.observers)):
                wz["a%d" % k] = np.concatenate([w_prev[k][0], o1.waveform(k)[1]])
                wz["b%d" % k] = np.concatenate([w_prev[k][1], o2.waveform(k)[1]])
            np.savez(os.path.join(seg["dir"], "owaves_seg%d.npz" % seg["k"]), **wz)
            pairs["oracle_vs_oracle2"] = hist_prev.get("oracle_vs_oracle2", []) + pairs["oracle_vs_oracle2"]
            json.dump(pairs, open(os.path.join(seg["dir"], "ohistory_seg%d.json" % seg["k"]), "w"))
            res["segments"] = {"count": a.segments, "done": seg["k"] + 1, "iterations_each": seg["S"],
                               "note": "run cut into segments; each oracle build restarts from the state its own previous segment saved"}
            res["steps"] = seg["first"] + seg["S"]
            res["full_length"] = res["steps"] == total_steps
            res["checkpoints"] = [c["n"] for c in pairs["oracle_vs_oracle2"]]
        o1.close()
        o2.close()
    else:
        from paper_1206_0270_b200 import Solver

        def saved(name):
            """state a solver saved at the end of the previous segment (its own: errors accumulate as in one run)"""
            if seg is None or seg["k"] == 0:
                return ini
            z = np.load(os.path.join(seg["dir"], "%s_seg%d.npy" % (name, seg["k"] - 1)))
            return [np.ascontiguousarray(z[c]) for c in range(4)]

        def make_gpu(coef_mode):
            g = Solver.from_config(cfg)
            if coef_mode:
                g.set_option("coef_mode", 1)
            g.set_initial(*saved("gpu2" if coef_mode else "gpu"))
            g.set_source(orbit)
            for x in cfg.observers:
                g.add_observer(x, W)
            return g

        g = make_gpu(0)
        res["kernel"] = int(g.stat("kernel"))     # 2 = resident kernel (state on chip), 0 = marching kernel
        g2 = None if (a.no_sensitivity or cfg.n_theta > 128) else make_gpu(1)
        o = None if a.no_oracle else make_oracle()
        if o is not None and seg is not None and seg["k"] > 0:
            o.set_initial(*saved("oracle"))
        sg = [Series() for _ in cfg.observers]
        sg2 = [Series() for _ in cfg.observers]
        so_prev = [np.empty((0, cfg.n_modes), dtype=complex) for _ in cfg.observers]   # oracle samples of earlier segments
        hist_prev = {}
        if seg is not None and seg["k"] > 0:
            z = np.load(os.path.join(seg["dir"], "waves_seg%d.npz" % (seg["k"] - 1)))
            for k in range(len(cfg.observers)):
                sg[k].add(z["g%d" % k]); sg2[k].add(z["h%d" % k]); so_prev[k] = z["o%d" % k]
            hist_prev = json.load(open(os.path.join(seg["dir"], "history_seg%d.json" % (seg["k"] - 1))))
        done = 0
        for mk in marks:
            g.sync()
            t0 = time.perf_counter()
            g.step(mk - done)
            g.sync()
            t_gpu += time.perf_counter() - t0
            if g2 is not None:
                g2.step(mk - done)
            if o is not None:
                t0 = time.perf_counter()
                o.step(mk - done)
                t_cpu += time.perf_counter() - t0
            done = mk
            st = g.get_state()
            for k, x in enumerate(cfg.observers):
                sg[k].add(g.extract(x)[1])
                if g2 is not None:
                    sg2[k].add(g2.extract(x)[1])
            off = seg["first"] if seg is not None else 0
            if o is not None:
                dphi, dpi, nphi, npi = state_distance(st, o.get_state())
                waves = [wave_distance(sg[k].all(), np.concatenate([so_prev[k], o.waveform(k)[1]])) for k in range(len(cfg.observers))]
                pairs.setdefault("gpu_vs_oracle", []).append(
                    {"n": mk + off, "rel_l2_phi": dphi, "rel_l2_pi": dpi, "norm_phi": nphi, "norm_pi": npi, "waveforms": waves})
                print("n=%d gpu_vs_oracle phi %.2e pi %.2e w %s" % (mk, dphi, dpi, waves), flush=True)
            if g2 is not None:
                dphi, dpi, nphi, npi = state_distance(g2.get_state(), st)
                waves = [wave_distance(sg2[k].all(), sg[k].all()) for k in range(len(cfg.observers))]
                pairs.setdefault("gpu_vs_gpu2", []).append(
                    {"n": mk + off, "rel_l2_phi": dphi, "rel_l2_pi": dpi, "norm_phi": nphi, "norm_pi": npi, "waveforms": waves})
                print("n=%d gpu_vs_gpu2 phi %.2e pi %.2e w %s" % (mk, dphi, dpi, waves), flush=True)
        res["gpu_gpts"] = cfg.n_pts * steps / t_gpu / 1e9
        if seg is not None:      # hand the states, series and histories to the next segment
            for name, sol in (("gpu", g), ("gpu2", g2), ("oracle", o)):
                if sol is not None:
                    np.save(os.path.join(seg["dir"], "%s_seg%d.npy" % (name, seg["k"])), np.stack(sol.get_state()))
            wz = {}
            for k in range(len(cfg.observers)):
                wz["g%d" % k] = sg[k].all(); wz["h%d" % k] = sg2[k].all() if g2 is not None else np.empty((0, cfg.n_modes), dtype=complex)
                wz["o%d" % k] = np.concatenate([so_prev[k], o.waveform(k)[1]]) if o is not None else so_prev[k]
            np.savez(os.path.join(seg["dir"], "waves_seg%d.npz" % seg["k"]), **wz)
            for name in pairs:
                pairs[name] = hist_prev.get(name, []) + pairs[name]
            json.dump(pairs, open(os.path.join(seg["dir"], "history_seg%d.json" % seg["k"]), "w"))
            for name in ("gpu", "gpu2", "oracle"):       # the previous segment's states are no longer needed
                old = os.path.join(seg["dir"], "%s_seg%d.npy" % (name, seg["k"] - 1))
                if os.path.exists(old):
                    os.remove(old)
            res["segments"] = {"count": a.segments, "done": seg["k"] + 1, "iterations_each": seg["S"],
                               "note": "one call on the GPU box is limited to an hour: the run is cut into segments; every solver "
                                       "restarts from the state its own previous segment saved, with a trajectory table starting at t0"}
            res["steps"] = seg["first"] + seg["S"]
            res["full_length"] = res["steps"] == total_steps
            res["checkpoints"] = [c["n"] for c in pairs.get("gpu_vs_oracle", pairs.get("gpu_vs_gpu2", []))]
        g.close()
        if g2 is not None:
            g2.close()
        if o is not None:
            o.close()
    if t_cpu > 0:
        res["oracle_mpts"] = cfg.n_pts * steps / t_cpu / 1e6
        res["oracle_seconds"] = t_cpu
    for name, cps in pairs.items():
        last = cps[-1]
        holds = 0
        for c in cps:      # largest checkpoint up to which Phi, Pi and every audible waveform are within the bar
            ws = [w for w in c["waveforms"] if w != "silent"]
            if max([c["rel_l2_phi"], c["rel_l2_pi"]] + ws) <= BAR:
                holds = c["n"]
            else:
                break
        res[name] = {"final": last, "bar_holds_until": holds, "bar": BAR, "history": cps}
    os.makedirs(os.path.dirname(a.out), exist_ok=True)
    with open(a.out, "a") as f:
        f.write(json.dumps(res) + "\n")
    print(json.dumps(res))


if __name__ == "__main__":
    main()
