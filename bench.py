#!/usr/bin/env python
"""bench.py -- throughput of the hot path (one "step" = one full Lax-Wendroff iteration: half step,
pole ghosts, full step, radial edges, source deposit, waveform tap) on BASELINE.json's production
config (#5: Kerr a = 0.99, m = 2, 131072 x 128, inspiralling smoothed-delta source).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1..5]

Prints ONE JSON line (contract in the task statement / DESIGN.md "Measurement").
N > 1 (torchrun): the path does not shard without a halo exchange the paper rejected
(PAPER.md:155), so every rank evolves an independent replica ("temporal"
parallelisation: different trajectory segments); no data-path collective; "scaling": "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1206_0270_b200 import workloads as wl  # noqa: E402

BYTES_PER_PT_STEP = 64.0      # 4 FP64 planes read once + written once
METRIC = "FP64 grid-point updates/s"
UNIT = "GPts/s"


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


TRAFFIC_JSON = os.path.join(ROOT, "profiles", "traffic.json")


def ncu_traffic_bytes(cfg):
    """(DRAM bytes per launch of the step kernel, where the figure comes from) from the committed ncu capture,
    if one matches this workload.  It is NOT measured in this run (ncu cannot run inside a timed region):
    `bench.py --ncu-traffic RAW.csv` refreshes the file from an `ncu --page raw --csv` export."""
    if os.path.exists(TRAFFIC_JSON):
        try:
            d = json.load(open(TRAFFIC_JSON))
            if d.get("workload") == cfg.name:
                return float(d["dram_bytes_per_launch"]), d.get("source", "profiles/traffic.json")
        except Exception:
            pass
    return None, None


def refresh_traffic(csv_path, cfg):
    """profiles/traffic.json from the raw page of one `ncu --set full` capture (`ncu -i X.ncu-rep --page raw --csv`):
    mean over the captured launches of teuk_step_kernel of dram__bytes_read.sum + dram__bytes_write.sum."""
    import csv
    rows = list(csv.reader(open(csv_path)))
    hdr = rows[0]
    units = rows[1]
    kn, rd, wr = hdr.index("Kernel Name"), hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    tot_r, tot_w, n, name = 0.0, 0.0, 0, None
    for r in rows[2:]:
        if len(r) <= max(rd, wr) or "teuk_step" not in r[kn]:
            continue
        tot_r += float(r[rd].replace(",", "")) * scale[units[rd]]
        tot_w += float(r[wr].replace(",", "")) * scale[units[wr]]
        n += 1
        name = r[kn]
    if n == 0:
        raise SystemExit("no teuk_step kernel launch in " + csv_path)
    d = {"workload": cfg.name, "kernel": name, "dram_bytes_per_launch": (tot_r + tot_w) / n,
         "dram_bytes_read": tot_r / n, "dram_bytes_write": tot_w / n, "launches_averaged": n,
         "source": "ncu --set full capture, raw page %s (python bench.py --ncu-traffic)" % os.path.basename(csv_path)}
    json.dump(d, open(TRAFFIC_JSON, "w"), indent=1)
    print(json.dumps(d))


# FP64 instructions per point per iteration of the stage code (teuk_stage.cuh lw_stage, both stages), counted from
# the executed-instruction column of the ncu source page of teuk_step_kernel<4,...> on config 5
# (profiles/r2_step_kernel.md, profiles/r2_fp64_peak.md): DFMA with three distinct register operands, other DFMA, DADD, DMUL.
FP64_MIX = {"dfma3": 46.4, "dfma2": 10.3, "dadd": 18.2, "dmul": 22.6}


def alu_peak(cfg, clocks):
    """ "alu" ceiling of the step kernel in GPts/s from the library's FP64 microbenchmark (teuk_measure_fp64,
    DESIGN.md 5.1): the instruction mix above issued back to back at the measured rate of each kind."""
    from paper_1206_0270_b200 import measure_fp64
    r = {k: measure_fp64(i) for i, k in enumerate(("dfma2", "dfma3", "dadd", "dmul"))}
    sec_per_pt = sum(FP64_MIX[k] / r[k] for k in FP64_MIX)
    return {"gpts": 1.0 / sec_per_pt / 1e9, "lane_ops_per_s": r, "fp64_per_pt_step": sum(FP64_MIX.values()),
            "mix": FP64_MIX}


class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample_config(cfg, rows):
    """The workload itself (rows = 0, the default), or, for development runs, a radial crop of `rows` rows
    around the particle."""
    if rows <= 0 or cfg.n_r <= rows:
        return cfg
    dx = cfg.dx
    lo = -rows // 8
    x0 = round((0.0 - cfg.rs_min) / dx) + lo          # crop starts a little inside x = 0
    rs_min = cfg.rs_min + x0 * dx
    rs_max = rs_min + (rows - 1) * dx
    obs = 50.0 if rs_min < 50.0 < rs_max - 2 * dx else rs_min + 0.75 * (rs_max - rs_min)
    return cfg.scaled(name=cfg.name + "_crop%d" % rows, n_r=rows, rs_min=rs_min, rs_max=rs_max,
                      dt_over_dx=cfg.dt_over_dx, observers=(obs,))


def time_oracle(cfg, steps, warmup, rows, source_kind=0):
    """The oracle as it stands on the host cores; returns (GPts/s, threads, sample description)."""
    from oracle import oracle as orc
    c = oracle_sample_config(cfg, rows)
    o = orc.OracleSolver.from_config(c)
    o.set_initial(*wl.initial_data(c))
    orbit = wl.orbit_table(c, n_steps=steps + warmup) if c.source else None
    if orbit is not None:
        # keep the full config's trajectory rate: T refers to cfg.steps * cfg.dt (c.dt == cfg.dt)
        o.set_source(orbit)
        o.set_source_kind(source_kind)
    o.add_observer(c.observers[0], wl.observer_weights(c))
    o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    o.close()
    threads = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    if c is cfg:
        sample = "%d iterations (after %d untimed) of the whole %d x %d x %d-mode grid of the workload incl. source and observer" % (
            steps, warmup, cfg.n_r, cfg.n_theta, cfg.n_modes)
    else:
        sample = "%d iterations of a %d x %d radial crop (of %d x %d) incl. source window and observer" % (
            steps, c.n_r, c.n_theta, cfg.n_r, cfg.n_theta)
    return c.n_pts * steps / dt / 1e9, dt, threads, sample


def replica_orbit(cfg, rank, n_steps):
    """Trajectory table of replica `rank`: segment `rank` of the run (PAPER.md:167 temporal
    parallelisation), i.e. the samples a single long table would hold from iteration rank*n_steps on."""
    if not cfg.source:
        return None
    t0 = rank * n_steps * cfg.dt if cfg.source in ("inspiral", "circular") else 0.0
    return wl.orbit_table(cfg, n_steps=n_steps, t0=t0)


def max_over_ranks(value, device, world):
    """Device-time reduction of the contract: the slowest rank defines the step time."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def run_reference(args, cfg, rank, world):
    """--impl reference: the CPU oracle (the tier's reference arm), rank 0 only."""
    if rank != 0:
        return
    rows = args.oracle_rows
    val, dt, threads, sample = time_oracle(cfg, args.steps, args.warmup, rows, args.source_kind)
    c = oracle_sample_config(cfg, rows)
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "grid": [cfg.n_r, cfg.n_theta], "modes": list(cfg.modes), "a": cfg.a,
                   "sample_grid": [c.n_r, c.n_theta], "l2": "n/a (CPU)"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--oracle-rows", type=int, default=0,
                    help="0 (default): the oracle runs the whole grid of the workload; > 0: a radial crop of that many rows")
    ap.add_argument("--ncu-traffic", default=None, metavar="RAW.csv",
                    help="refresh profiles/traffic.json from an `ncu --page raw --csv` export and exit")
    ap.add_argument("--fp64-peak", action="store_true", help="print the FP64 issue-rate microbenchmark (teuk_measure_fp64) and exit")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--quick", action="store_true", help="development: device-resident timing only")
    ap.add_argument("--slab-rows", type=int, default=0)
    ap.add_argument("--graph", type=int, default=1)
    ap.add_argument("--coef-mode", type=int, default=0, help="0 rebuild coefficients (default), 1 stream 2D planes")
    ap.add_argument("--source-kind", type=int, default=0, help="0 Gaussian deposit (the configs'), 1 / 2 discrete delta")
    ap.add_argument("--source-terms", type=int, default=0,
                    help="0: the config's single-term deposit; N = 1..6: deposit N rank-1 terms with derivative profiles "
                         "(teuk_set_source_terms, f2) to time the TERMS instantiation of the kernels")
    ap.add_argument("--temporal-block", type=int, default=0, help="0 library default, 1 or 2 iterations per HBM round trip")
    ap.add_argument("--pdl", type=int, default=-1, help="-1 library default, 0/1 programmatic dependent launch inside graph batches")
    ap.add_argument("--wide", type=int, default=-1, help="-1 library default, 0 one warp per row / theta segment, 1 a group of warps per row")
    ap.add_argument("--kernel", type=int, default=-1, help="-1 library default (automatic), 0 marching kernel, 1 smem-resident marching kernel, 2 resident (state on chip)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    cfg = wl.CONFIGS[args.config]
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.ncu_traffic:
        refresh_traffic(args.ncu_traffic, cfg)
        return
    if args.impl == "reference":
        run_reference(args, cfg, rank, world)
        return
    if args.fp64_peak:
        print(json.dumps(alu_peak(cfg, None)))
        return

    import torch
    import torch.distributed as dist
    from paper_1206_0270_b200 import Solver

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    K, W = args.steps, args.warmup
    # Untimed iterations on top of the W warm-up steps, so that everything a long teuk_step(K) call uses exists
    # before the timed region starts: the first call runs one plain launch, then builds and replays the CUDA
    # graph of one ping-pong parity (32 iterations), the second call that of the other parity.
    XW = 2 * 33
    # replica r evolves trajectory segment r: its table starts K+W+XW iterations later
    orbit = replica_orbit(cfg, rank, K + W + XW)
    weights = wl.observer_weights(cfg)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        g = Solver.from_config(cfg)
        g.use_torch_stream()
        g.set_option("graph", args.graph)
        if args.slab_rows:
            g.set_option("slab_rows", args.slab_rows)
        if args.kernel >= 0:
            g.set_option("kernel", args.kernel)
        if args.pdl >= 0:
            g.set_option("pdl", args.pdl)
        if args.wide >= 0:
            g.set_option("wide", args.wide)
        if args.coef_mode:
            g.set_option("coef_mode", args.coef_mode)
        if args.temporal_block:
            g.set_option("temporal_block", args.temporal_block)
        if args.source_kind:
            g.set_option("source_kind", args.source_kind)
        # synthetic state resident in HBM: seeded random data on all four planes (throughput does not
        # depend on values; zero data as in the config would let nothing but the source window move)
        gen = torch.Generator(device="cuda").manual_seed(wl.SEED_BASE + cfg.cid + rank)
        dev = [torch.randn(cfg.n_modes, cfg.n_r, cfg.n_theta, dtype=torch.float64, device="cuda", generator=gen)
               * 1e-3 for _ in range(4)]
        g.set_initial(*dev)
        g.set_source(orbit)
        if args.source_terms and orbit is not None:
            # f2: the first N of (delta, d/dx, d/dtheta, d2/dx2, d2/dxdtheta, d2/dtheta2), each with the table's amplitude
            specs = [(0, 0), (1, 0), (0, 1), (2, 0), (1, 1), (0, 2)][:args.source_terms]
            amp = orbit["amp_re"] + 1j * orbit["amp_im"]
            g.set_source_terms([(a_, b_, amp * (cfg.dx ** a_) * (cfg.dtheta ** b_)) for a_, b_ in specs])
        for x in cfg.observers:
            g.add_observer(x, weights)
        # ---- device-resident timing -----------------------------------------------------------
        g.step(W)
        g.step(33)
        g.step(33)
        barrier()
        sampler = ClockSampler(local_rank)
        if rank == 0:
            sampler.start()
        l0 = g.stat("launches")
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(stream)
        g.step(K)            # K iterations: one plain launch, CUDA-graph replays of 32, remainder, flush tap
        e1.record(stream)
        barrier()
        ms = e0.elapsed_time(e1)
        launches = g.stat("launches") - l0
        slab_rows = g.stat("slab_rows")
        kernel_used = g.stat("kernel")
        wide_used = g.stat("wide")
        clocks = sampler.stop() if rank == 0 else None
        ms = max_over_ranks(ms, "cuda", world)
        value = world * cfg.n_pts * K / (ms * 1e-3) / 1e9
        # the series recorded so far (W + K samples) are drained to keep the next phase clean
        for x in cfg.observers:
            g.extract(x, allow_nonfinite=True)

        # ---- end to end through the C ABI with HOST buffers -----------------------------------
        if not args.quick:
            host_in = [torch.randn(cfg.n_modes, cfg.n_r, cfg.n_theta, dtype=torch.float64).pin_memory()
                       for _ in range(4)]
            for h in host_in:
                h.mul_(1e-3)
            host_out = [torch.empty_like(h).pin_memory() for h in host_in]
        e2e_ms = []
        series = []
        orbit_e2e = replica_orbit(cfg, rank, K)
        for rep in range(0 if args.quick else 2):   # first repetition warms the pinned paths
            barrier()
            t0 = time.perf_counter()
            g.set_initial(*host_in)                 # H2D: 4 planes
            g.set_source(orbit_e2e)                 # H2D: trajectory table (a --source-terms run times the e2e leg with the single term)
            g.step(K)
            series = [g.extract(x, allow_nonfinite=True) for x in cfg.observers]   # D2H: waveforms
            g.get_state(host_out)                   # D2H: 4 planes
            barrier()
            e2e_ms.append(1e3 * (time.perf_counter() - t0))
        e2e_t = max_over_ranks(e2e_ms[-1] if e2e_ms else float("inf"), "cuda", world)
        e2e = world * cfg.n_pts * K / (e2e_t * 1e-3) / 1e9
        state_bytes = 4 * cfg.n_pts * 8
        orbit_bytes = 0 if orbit_e2e is None else 8 * (2 + 2 * cfg.n_modes) * orbit_e2e["n_samples"]
        wave_bytes = sum(len(s[0]) * (8 + 16 * cfg.n_modes) for s in series)
        g.close()

    if rank == 0:
        peak, peak_src = measured_peak_gbs()
        achieved = BYTES_PER_PT_STEP * cfg.n_pts * K / (ms * 1e-3) / 1e9   # per GPU: ms is the max over ranks
        traffic, traffic_src = ncu_traffic_bytes(cfg)
        hbm_bound = 2 * 4 * cfg.n_pts * 8 > 2.5e8       # both state copies exceed the 126 MB L2
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "grid": [cfg.n_r, cfg.n_theta], "modes": list(cfg.modes), "a": cfg.a,
                       "dt": cfg.dt, "source": cfg.source, "source_kind": args.source_kind, "source_terms": args.source_terms, "coef_mode": args.coef_mode, "slab_rows": int(slab_rows), "kernel": int(kernel_used), "wide": int(wide_used), "temporal_block": args.temporal_block or "default", "observers": list(cfg.observers),
                       "state_mb": 4 * cfg.n_pts * 8 / 1e6, "parallelism": "replicas x%d" % world,
                       "extra_untimed_warmup": XW,
                       "l2": "inputs larger than L2 (two 537 MB state copies stream through a 126 MB L2)"
                       if 4 * cfg.n_pts * 8 > 2.5e8 else
                       ("state resident in shared memory between iterations (resident kernel): not an HBM measurement"
                        if kernel_used == 2 else "state fits in L2: not an HBM measurement")},
            "clocks": clocks,
            "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": (state_bytes + orbit_bytes) / K,
                    "d2h_bytes_per_step": (state_bytes + wave_bytes) / K,
                    "note": "set_initial + set_source + step(K) + extract + get_state with pinned host buffers"},
            "gpu_launches": int(launches),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                         "kernel": "teuk_step_resident_kernel" if kernel_used == 2 else ("teuk_step_wide_kernel" if wide_used else "teuk_step_kernel"),
                         "bytes_per_pt_step": BYTES_PER_PT_STEP},
        }
        if K < 200:
            line["note"] = "burst (%d steps: the SM clock has not settled under the power cap; sustained figures need >= 1000 steps)" % K
        if not args.quick or not hbm_bound:
            # the FP64 side: co-limit of the HBM roofline on config 5, THE limit where the state stays in L2 / on chip
            alu = alu_peak(cfg, clocks)
            line["roofline_alu"] = {"bound": "alu", "achieved": value / world, "peak": alu["gpts"], "unit": "GPts/s",
                                    "frac": value / world / alu["gpts"], "lane_ops_per_s": alu["lane_ops_per_s"],
                                    "fp64_instructions_per_pt_step": alu["fp64_per_pt_step"],
                                    "peak_source": "teuk_measure_fp64 x the stage's SASS instruction mix (DESIGN.md 5.1), measured in this run after the timed region"}
            if not hbm_bound:
                line["roofline"] = dict(line["roofline_alu"], kernel=line["roofline"]["kernel"], traffic=None,
                                        note="state fits in L2 / on chip: the FP64 pipe, not HBM, bounds this workload")
        if world == 1 and not args.no_cpu_baseline and not args.quick:
            val, dt, threads, sample = time_oracle(cfg, 50, 3, args.oracle_rows, args.source_kind)
            line["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
