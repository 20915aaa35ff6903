"""The N > 1 path (replicas only) on CPU: world_size 2 over gloo.

Covers the host logic bench.py uses under torchrun: per-rank trajectory segments, the max-over-ranks
time reduction, and the rule that only rank 0 runs and prints the reference arm."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1206_0270_b200 import workloads as wl  # noqa: E402


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    cfg = wl.CONFIGS[5]
    n = 6
    orbit = bench.replica_orbit(cfg, rank, n)
    slowest = bench.max_over_ranks(10.0 + 5.0 * rank, "cpu", world)
    gathered = [None] * world
    dist.all_gather_object(gathered, (orbit["rs_p"], orbit["amp_re"], orbit["amp_im"]))
    if rank == 0:
        torch.save({"slowest": slowest, "gathered": gathered}, out)
    dist.barrier()
    dist.destroy_process_group()


def test_replica_segments_and_time_reduction(tmp_path):
    out = str(tmp_path / "r.pt")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    res = torch.load(out, weights_only=False)
    assert res["slowest"] == 15.0                       # max over ranks, not the mean or rank 0's
    cfg = wl.CONFIGS[5]
    n = 6
    long_table = wl.orbit_table(cfg, n_steps=2 * n)    # one table over both segments
    for rank in range(2):
        rs_p, are, aim = res["gathered"][rank]
        sl = slice(2 * n * rank, 2 * n * rank + 2 * n + 1)
        assert np.allclose(rs_p, long_table["rs_p"][sl], rtol=1e-13, atol=0)
        assert np.allclose(are, long_table["amp_re"][:, sl], rtol=0, atol=1e-12 * np.abs(long_table["amp_re"]).max())
        assert np.allclose(aim, long_table["amp_im"][:, sl], rtol=0, atol=1e-12 * np.abs(long_table["amp_im"]).max())
    assert not np.array_equal(res["gathered"][0][0], res["gathered"][1][0])


def test_reference_arm_prints_once_under_torchrun():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "2", "--warmup", "3", "--oracle-rows", "512"]
    env = dict(os.environ, OMP_NUM_THREADS="2")
    p = subprocess.run(cmd, capture_output=True, text=True, cwd=ROOT, env=env, timeout=600)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [json.loads(l) for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["unit"] == "GPts/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
