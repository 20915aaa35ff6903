"""Replica driver: planning, stitching and the world-size-2
path on CPU with the oracle standing in for the solver; the physics of the overlap on the GPU."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1206_0270_b200 import replicas, workloads as wl  # noqa: E402

CFG = wl.small_test_configs()[3].scaled(name="replica_small", n_r=301, rs_min=-10.0, rs_max=35.0, steps=240,
                                        observers=(25.0,))


def _oracle_factory(cfg):
    from oracle import oracle as orc
    return orc.OracleSolver.from_config(cfg)


def test_plan_segments():
    segs = replicas.plan_segments(1000, 3, 150, 0.01)
    assert [(s.start, s.stop, s.lead) for s in segs] == [(0, 333, 0), (333, 667, 150), (667, 1000, 150)]
    assert segs[1].t0 == pytest.approx(1.83) and segs[0].t0 == 0.0
    assert replicas.plan_segments(10, 2, 100, 1.0)[1].lead == 5          # overlap clipped at t = 0
    with pytest.raises(ValueError):
        replicas.plan_segments(3, 5, 0, 1.0)


def test_full_overlap_reproduces_the_long_run_exactly(orc):
    """With an overlap reaching back to t = 0 every replica repeats the long run up to its window, so the
    patched series must equal the single run bit for bit: pins table offsets, time stamps and stitching."""
    W = wl.observer_weights(CFG)
    t, w, segs = replicas.run_segmented(CFG, 3, 10 ** 9, 25.0, W, solver_factory=_oracle_factory)
    o = orc.OracleSolver.from_config(CFG)
    o.set_initial()
    o.set_source(wl.orbit_table(CFG))
    o.add_observer(25.0, W)
    o.step(CFG.steps)
    t1, w1 = o.waveform(0)
    o.close()
    assert len(t) == CFG.steps and np.allclose(t, t1, rtol=1e-12, atol=0)
    assert np.array_equal(w, w1) and np.abs(w1).max() > 0
    assert [s.lead for s in segs] == [0, 80, 160]


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    W = wl.observer_weights(CFG)
    t, w, _ = replicas.run_segmented(CFG, 4, 30, 25.0, W, solver_factory=_oracle_factory, rank=rank, world=world,
                                     gather=replicas.torch_gather)
    if rank == 0:
        torch.save({"t": t, "w": w}, out)
    else:
        assert len(t) == 0
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_two_matches_single_process(tmp_path):
    out = str(tmp_path / "seg.pt")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    res = torch.load(out, weights_only=False)
    W = wl.observer_weights(CFG)
    t, w, _ = replicas.run_segmented(CFG, 4, 30, 25.0, W, solver_factory=_oracle_factory)
    assert np.array_equal(res["t"], t) and np.array_equal(res["w"], w) and len(t) == CFG.steps


@pytest.mark.gpu
def test_gpu_replicas_reproduce_the_long_run():
    """The CUDA solver behind the driver: with an overlap reaching back to t = 0 the patched series equals the
    single run bit for bit; with a finite overlap the first window is still exact and every window has
    the right time stamps.  (Whether a given overlap is long enough for the switch-on burst to leave is a
    property of the source and the grid, not of the driver: with this model source the steady
    signal is ~1e-6 of the burst, so no accuracy claim is tested.)"""
    from paper_1206_0270_b200 import Solver
    cfg = wl.small_test_configs()[3].scaled(name="replica_gpu", n_r=1203, rs_min=-30.0, rs_max=45.0, steps=3000,
                                            observers=(30.0,))
    W = wl.observer_weights(cfg)
    g = Solver.from_config(cfg)
    g.set_initial()
    g.set_source(wl.orbit_table(cfg))
    g.add_observer(30.0, W)
    g.step(cfg.steps)
    t1, w1 = g.extract(30.0)
    g.close()
    t, w, segs = replicas.run_segmented(cfg, 3, 10 ** 9, 30.0, W)
    assert np.allclose(t, t1, rtol=1e-12, atol=0) and np.array_equal(w, w1) and np.abs(w1).max() > 0
    t, w, segs = replicas.run_segmented(cfg, 3, 200, 30.0, W)
    assert np.allclose(t, t1, rtol=1e-12, atol=0) and np.array_equal(w[:1000], w1[:1000])
    assert [s.lead for s in segs] == [0, 200, 200] and np.all(np.isfinite(w.view(float)))
