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
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

from paper_1206_0270_b200 import replicas, workloads as wl  # noqa: E402

CFG = wl.small_test_configs()[3].scaled(name="replica_small", n_r=301, rs_min=-10.0, rs_max=35.0, steps=240,
                                        observers=(25.0,))


MODES_CFG = wl.small_test_configs()[4].scaled(name="modes_small", n_r=241, rs_min=-10.0, rs_max=30.0, steps=120,
                                              observers=(20.0,))
RICH_CFG = wl.small_test_configs()[0].scaled(name="richardson_small", n_r=321, rs_min=-20.0, rs_max=60.0,
                                             n_theta=16, steps=1280, observers=(30.0,))
RICH_SMALL = RICH_CFG.scaled(name="richardson_tiny", n_r=81, n_theta=8, steps=160)


from oracle_adapter import oracle_factory as _oracle_factory  # noqa: E402  (tests/: the oracle behind the Solver method names)


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
    tm, wm = replicas.run_modes(MODES_CFG, 20.0, wl.observer_weights(MODES_CFG), solver_factory=_oracle_factory,
                                rank=rank, world=world, gather=replicas.torch_gather)
    tr, lev, ext = replicas.run_richardson(RICH_SMALL, 30.0, factors=(1, 2), solver_factory=_oracle_factory,
                                           rank=rank, world=world, gather=replicas.torch_gather)
    if rank == 0:
        torch.save({"t": t, "w": w, "tm": tm, "wm": wm, "tr": tr, "ext": ext[0]}, out)
    else:
        assert len(t) == 0 and len(tm) == 0 and len(tr) == 0 and ext == []
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_two_matches_single_process(tmp_path):
    out = str(tmp_path / "seg.pt")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    res = torch.load(out, weights_only=False)
    W = wl.observer_weights(CFG)
    t, w, _ = replicas.run_segmented(CFG, 4, 30, 25.0, W, solver_factory=_oracle_factory)
    assert np.array_equal(res["t"], t) and np.array_equal(res["w"], w) and len(t) == CFG.steps
    tm, wm = replicas.run_modes(MODES_CFG, 20.0, wl.observer_weights(MODES_CFG), solver_factory=_oracle_factory)
    assert np.array_equal(res["tm"], tm) and np.array_equal(res["wm"], wm) and wm.shape[1] == 5
    tr, _, ext = replicas.run_richardson(RICH_SMALL, 30.0, factors=(1, 2), solver_factory=_oracle_factory)
    assert np.array_equal(res["tr"], tr) and np.array_equal(res["ext"], ext[0]) and len(tr) == RICH_SMALL.steps


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


# ---- the other independent units of SURVEY.md 8(e): azimuthal modes and Richardson resolutions ----------
def test_mode_replicas_equal_the_batched_run_exactly(orc):
    """the m-modes are decoupled, so one replica per mode must give the batched columns bit for bit
    (pins the slicing of initial data and of the amplitude table A'_m, and the column order)."""
    W = wl.observer_weights(MODES_CFG)
    t, w = replicas.run_modes(MODES_CFG, 20.0, W, solver_factory=_oracle_factory)
    o = orc.OracleSolver.from_config(MODES_CFG)
    o.set_initial(*wl.initial_data(MODES_CFG))
    o.set_source(wl.orbit_table(MODES_CFG))
    o.add_observer(20.0, W)
    o.step(MODES_CFG.steps)
    t1, w1 = o.waveform(0)
    o.close()
    assert w.shape == (MODES_CFG.steps, 5) and np.array_equal(t, t1) and np.array_equal(w, w1)
    assert all(np.abs(w1[:, k]).max() > 0 for k in range(5))
    assert len({float(np.abs(w1[-1, k])) for k in range(5)}) == 5                          # columns differ


def test_refine_keeps_domain_nodes_and_time():
    c = replicas.refine(RICH_CFG, 2)
    assert (c.n_r, c.n_theta, c.steps) == (641, 32, 2560)
    assert c.dx == pytest.approx(RICH_CFG.dx / 2) and c.dt == pytest.approx(RICH_CFG.dt / 2)
    assert c.steps * c.dt == pytest.approx(RICH_CFG.steps * RICH_CFG.dt)
    with pytest.raises(ValueError):
        replicas.run_richardson(RICH_CFG, 30.0, factors=(2, 3), solver_factory=_oracle_factory)


def test_richardson_extrapolation_gains_an_order(orc):
    """PAPER.md:117.  Three resolutions: the differences shrink by ~4 per halving (second order) and the
    extrapolated series of the two coarse levels is closer to the extrapolated series of the two fine levels
    than the unextrapolated middle level is to the fine one."""
    t, levels, ext = replicas.run_richardson(RICH_CFG, 30.0, factors=(1, 2, 4), solver_factory=_oracle_factory)
    assert len(t) == RICH_CFG.steps and np.allclose(t, RICH_CFG.dt * np.arange(1, RICH_CFG.steps + 1))
    assert all(l.shape == (RICH_CFG.steps, 1) for l in levels) and len(ext) == 2
    sel = t > 8.0                                            # after the pulse has reached the observer
    assert np.linalg.norm(levels[2][sel]) > 1e-2
    d01 = np.linalg.norm(levels[0][sel] - levels[1][sel])
    d12 = np.linalg.norm(levels[1][sel] - levels[2][sel])
    assert 3.5 < d01 / d12 < 4.6, d01 / d12
    assert np.linalg.norm(ext[0][sel] - ext[1][sel]) < 0.5 * d12
    # world-size split: rank 0 of 2 holds levels 0 and 2 only and must ask for a gather
    with pytest.raises(ValueError):
        replicas.run_richardson(RICH_CFG, 30.0, factors=(1, 2), solver_factory=_oracle_factory, rank=0, world=2)


@pytest.mark.gpu
def test_gpu_mode_and_richardson_replicas():
    """CUDA solver behind the driver: per-mode replicas equal the batched launch (gridDim.y = mode) bit for bit;
    the Richardson levels agree with the oracle-driven levels to the parity bar and the extrapolation gains."""
    from paper_1206_0270_b200 import Solver
    W = wl.observer_weights(MODES_CFG)
    t, w = replicas.run_modes(MODES_CFG, 20.0, W)
    g = Solver.from_config(MODES_CFG)
    g.set_initial(*wl.initial_data(MODES_CFG))
    g.set_source(wl.orbit_table(MODES_CFG))
    g.add_observer(20.0, W)
    g.step(MODES_CFG.steps)
    t1, w1 = g.extract(20.0)
    g.close()
    assert np.array_equal(t, t1) and np.array_equal(w, w1) and np.abs(w1).min(axis=0).shape == (5,)
    tg, lg, eg = replicas.run_richardson(RICH_CFG, 30.0, factors=(1, 2, 4))
    to, lo, eo = replicas.run_richardson(RICH_CFG, 30.0, factors=(1, 2, 4), solver_factory=_oracle_factory)
    assert np.allclose(tg, to, rtol=1e-13, atol=0)
    for a, b in zip(lg + eg, lo + eo):
        assert np.linalg.norm(a - b) <= 1e-10 * np.linalg.norm(b)
    sel = tg > 8.0
    assert np.linalg.norm(eg[0][sel] - eg[1][sel]) < 0.5 * np.linalg.norm(lg[1][sel] - lg[2][sel])
    # discrete-delta deposit through the same driver (option passed to either solver type)
    cg = replicas.run_richardson(CFG, 25.0, factors=(1, 2), source_kind=1)
    co = replicas.run_richardson(CFG, 25.0, factors=(1, 2), source_kind=1, solver_factory=_oracle_factory)
    assert np.linalg.norm(cg[2][0] - co[2][0]) <= 1e-10 * np.linalg.norm(co[2][0]) > 0
