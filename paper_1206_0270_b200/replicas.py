"""Replica driver: the paper's "temporal" parallelisation.

The problem is linear and the trajectory is generated separately, so a long inspiral can be cut into
time segments that are evolved INDEPENDENTLY (one replica per GPU, no communication during evolution):
every segment starts from zero data a fixed overlap before its window, the burst of spurious radiation
from the sudden switch-on leaves the grid during the overlap, and only the samples of the window are
kept.  The waveforms of all segments are then patched together.  The other independent units of SURVEY.md 8(e)
are covered the same way: azimuthal modes (`run_modes`) and the resolutions of a Richardson
sequence (`run_richardson`).  Nothing here is on the hot path: it plans the replicas, hands
each one to a solver built by `solver_factory` (the CUDA `Solver` by default; anything with its set_initial /
set_source / set_option / add_observer / step / extract / close methods) and assembles the series.  With torch.distributed initialised, rank r takes segments r, r + world, ...
and rank 0 gathers the pieces (no collective during the evolution).
"""
from __future__ import annotations

import dataclasses
from typing import Callable, List, Optional, Sequence, Tuple

import numpy as np

from . import workloads as wl


@dataclasses.dataclass(frozen=True)
class Segment:
    index: int
    start: int      # first iteration of the window in the long run (samples start+1 .. stop are kept)
    stop: int
    lead: int       # overlap iterations evolved before the window and thrown away
    t0: float       # physical time at which the replica starts (zero data)


def plan_segments(total_steps: int, n_segments: int, overlap_steps: int, dt: float) -> List[Segment]:
    """Equal windows; every segment but the first is preceded by `overlap_steps` discarded iterations."""
    if n_segments < 1 or total_steps < n_segments or overlap_steps < 0:
        raise ValueError("need 1 <= n_segments <= total_steps and overlap_steps >= 0")
    edges = [round(k * total_steps / n_segments) for k in range(n_segments + 1)]
    out = []
    for k in range(n_segments):
        lead = min(overlap_steps, edges[k])
        out.append(Segment(k, edges[k], edges[k + 1], lead, (edges[k] - lead) * dt))
    return out


def run_segment(cfg: wl.Config, seg: Segment, x_obs: float, weights, solver_factory: Callable):
    """Evolve one replica; return (t[k], w[k][n_modes]) for the samples of its window only."""
    n = seg.lead + (seg.stop - seg.start)
    s = solver_factory(cfg)
    try:
        s.set_initial()                                   # zero data
        s.set_source(wl.orbit_table(cfg, n_steps=n, t0=seg.t0))
        s.add_observer(x_obs, weights)
        s.step(n)
        t, w = s.extract(x_obs)
    finally:
        s.close()
    keep = slice(seg.lead, n)
    return t[keep] + seg.t0, w[keep]


def _default_factory(cfg: wl.Config):
    from .teuk import Solver
    return Solver.from_config(cfg)


def run_segmented(cfg: wl.Config, n_segments: int, overlap_steps: int, x_obs: float, weights=None,
                  total_steps: Optional[int] = None, solver_factory: Optional[Callable] = None,
                  rank: int = 0, world: int = 1, gather: Optional[Callable] = None
                  ) -> Tuple[np.ndarray, np.ndarray, List[Segment]]:
    """Patched waveform of a run of `total_steps` iterations cut into `n_segments` replicas.

    `gather(list_of_pieces)` must return the list of every rank's pieces on rank 0 (e.g. built on
    torch.distributed.gather_object); with world == 1 it is not needed.  Returns (t, w, segments)."""
    if cfg.source not in ("circular", "inspiral"):
        raise ValueError("segments need a trajectory table that can start at t0 > 0")
    total = cfg.steps if total_steps is None else total_steps
    segs = plan_segments(total, n_segments, overlap_steps, cfg.dt)
    factory = solver_factory or _default_factory
    mine = [(sg.index,) + run_segment(cfg, sg, x_obs, weights, factory) for sg in segs if sg.index % world == rank]
    pieces = _collect(mine, rank, world, gather)
    if pieces is None:
        return np.empty(0), np.empty((0, cfg.n_modes), dtype=complex), segs
    pieces.sort(key=lambda p: p[0])
    t = np.concatenate([p[1] for p in pieces])
    w = np.concatenate([p[2] for p in pieces])
    return t, w, segs


def _collect(mine, rank, world, gather):
    """Pieces of every rank on rank 0 (None elsewhere); no communication when world == 1."""
    if world == 1:
        return mine
    if gather is None:
        raise ValueError("world > 1 needs a gather function")
    allp = gather(mine)
    if rank != 0:
        return None
    return [p for rank_pieces in allp for p in rank_pieces]


def _evolve(cfg: wl.Config, steps: int, x_obs: float, weights, factory: Callable, orbit=None, initial=None,
            source_kind: int = 0):
    s = factory(cfg)
    try:
        s.set_initial(*(initial if initial is not None else wl.initial_data(cfg)))
        if cfg.source:
            s.set_source(orbit if orbit is not None else wl.orbit_table(cfg, n_steps=steps))
            if source_kind:
                s.set_option("source_kind", source_kind)
        s.add_observer(x_obs, weights)
        s.step(steps)
        return s.extract(x_obs)
    finally:
        s.close()


def run_modes(cfg: wl.Config, x_obs: float, weights=None, steps: Optional[int] = None,
              solver_factory: Optional[Callable] = None, rank: int = 0, world: int = 1,
              gather: Optional[Callable] = None) -> Tuple[np.ndarray, np.ndarray]:
    """The azimuthal modes are decoupled: each m is evolved by its own replica (rank r takes
    modes r, r + world, ...) and the waveform columns are put back in `cfg.modes` order.  The result equals
    the batched run of all modes in one solver bit for bit.  Returns (t, w[k][n_modes]) on rank 0."""
    n = cfg.steps if steps is None else steps
    factory = solver_factory or _default_factory
    ini = wl.initial_data(cfg)
    orbit = wl.orbit_table(cfg, n_steps=n) if cfg.source else None
    mine = []
    for k, m in enumerate(cfg.modes):
        if k % world != rank:
            continue
        one = cfg.scaled(modes=(m,))
        orb = None
        if orbit is not None:
            orb = dict(orbit)
            orb["amp_re"] = np.ascontiguousarray(orbit["amp_re"][k:k + 1])
            orb["amp_im"] = np.ascontiguousarray(orbit["amp_im"][k:k + 1])
        t, w = _evolve(one, n, x_obs, weights, factory, orb, [np.ascontiguousarray(a[k:k + 1]) for a in ini])
        mine.append((k, t, w))
    pieces = _collect(mine, rank, world, gather)
    if pieces is None:
        return np.empty(0), np.empty((0, cfg.n_modes), dtype=complex)
    pieces.sort(key=lambda p: p[0])
    return pieces[0][1], np.concatenate([p[2] for p in pieces], axis=1)


def refine(cfg: wl.Config, factor: int) -> wl.Config:
    """Grid of `cfg` refined `factor` times in r*, theta and t (same domain, same dt/dx, coarse r* nodes stay
    nodes); the run covers the same physical time."""
    if factor < 1:
        raise ValueError("factor >= 1")
    return cfg.scaled(name="%s_x%d" % (cfg.name, factor), n_r=(cfg.n_r - 1) * factor + 1,
                      n_theta=cfg.n_theta * factor, steps=cfg.steps * factor)


def run_richardson(cfg: wl.Config, x_obs: float, factors: Sequence[int] = (1, 2), order: int = 2,
                   steps: Optional[int] = None, solver_factory: Optional[Callable] = None,
                   weights_fn: Callable = wl.observer_weights, source_kind: int = 0, rank: int = 0,
                   world: int = 1, gather: Optional[Callable] = None):
    """Richardson extrapolation of the second-order waveforms ("our code simply performs
    Richardson extrapolations of its second-order numerical solutions"): one replica per resolution (rank r
    takes levels r, r + world, ...), the series compared at the coarsest level's sample times.

    Returns (t, levels, extrapolated) on rank 0: `levels[q]` is level q's waveform at the coarse times and
    `extrapolated[q]` = (f^p levels[q+1] - levels[q]) / (f^p - 1) with f = factors[q+1]/factors[q], p = order,
    for each consecutive pair.  The caller is responsible for the refined grids being stable (A1)."""
    if len(factors) < 2 or any(b <= a or b % factors[0] for a, b in zip(factors, factors[1:])) or factors[0] < 1:
        raise ValueError("factors must be increasing multiples of the first")
    n = cfg.steps if steps is None else steps
    factory = solver_factory or _default_factory
    mine = []
    for q, f in enumerate(factors):
        if q % world != rank:
            continue
        c = refine(cfg, f)
        t, w = _evolve(c, n * f, x_obs, weights_fn(c), factory, source_kind=source_kind)
        stride = f // factors[0]
        mine.append((q, t[stride - 1::stride], w[stride - 1::stride]))
    pieces = _collect(mine, rank, world, gather)
    if pieces is None:
        return np.empty(0), [], []
    pieces.sort(key=lambda p: p[0])
    levels = [p[2] for p in pieces]
    extrap = []
    for q in range(len(levels) - 1):
        g = float(factors[q + 1] / factors[q]) ** order
        extrap.append((g * levels[q + 1] - levels[q]) / (g - 1.0))
    return pieces[0][1], levels, extrap


def torch_gather(pieces):
    """gather() for run_segmented on top of torch.distributed (any backend)."""
    import torch.distributed as dist
    out = [None] * dist.get_world_size() if dist.get_rank() == 0 else None
    dist.gather_object(pieces, out, dst=0)
    return out
