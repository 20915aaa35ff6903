"""Replica driver: the paper's "temporal" parallelisation.

The problem is linear and the trajectory is generated separately, so a long inspiral can be cut into
time segments that are evolved INDEPENDENTLY (one replica per GPU, no communication during evolution):
every segment starts from zero data a fixed overlap before its window, the burst of spurious radiation
from the sudden switch-on leaves the grid during the overlap, and only the samples of the window are
kept.  The waveforms of all segments are then patched together.  Nothing here is on the hot path: it
plans the segments, hands each one to a solver built by `solver_factory` (the CUDA `Solver` by default)
and concatenates the series.  With torch.distributed initialised, rank r takes segments r, r + world, ...
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
        if hasattr(s, "extract"):
            t, w = s.extract(x_obs)
        else:                                             # oracle-style interface (tests)
            t, w = s.waveform(0)
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
    pieces = mine
    if world > 1:
        if gather is None:
            raise ValueError("world > 1 needs a gather function")
        allp = gather(mine)
        if rank != 0:
            return np.empty(0), np.empty((0, cfg.n_modes), dtype=complex), segs
        pieces = [p for rank_pieces in allp for p in rank_pieces]
    pieces.sort(key=lambda p: p[0])
    t = np.concatenate([p[1] for p in pieces])
    w = np.concatenate([p[2] for p in pieces])
    return t, w, segs


def torch_gather(pieces):
    """gather() for run_segmented on top of torch.distributed (any backend)."""
    import torch.distributed as dist
    out = [None] * dist.get_world_size() if dist.get_rank() == 0 else None
    dist.gather_object(pieces, out, dst=0)
    return out
