"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default slab
length, CUDA-graph replays, TMA path): (i) every point of the full grid after a short run from seeded
random data, (ii) after a longer run, sampled r* windows that the oracle recomputes from the GPU's own
earlier state (a window of rows depends only on its neighbours one row away per iteration)."""
import numpy as np
import pytest

from paper_1206_0270_b200 import workloads as wl

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module")
def teuk():
    import torch
    assert torch.cuda.is_available()
    from paper_1206_0270_b200 import teuk as t
    t.load()
    return t


def _rel(got, ref):
    den = np.linalg.norm(ref)
    return float(np.linalg.norm(got - ref) / den) if den > 0 else float(np.linalg.norm(got))


@pytest.mark.parametrize("cid,steps", [(5, 40), (4, 40), (3, 64)])
def test_full_grid_short_run(orc, teuk, cid, steps):
    cfg = wl.CONFIGS[cid]
    ini = wl.random_state(cfg, 500 + cid)
    orbit = wl.orbit_table(cfg, n_steps=steps)
    W = wl.observer_weights(cfg)
    x_obs = cfg.observers[-1]
    g = teuk.Solver.from_config(cfg)
    o = orc.OracleSolver.from_config(cfg)
    for s in (g, o):
        s.set_initial(*ini)
        s.set_source(orbit)
        s.add_observer(x_obs, W)
    g.step(steps)              # 1 plain launch + one 32-iteration graph replay + plain remainder
    o.step(steps)
    sg, so = g.get_state(), o.get_state()
    for a, b in zip(sg, so):
        assert np.all(np.isfinite(a))
        assert _rel(a, b) <= TOL
        # element by element, not only in the norm
        assert np.max(np.abs(a - b)) <= 1e-9 * np.max(np.abs(b))
    tg, wg = g.extract(x_obs)
    to, wo = o.waveform(0)
    assert len(tg) == steps and _rel(wg, wo) <= TOL
    g.close()
    o.close()


@pytest.mark.parametrize("cid,steps", [(1, 300), (2, 150)])
def test_full_grid_resident_kernel(orc, teuk, cid, steps):
    """Configs 1 and 2 at full size in the launch configuration bench.py times for them: the resident kernel (the
    library's default there: 128 blocks x 4 rows, 147 blocks x 28 rows), every point against the oracle from seeded
    random data, and bit for bit against the marching kernel."""
    cfg = wl.CONFIGS[cid]
    ini = wl.random_state(cfg, 600 + cid)
    W = wl.observer_weights(cfg)
    x_obs = cfg.observers[-1]
    o = orc.OracleSolver.from_config(cfg)
    o.set_initial(*ini)
    o.add_observer(x_obs, W)
    o.step(steps)
    so = o.get_state()
    to, wo = o.waveform(0)
    o.close()
    out = []
    for kernel in (-1, 0):
        g = teuk.Solver.from_config(cfg)
        g.set_option("kernel", kernel)
        assert g.stat("kernel") == (2 if kernel < 0 else 0)
        g.set_initial(*ini)
        g.add_observer(x_obs, W)
        g.step(steps)
        out.append((g.get_state(), g.extract(x_obs)))
        g.close()
    for a, b in zip(out[0][0], so):
        assert np.all(np.isfinite(a)) and _rel(a, b) <= TOL
        assert np.max(np.abs(a - b)) <= 1e-9 * np.max(np.abs(b))
    assert len(out[0][1][0]) == steps and _rel(out[0][1][1], wo) <= TOL
    for a, b in zip(out[0][0], out[1][0]):
        assert np.array_equal(a, b)
    assert np.array_equal(out[0][1][1], out[1][1][1])


def test_config5_sampled_windows_after_long_run(orc, teuk):
    cfg = wl.CONFIGS[5]
    n_long, n_check, half = 600, 3, 40
    orbit = wl.orbit_table(cfg, n_steps=n_long + n_check)
    ini = wl.random_state(cfg, 77)
    g = teuk.Solver.from_config(cfg)
    g.set_initial(*ini)
    g.set_source(orbit)
    g.step(n_long)
    before = g.get_state()
    g.step(n_check)
    after = g.get_state()
    g.close()
    assert all(np.all(np.isfinite(a)) for a in after)
    x, _ = wl.grid_axes(cfg)
    i_p = int(round((orbit["rs_p"][2 * n_long] - cfg.rs_min) / cfg.dx))
    i_obs = int((50.0 - cfg.rs_min) / cfg.dx)
    rng = np.random.default_rng(5)
    centres = [half, cfg.n_r - half, i_p, i_p + 30, i_obs] + list(rng.integers(200, cfg.n_r - 200, 6))
    sub_orbit = dict(orbit)
    for k in ("rs_p", "theta_p"):
        sub_orbit[k] = np.ascontiguousarray(orbit[k][2 * n_long:])
    for k in ("amp_re", "amp_im"):
        sub_orbit[k] = np.ascontiguousarray(orbit[k][:, 2 * n_long:])
    sub_orbit["n_samples"] = len(sub_orbit["rs_p"])
    worst = 0.0
    for c in centres:
        lo, hi = max(0, int(c) - half), min(cfg.n_r, int(c) + half)
        sub = cfg.scaled(name="win", n_r=hi - lo, rs_min=float(x[lo]), rs_max=float(x[hi - 1]))
        o = orc.OracleSolver.from_config(sub)
        o.set_initial(*[np.ascontiguousarray(b[:, lo:hi]) for b in before])
        o.set_source(sub_orbit)
        o.step(n_check)
        ref = o.get_state()
        o.close()
        # rows whose domain of dependence stays inside the window (true grid edges are exact edges)
        a = 0 if lo == 0 else n_check
        b = (hi - lo) if hi == cfg.n_r else (hi - lo) - n_check
        for q in range(4):
            got = after[q][:, lo + a:lo + b]
            exp = ref[q][:, a:b]
            scale = np.max(np.abs(exp))
            assert scale > 0
            err = float(np.max(np.abs(got - exp)) / scale)
            worst = max(worst, err)
            assert err <= TOL, (c, q, err)
    assert worst < TOL
