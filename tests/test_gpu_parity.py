"""Parity of the CUDA path (through the C ABI of include/teuk.h) with the CPU oracle, element by
element on the same seeded inputs.  Tolerance: relative L2 <= 1e-10 in Phi, Pi and each observer's
waveform (BASELINE.json north_star); one-iteration checks use 1e-12."""
import math

import numpy as np
import pytest

from paper_1206_0270_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-10


@pytest.fixture(scope="module")
def teuk():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1206_0270_b200 import teuk as t
    t.load()
    return t


def rel_l2(got, ref):
    got, ref = np.asarray(got), np.asarray(ref)
    den = np.linalg.norm(ref)
    if den == 0.0:
        return float(np.linalg.norm(got))
    return float(np.linalg.norm(got - ref) / den)


def run_pair(orc, teuk, cfg, steps, initial=None, observers=None, options=None, orbit_steps=None, chunks=None,
             source_kind=0):
    """Run oracle and GPU on the same inputs; return dict of states and waveforms."""
    ini = wl.initial_data(cfg) if initial is None else initial
    orbit = wl.orbit_table(cfg, n_steps=orbit_steps if orbit_steps is not None else max(steps, 1))
    W = wl.observer_weights(cfg)
    observers = list(cfg.observers) if observers is None else observers
    o = orc.OracleSolver.from_config(cfg)
    g = teuk.Solver.from_config(cfg)
    for k, v in (options or {}).items():
        g.set_option(k, v)
    o.set_initial(*ini)
    g.set_initial(*ini)
    o.set_source(orbit)
    g.set_source(orbit)
    if source_kind:
        o.set_source_kind(source_kind)
        g.set_option("source_kind", source_kind)
    for x in observers:
        o.add_observer(x, W)
        g.add_observer(x, W)
    o.step(steps)
    for c in (chunks or [steps]):
        g.step(c)
    so, sg = o.get_state(), g.get_state()
    wo = [o.waveform(k) for k in range(len(observers))]
    wg = [g.extract(x) for x in observers]
    launches = g.stat("launches")
    o.close()
    g.close()
    return dict(so=so, sg=sg, wo=wo, wg=wg, launches=launches)


def check_pair(res, tol=TOL, need_signal=True):
    phi_o = res["so"][0] + 1j * res["so"][1]
    phi_g = res["sg"][0] + 1j * res["sg"][1]
    pi_o = res["so"][2] + 1j * res["so"][3]
    pi_g = res["sg"][2] + 1j * res["sg"][3]
    if need_signal:
        assert np.linalg.norm(phi_o) > 0 and np.linalg.norm(pi_o) > 0
    assert np.all(np.isfinite(phi_g)) and np.all(np.isfinite(pi_g))
    e_phi, e_pi = rel_l2(phi_g, phi_o), rel_l2(pi_g, pi_o)
    assert e_phi <= tol and e_pi <= tol, (e_phi, e_pi)
    for (to, wo), (tg, wg) in zip(res["wo"], res["wg"]):
        assert len(to) == len(tg) and np.allclose(to, tg, rtol=1e-14, atol=0)
        if np.linalg.norm(wo) < 1e-200:
            assert np.linalg.norm(wg) < 1e-200      # silent observer
            continue
        e_w = rel_l2(wg, wo)
        assert e_w <= tol, e_w
    return e_phi, e_pi


SMALL = wl.small_test_configs()


# "kernel" 0 = marching kernel, one launch per iteration; 2 = resident kernel, state on chip, one launch per call
# (what the default -1 picks for grids of this size)
@pytest.mark.parametrize("kernel", [0, 2])
@pytest.mark.parametrize("cfg", SMALL, ids=[c.name for c in SMALL])
def test_one_iteration_random_state(orc, teuk, cfg, kernel):
    """All four planes random: every term of Eq. (3)-(4), ghosts, edges and the deposit at once."""
    res = run_pair(orc, teuk, cfg, 1, initial=wl.random_state(cfg, 100 + cfg.cid), options={"kernel": kernel})
    check_pair(res, tol=1e-12)
    res = run_pair(orc, teuk, cfg, 3, initial=wl.random_state(cfg, 200 + cfg.cid), options={"kernel": kernel})
    check_pair(res, tol=1e-12)


@pytest.mark.parametrize("kernel", [0, 2])
@pytest.mark.parametrize("cfg", SMALL, ids=[c.name for c in SMALL])
def test_multi_step_parity(orc, teuk, cfg, kernel):
    """The config's own data, source and observers, after its step count."""
    steps = cfg.steps
    res = run_pair(orc, teuk, cfg, steps, options={"kernel": kernel})
    check_pair(res)
    assert len(res["wg"][0][0]) == steps


def test_config2_quick_tier(orc, teuk):
    cfg = wl.CONFIGS[2]
    check_pair(run_pair(orc, teuk, cfg, 1000))


def test_config3_quick_tier(orc, teuk):
    cfg = wl.CONFIGS[3]
    check_pair(run_pair(orc, teuk, cfg, 300))


def test_config4_quick_tier(orc, teuk):
    cfg = wl.CONFIGS[4]
    check_pair(run_pair(orc, teuk, cfg, 100))


@pytest.mark.parametrize("n_theta", [4, 20, 32, 45, 50, 64, 96, 100, 128, 131, 200, 256])
def test_theta_sizes_and_ragged_lanes(orc, teuk, n_theta):
    """Every lane/vector layout: V = 1, 2, 4, 8, vector and scalar access, idle lanes."""
    cfg = SMALL[3].scaled(name="th%d" % n_theta, n_r=211, n_theta=n_theta, dt_over_dx=0.02, steps=12,
                          modes=(2, 1))
    res = run_pair(orc, teuk, cfg, 12, initial=wl.random_state(cfg, n_theta))
    check_pair(res, tol=1e-11)


@pytest.mark.parametrize("n_r", [4, 5, 6, 17, 18, 19, 33, 130])
def test_tiny_radial_grids_and_slab_tails(orc, teuk, n_r):
    cfg = wl.CONFIGS[1].scaled(name="nr%d" % n_r, n_r=n_r, rs_min=5.0, rs_max=5.0 + 0.4 * (n_r - 1), steps=5,
                               observers=(5.0, 5.0 + 0.4 * (n_r - 1) - 0.1), a=0.5)
    for slab in (0, 1, 3, 16):
        res = run_pair(orc, teuk, cfg, 5, initial=wl.random_state(cfg, n_r), options={"slab_rows": slab})
        check_pair(res, tol=1e-12)


def test_dirichlet_outer_edge(orc, teuk):
    cfg = SMALL[2].scaled(name="dirichlet", outer_bc=1, steps=50)
    check_pair(run_pair(orc, teuk, cfg, 50, initial=wl.random_state(cfg, 5)), tol=1e-11)


def test_graph_and_plain_launches_agree_bitwise(orc, teuk):
    cfg = SMALL[3]
    out = []
    for graph, chunks in ((1, [150]), (0, [150]), (1, [1, 70, 33, 46])):
        g = teuk.Solver.from_config(cfg)
        g.set_option("kernel", 0)
        g.set_option("graph", graph)
        g.set_initial(*wl.random_state(cfg, 3))
        g.set_source(wl.orbit_table(cfg, n_steps=150))
        g.add_observer(30.0, wl.observer_weights(cfg))
        for c in chunks:
            g.step(c)
        out.append((g.get_state(), g.extract(30.0)))
        g.close()
    for k in (1, 2):
        for a, b in zip(out[0][0], out[k][0]):
            assert np.array_equal(a, b)
        assert np.array_equal(out[0][1][1], out[k][1][1]) and len(out[k][1][0]) == 150


def test_programmatic_dependent_launch_is_bitwise_identical(orc, teuk):
    """"pdl" = 1 (default) launches iterations 2..32 of a CUDA-graph batch as programmatic dependents of the previous
    one (their prologue overlaps its tail): same fields and waveforms as fully serialised launches; and the number of
    slabs the rows are dealt to does not change anything either."""
    cfg = SMALL[3]
    out = []
    for pdl, slab_rows in ((1, 0), (0, 0), (1, 7), (0, 1)):
        g = teuk.Solver.from_config(cfg)
        g.set_option("kernel", 0)
        g.set_option("pdl", pdl)
        g.set_option("slab_rows", slab_rows)
        g.set_initial(*wl.random_state(cfg, 4))
        g.set_source(wl.orbit_table(cfg, n_steps=200))
        g.add_observer(30.0, wl.observer_weights(cfg))
        g.step(133)                     # one plain launch, four graph batches, remainder
        g.step(67)
        n = g.stat("slabs")
        assert 1 <= n <= cfg.n_r - 2 and g.stat("slab_rows") == -(-(cfg.n_r - 2) // n)
        out.append((g.get_state(), g.extract(30.0)))
        g.close()
    for k in (1, 2, 3):
        for a, b in zip(out[0][0], out[k][0]):
            assert np.array_equal(a, b)
        assert np.array_equal(out[0][1][1], out[k][1][1]) and len(out[k][1][0]) == 200


def test_ring_buffer_wraps_and_drains(orc, teuk):
    """More iterations than the device ring holds (32768): samples are drained by async copies."""
    cfg = wl.CONFIGS[1].scaled(name="ring", n_r=24, n_theta=8, rs_min=10.0, rs_max=19.2, steps=40000,
                               dt_over_dx=0.005, observers=(12.3,))
    res = run_pair(orc, teuk, cfg, 40000, chunks=[5, 32763, 1, 7231])
    # at the bar of BASELINE.json (1e-10): two roundings of the oracle itself (default build vs FMA-contracted
    # build) end 6e-15 apart on this run (9e-15 in Pi); with dt = 0.02 dx the 24-point cavity amplifies the field
    # to 1e12 and the same pair ends 6e-14 apart
    check_pair(res)
    t = res["wg"][0][0]
    assert len(t) == 40000 and abs(t[-1] - 40000 * cfg.dt) < 1e-9


def test_partial_extract_and_resume(orc, teuk):
    cfg = SMALL[0]
    g = teuk.Solver.from_config(cfg)
    g.set_initial(*wl.initial_data(cfg))
    g.add_observer(30.0)
    g.step(10)
    t1, w1 = g.extract(30.0, capacity=4)
    g.step(5)
    t2, w2 = g.extract(30.0)
    assert len(t1) == 4 and len(t2) == 11
    assert np.allclose(np.concatenate([t1, t2]), cfg.dt * np.arange(1, 16))
    g.set_initial(*wl.initial_data(cfg))          # resets the series
    g.step(3)
    t3, w3 = g.extract(30.0)
    assert len(t3) == 3 and np.array_equal(w3, np.concatenate([w1, w2])[:3])
    g.close()


def test_device_pointers_and_torch_stream(orc, teuk):
    import torch
    cfg = SMALL[2]
    ini = wl.random_state(cfg, 11)
    g = teuk.Solver.from_config(cfg)
    g.use_torch_stream()
    dev = [torch.from_numpy(a).cuda() for a in ini]
    g.set_initial(*dev)
    g.step(7)
    out = [torch.empty_like(d) for d in dev]
    g.get_state(out)
    torch.cuda.synchronize()
    h = teuk.Solver.from_config(cfg)
    h.set_initial(*ini)
    h.step(7)
    ref = h.get_state()
    for a, b in zip(out, ref):
        assert np.array_equal(a.cpu().numpy(), b)
    g.close()
    h.close()


def test_argument_errors(teuk):
    with pytest.raises(teuk.TeukError) as e:
        teuk.Solver(1.0, 1.0, [2], -10, 10, 64, 32, 0.01)       # |a| = M
    assert e.value.code == teuk.TEUK_EINVAL
    with pytest.raises(teuk.TeukError):
        teuk.Solver(0.5, 1.0, [2], -10, 10, 3, 32, 0.01)        # n_r < 4
    with pytest.raises(teuk.TeukError):
        teuk.Solver(0.5, 1.0, [2], -10, 10, 64, 5000, 0.01)     # n_theta > 4096
    cfg = SMALL[3]
    g = teuk.Solver.from_config(cfg)
    g.set_source(wl.orbit_table(cfg, n_steps=5))
    g.step(5)
    with pytest.raises(teuk.TeukError) as e:
        g.step(1)                                               # trajectory table exhausted
    assert e.value.code == teuk.TEUK_EINVAL
    with pytest.raises(teuk.TeukError):
        g.add_observer(1e9)
    with pytest.raises(teuk.TeukError):
        g.set_option("no_such_option", 1)
    g.step(0)
    g.close()


def test_nonfinite_sentinel(teuk):
    cfg = SMALL[0]
    ini = list(wl.initial_data(cfg))
    ini[0] = ini[0].copy()
    ini[0][0, 200, 5] = float("nan")
    g = teuk.Solver.from_config(cfg)
    g.set_initial(*ini)
    g.add_observer(cfg.rs_min + 200 * cfg.dx + 0.01)
    g.step(2)
    with pytest.raises(teuk.TeukError) as e:
        g.extract(cfg.rs_min + 200 * cfg.dx + 0.01)
    assert e.value.code == teuk.TEUK_ENONFINITE
    g.close()


@pytest.mark.parametrize("n_theta", [8, 32, 45, 64, 100, 128, 131, 200, 256])
def test_kernel_variants_agree_bitwise(orc, teuk, n_theta):
    """The register-resident and the shared-memory-resident kernels do the same arithmetic per point:
    fields must agree bit for bit; waveforms differ only in the summation order over theta."""
    cfg = SMALL[3].scaled(name="kv%d" % n_theta, n_r=333, n_theta=n_theta, dt_over_dx=0.02, steps=40, modes=(2, 3))
    out = []
    for kernel in (0, 1):
        g = teuk.Solver.from_config(cfg)
        g.set_option("kernel", kernel)
        g.set_initial(*wl.random_state(cfg, 9))
        g.set_source(wl.orbit_table(cfg, n_steps=40))
        g.add_observer(30.0, wl.observer_weights(cfg))
        g.step(7)
        g.step(33)
        out.append((g.get_state(), g.extract(30.0)))
        g.close()
    for a, b in zip(out[0][0], out[1][0]):
        assert np.array_equal(a, b)
    assert rel_l2(out[1][1][1], out[0][1][1]) < 1e-13


@pytest.mark.parametrize("n_r,n_theta,modes", [(4, 8, (2,)), (5, 32, (1, 2)), (9, 45, (2,)), (150, 64, (2, -1, 0)),
                                                (333, 128, (2,)), (700, 100, (3, 2)), (1500, 20, (2,)), (2600, 64, (2,))])
def test_resident_kernel_is_bitwise_identical(orc, teuk, n_r, n_theta, modes):
    """kernel 2 (state resident in shared memory, one cooperative launch per teuk_step call, block-to-block row
    exchange through L2) against kernel 0: same stage arithmetic, so fields AND waveforms must agree bit for bit,
    for any chunking of the calls, with observers in the first and last cell and the source window crossing
    block boundaries.  Shapes: fewer rows than SMs, several rows per block, ragged last block, idle lanes."""
    L = 0.4 * (n_r - 1)
    cfg = SMALL[3].scaled(name="res%dx%d" % (n_r, n_theta), n_r=n_r, n_theta=n_theta, rs_min=-5.0, rs_max=-5.0 + L,
                          dt_over_dx=0.004, steps=80, modes=modes, observers=(-5.0, -5.0 + L - 0.01, -5.0 + 0.37 * L))
    W = wl.observer_weights(cfg)
    out = []
    for kernel, chunks, cache in ((0, [77], 1), (2, [77], 1), (2, [1, 2, 3, 40, 31], 0), (-1, [5, 72], 1)):
        g = teuk.Solver.from_config(cfg)
        g.set_option("kernel", kernel)
        g.set_option("resident_cache", cache)     # time-independent coefficients kept in shared memory, or rebuilt
        assert g.stat("kernel") == (0 if kernel == 0 else 2)
        g.set_initial(*wl.random_state(cfg, 23))
        g.set_source(wl.orbit_table(cfg, n_steps=80))
        for x in cfg.observers:
            g.add_observer(x, W)
        for c in chunks:
            g.step(c)
        out.append((g.get_state(), [g.extract(x) for x in cfg.observers], g.stat("launches")))
        g.close()
    for k in (1, 2, 3):
        for a, b in zip(out[0][0], out[k][0]):
            assert np.array_equal(a, b), k
        for (t0, w0), (t1, w1) in zip(out[0][1], out[k][1]):
            assert len(t1) == 77 and np.array_equal(t0, t1) and np.array_equal(w0, w1), k
    assert out[1][2] < out[0][2]          # one launch per call instead of one per iteration


def test_resident_kernel_applicability(teuk):
    """kernel 2 is refused (EINVAL, not a silent fallback) when the state does not fit on chip; the automatic
    choice then runs kernel 0; an explicit slab length, coef_mode 1 or temporal_block 2 keep kernel 0."""
    big = wl.CONFIGS[3]
    g = teuk.Solver.from_config(big)
    assert g.stat("kernel") == 0 and g.stat("resident_blocks") == 0
    with pytest.raises(teuk.TeukError) as e:
        g.set_option("kernel", 2)
    assert e.value.code == teuk.TEUK_EINVAL
    g.close()
    g = teuk.Solver.from_config(wl.CONFIGS[2])
    assert g.stat("kernel") == 2 and 1 <= g.stat("resident_blocks") <= 148 and g.stat("resident_rows") >= 27
    g.set_option("slab_rows", 5)
    assert g.stat("kernel") == 0
    g.set_option("slab_rows", 0)
    g.set_option("coef_mode", 1)
    assert g.stat("kernel") == 0
    g.set_option("coef_mode", 0)
    g.set_option("temporal_block", 2)
    assert g.stat("kernel") == 0
    with pytest.raises(teuk.TeukError):
        g.set_option("kernel", 2)
    g.set_option("temporal_block", 1)
    g.set_option("kernel", 2)
    with pytest.raises(teuk.TeukError):
        g.set_option("coef_mode", 1)
    with pytest.raises(teuk.TeukError):
        g.set_option("temporal_block", 2)
    g.close()


def test_resident_kernel_long_run_and_ring_drain(orc, teuk):
    """More iterations than the device ring holds, in the resident kernel: one launch per ring-full of samples."""
    cfg = wl.CONFIGS[1].scaled(name="ring2", n_r=24, n_theta=8, rs_min=10.0, rs_max=19.2, steps=40000,
                               dt_over_dx=0.005, observers=(12.3,))
    res = run_pair(orc, teuk, cfg, 40000, chunks=[5, 32763, 1, 7231], options={"kernel": 2})
    check_pair(res)             # at the bar (see test_ring_buffer_wraps_and_drains)
    assert len(res["wg"][0][0]) == 40000 and res["launches"] < 100


@pytest.mark.parametrize("cfg", SMALL, ids=[c.name for c in SMALL])
def test_smem_kernel_parity(orc, teuk, cfg):
    res = run_pair(orc, teuk, cfg, min(cfg.steps, 300), options={"kernel": 1})
    check_pair(res)
    for slab in (1, 5):
        res = run_pair(orc, teuk, cfg, 4, initial=wl.random_state(cfg, 31), options={"kernel": 1, "slab_rows": slab})
        check_pair(res, tol=1e-12)


@pytest.mark.parametrize("cfg", SMALL, ids=[c.name for c in SMALL])
def test_streamed_coefficient_planes_parity(orc, teuk, cfg):
    """coef_mode 1 (the stored-matrices arm of the bytes-vs-flops comparison) against the oracle."""
    res = run_pair(orc, teuk, cfg, min(cfg.steps, 200), options={"coef_mode": 1})
    check_pair(res)
    res = run_pair(orc, teuk, cfg, 3, initial=wl.random_state(cfg, 41), options={"coef_mode": 1, "slab_rows": 7})
    check_pair(res, tol=1e-12)


@pytest.mark.parametrize("n_theta", [20, 45, 64, 100, 128])
def test_streamed_coefficient_planes_theta_sizes(orc, teuk, n_theta):
    cfg = SMALL[3].scaled(name="cm%d" % n_theta, n_r=150, n_theta=n_theta, dt_over_dx=0.02, steps=8, modes=(2, 1))
    res = run_pair(orc, teuk, cfg, 8, initial=wl.random_state(cfg, n_theta), options={"coef_mode": 1})
    check_pair(res, tol=1e-11)


def test_autotune_does_not_change_results(orc, teuk):
    """The slab-count measurement (inside teuk_create / teuk_set_option, never inside teuk_step) runs trial launches
    into scratch memory only -- also when it is repeated in the middle of a run, with a source and an observer."""
    cfg = SMALL[3]
    out = []
    for auto in (1, 0, 2):
        g = teuk.Solver.from_config(cfg)
        g.set_option("kernel", 0)
        g.set_option("autotune", 1 if auto else 0)
        g.set_initial(*wl.random_state(cfg, 17))
        g.set_source(wl.orbit_table(cfg, n_steps=60))
        g.add_observer(30.0, wl.observer_weights(cfg))
        if auto == 2:
            g.step(29)
            g.set_option("autotune", 1)       # measured again on the live state: nothing may change
            g.step(31)
        else:
            g.step(60)
        assert g.stat("steps") == 60 and g.stat("slab_rows") >= 1
        out.append((g.get_state(), g.extract(30.0)))
        g.close()
    for k in (1, 2):
        for a, b in zip(out[0][0], out[k][0]):
            assert np.array_equal(a, b)
        assert np.array_equal(out[0][1][1], out[k][1][1]) and len(out[k][1][0]) == 60


@pytest.mark.parametrize("n_theta", [129, 132, 200, 240, 256, 304, 360, 361, 513, 1000])
def test_theta_segments(orc, teuk, n_theta):
    """n_theta > 128: several warps per row, each with a 4-column halo (the paper's grid has 304 columns)."""
    cfg = SMALL[3].scaled(name="seg%d" % n_theta, n_r=97, n_theta=n_theta, dt_over_dx=0.002, steps=10, modes=(2, 1),
                          observers=(30.0, -29.9))
    res = run_pair(orc, teuk, cfg, 10, initial=wl.random_state(cfg, n_theta), chunks=[1, 2, 7])
    check_pair(res, tol=1e-11)
    res = run_pair(orc, teuk, cfg, 40, initial=wl.random_state(cfg, n_theta + 1))     # graph replay + separate taps
    check_pair(res, tol=1e-11)
    assert len(res["wg"][0][0]) == 40


def test_paper_grid_quick(orc, teuk):
    """32000 x 304, cropped in r* so the oracle finishes in seconds."""
    cfg = wl.CONFIGS[6].scaled(name="paper_grid_crop", n_r=2000, rs_min=-30.0, rs_max=-30.0 + 1999 * wl.CONFIGS[6].dx,
                               steps=100)
    check_pair(run_pair(orc, teuk, cfg, 100, observers=[50.0]))


def test_seeded_fuzz_of_shapes_and_options(orc, teuk):
    """Random (seeded) grid shapes, spins, mode sets, slab lengths, kernels and edge conditions: a few
    iterations from random data each, against the oracle."""
    rng = np.random.default_rng(20260270)
    for case in range(24):
        n_theta = int(rng.choice([5, 17, 32, 33, 48, 63, 64, 90, 127, 128, 130, 176, 257, 300]))
        n_r = int(rng.integers(4, 160))
        a = float(rng.choice([0.0, 0.3, 0.9, 0.998]))
        modes = tuple(int(m) for m in rng.choice([-3, -2, -1, 0, 1, 2, 3, 4], size=int(rng.integers(1, 4)), replace=False))
        lo = float(rng.uniform(-40.0, 5.0))
        dx = float(rng.uniform(0.05, 0.5))
        kernel = int(rng.integers(0, 2)) if n_theta <= 256 else 0
        coef_mode = int(rng.integers(0, 2)) if (kernel == 0 and n_theta <= 128) else 0
        opts = {"kernel": kernel, "slab_rows": int(rng.choice([0, 1, 2, 5, 9, 64])), "graph": int(rng.integers(0, 2)),
                "outer_bc": int(rng.integers(0, 2))}
        if coef_mode:
            opts["coef_mode"] = 1
        if kernel == 0 and case % 3 == 0:
            opts["kernel"] = -1                 # the automatic choice (resident kernel where it applies)
        steps = int(rng.integers(1, 6))
        kind = int(rng.integers(0, 3))
        cfg = wl.Config(100 + case, "fuzz%d" % case, a, 1.0, modes, lo, lo + dx * (n_r - 1), n_r, n_theta,
                        0.01 / max(1, n_theta // 64), steps, (lo + 0.37 * dx * (n_r - 1),), "zero", "circular",
                        outer_bc=opts["outer_bc"])
        res = run_pair(orc, teuk, cfg, steps, initial=wl.random_state(cfg, case), options=opts, source_kind=kind)
        try:
            check_pair(res, tol=1e-11)
        except AssertionError as e:
            raise AssertionError("case %d: n_r=%d n_theta=%d a=%g modes=%s opts=%s source_kind=%d: %s" % (case, n_r, n_theta, a, modes, opts, kind, e))


@pytest.mark.parametrize("n_r,n_theta", [(4, 8), (5, 32), (7, 64), (37, 128), (150, 64), (333, 128), (200, 100), (64, 20)])
def test_temporal_blocking_is_bitwise_identical(orc, teuk, n_r, n_theta):
    """temporal_block = 2 (warp pairs, level n+1 kept in shared memory) must reproduce temporal_block = 1
    bit for bit: fields and waveforms, odd and even iteration counts, any chunking, graphs on and off."""
    cfg = SMALL[3].scaled(name="tb%dx%d" % (n_r, n_theta), n_r=n_r, n_theta=n_theta, rs_min=-5.0, rs_max=-5.0 + 0.4 * (n_r - 1),
                          dt_over_dx=0.004, steps=80, modes=(2, -1), observers=(-5.0, -5.0 + 0.4 * (n_r - 1) - 0.01))
    W = wl.observer_weights(cfg)
    out = []
    for tb, graph, chunks, slab in ((1, 1, [77], 0), (2, 1, [77], 0), (2, 0, [1, 2, 3, 40, 31], 3), (2, 1, [5, 72], 1)):
        g = teuk.Solver.from_config(cfg)
        g.set_option("temporal_block", tb)
        g.set_option("graph", graph)
        if slab:
            g.set_option("slab_rows", slab)
        g.set_initial(*wl.random_state(cfg, 21))
        g.set_source(wl.orbit_table(cfg, n_steps=80))
        for x in cfg.observers:
            g.add_observer(x, W)
        for c in chunks:
            g.step(c)
        out.append((g.get_state(), [g.extract(x) for x in cfg.observers]))
        g.close()
    for k in (1, 2, 3):
        for a, b in zip(out[0][0], out[k][0]):
            assert np.array_equal(a, b), k
        for (t0, w0), (t1, w1) in zip(out[0][1], out[k][1]):
            assert len(t1) == 77 and np.array_equal(t0, t1) and np.array_equal(w0, w1), k


def test_temporal_blocking_parity_with_oracle(orc, teuk):
    for cfg in (SMALL[3], SMALL[4], SMALL[5]):
        res = run_pair(orc, teuk, cfg, min(cfg.steps, 151), options={"temporal_block": 2})
        check_pair(res)


# ---- discrete-delta deposits ------------------------------------------
@pytest.mark.parametrize("kind", [1, 2])
@pytest.mark.parametrize("cfg", SMALL[3:], ids=[c.name for c in SMALL[3:]])
def test_discrete_delta_source_parity(orc, teuk, cfg, kind):
    res = run_pair(orc, teuk, cfg, min(cfg.steps, 200), source_kind=kind)
    check_pair(res)


@pytest.mark.parametrize("kind", [1, 2])
def test_discrete_delta_source_variants(orc, teuk, kind):
    """Same deposit in every kernel variant: theta segments, shared-memory kernel, temporal blocking, planes."""
    cfg = SMALL[3]
    base = run_pair(orc, teuk, cfg, 61, source_kind=kind)
    check_pair(base)
    for opt in ({"kernel": 1}, {"temporal_block": 2}, {"graph": 0}, {"slab_rows": 7}):
        r = run_pair(orc, teuk, cfg, 61, source_kind=kind, options=opt)
        for a, b in zip(base["sg"], r["sg"]):
            assert np.array_equal(a, b), opt
    check_pair(run_pair(orc, teuk, cfg, 61, source_kind=kind, options={"coef_mode": 1}))
    wide = cfg.scaled(n_theta=304)
    check_pair(run_pair(orc, teuk, wide, 40, source_kind=kind))


def test_discrete_delta_differs_from_gaussian_and_first_step_closed_form(orc, teuk):
    """Non-vacuity: the option changes the fields; after one iteration from zero data Pi is non-zero on the
    few points of the deposit's support only (2 rows x 2 columns of the full stage plus the half stage's
    neighbours), against (2W+1)^2 for the Gaussian."""
    cfg = SMALL[3]
    nz = {}
    for kind in (0, 1, 2):
        res = run_pair(orc, teuk, cfg, 1, source_kind=kind, observers=[])
        check_pair(res, tol=1e-12)
        nz[kind] = int(np.count_nonzero(res["sg"][2]) + np.count_nonzero(res["sg"][3]))
    assert 0 < nz[1] < nz[2] < nz[0]
    assert nz[1] <= 2 * 5 * 6 and nz[2] <= 2 * 7 * 8


def test_source_kind_argument_errors(teuk):
    g = teuk.Solver.from_config(SMALL[3])
    for bad in (-1, 3):
        with pytest.raises(teuk.TeukError):
            g.set_option("source_kind", bad)
    g.close()


# ---- maximum sizes and degenerate cases of the interface ---------------------------------------------------
def test_maximum_theta_width(orc, teuk):
    """n_theta = 4096, the largest the ABI accepts (35 theta segments), with the minimum n_r = 4."""
    for n_r in (4, 9):
        cfg = SMALL[3].scaled(name="thmax", n_r=n_r, n_theta=4096, rs_min=5.0, rs_max=5.0 + 0.01 * (n_r - 1),
                              dt_over_dx=1e-4, steps=6, modes=(2,), observers=(5.005,), source=None)
        res = run_pair(orc, teuk, cfg, 6, initial=wl.random_state(cfg, 4096 + n_r))
        check_pair(res, tol=1e-11)


def test_maximum_mode_count(orc, teuk):
    """64 modes in one launch (gridDim.y = 64), m = -32 .. 31: both pole parities, m = 0, negative m."""
    modes = tuple(range(-32, 32))
    cfg = SMALL[3].scaled(name="m64", n_r=41, n_theta=32, modes=modes, dt_over_dx=0.002, steps=8,
                          rs_min=-5.0, rs_max=35.0, observers=(10.0,), source=None)
    res = run_pair(orc, teuk, cfg, 8, initial=wl.random_state(cfg, 64))
    check_pair(res, tol=1e-11)
    with pytest.raises(teuk.TeukError):
        teuk.Solver(0.5, 1.0, list(range(65)), -10, 10, 64, 32, 0.01)


def test_empty_calls(orc, teuk):
    """step(0), extract before any step, get_state right after create: defined, empty, zero."""
    cfg = SMALL[3]
    g = teuk.Solver.from_config(cfg)
    g.add_observer(cfg.observers[0], wl.observer_weights(cfg))
    g.step(0)
    t, w = g.extract(cfg.observers[0])
    assert len(t) == 0 and w.shape == (0, cfg.n_modes)
    assert all(np.all(a == 0.0) for a in g.get_state())
    assert g.stat("steps") == 0
    g.set_initial()
    g.set_source(None)                                   # source-free, zero data: stays exactly zero
    g.step(33)
    assert all(np.all(a == 0.0) for a in g.get_state())
    t, w = g.extract(cfg.observers[0])
    assert len(t) == 33 and np.all(w == 0.0)
    g.close()


# ---- f2: sums of rank-1 deposit terms with derivative profiles (teuk_set_source_terms) ----------------------
TERM_SPECS = [(0, 0), (1, 0), (0, 1), (2, 0), (1, 1), (0, 2)]


def _random_terms(cfg, n_samples, seed, specs=TERM_SPECS):
    rng = np.random.default_rng(seed)
    return [(a, b, rng.standard_normal((cfg.n_modes, n_samples)) + 1j * rng.standard_normal((cfg.n_modes, n_samples)))
            for a, b in specs]


def _run_terms(orc, teuk, cfg, steps, terms, kind, options=None, chunks=None):
    orbit = wl.orbit_table(cfg, n_steps=steps)
    W = wl.observer_weights(cfg)
    o = orc.OracleSolver.from_config(cfg)
    g = teuk.Solver.from_config(cfg)
    for k, v in (options or {}).items():
        g.set_option(k, v)
    for s_ in (o, g):
        s_.set_initial()
        s_.set_source(orbit)
        s_.set_source_terms(terms)
    o.set_source_kind(kind)
    g.set_option("source_kind", kind)
    for x in cfg.observers:
        o.add_observer(x, W)
        g.add_observer(x, W)
    o.step(steps)
    for c in (chunks or [steps]):
        g.step(c)
    res = dict(so=o.get_state(), sg=g.get_state(), wo=[o.waveform(k) for k in range(len(cfg.observers))],
               wg=[g.extract(x) for x in cfg.observers], launches=g.stat("launches"))
    o.close()
    g.close()
    return res


@pytest.mark.parametrize("kind", [0, 1, 2])
@pytest.mark.parametrize("kernel", [0, 2])
def test_source_terms_parity(orc, teuk, kind, kernel):
    """Six terms (delta, its first and second derivatives in r* and theta, the mixed one) with independent random
    amplitudes per mode and sample, from zero data: everything in the fields comes from the deposit."""
    for cfg in (SMALL[3].scaled(steps=60), SMALL[4].scaled(steps=40), SMALL[5].scaled(steps=30)):
        terms = _random_terms(cfg, 2 * cfg.steps + 1, 100 + kind)
        res = _run_terms(orc, teuk, cfg, cfg.steps, terms, kind, options={"kernel": kernel}, chunks=[1, 2, cfg.steps - 3])
        check_pair(res)


def test_source_terms_single_terms_and_launch_shapes(orc, teuk):
    """Each derivative profile on its own (a wrong sign or a swapped order cannot hide in a sum); kernel 0 with
    graphs, with plain launches and short slabs, and kernel 2 agree bit for bit."""
    cfg = SMALL[3].scaled(steps=40, n_r=333)
    ns = 2 * cfg.steps + 1
    for spec in TERM_SPECS[1:]:
        terms = _random_terms(cfg, ns, 7, specs=[spec])
        base = None
        for opt in ({"kernel": 0}, {"kernel": 2}, {"kernel": 0, "slab_rows": 3, "graph": 0}):
            res = _run_terms(orc, teuk, cfg, cfg.steps, terms, 0, options=opt)
            check_pair(res)
            if base is None:
                base = res
            else:
                for a, b in zip(base["sg"], res["sg"]):
                    assert np.array_equal(a, b), (spec, opt)


def test_source_terms_theta_segments_and_ragged_width(orc, teuk):
    """The paper's own grid is 304 columns wide: theta segments; and a width that is not a multiple
    of the lane width (scalar load path)."""
    for n_theta in (304, 45):
        cfg = SMALL[3].scaled(name="terms%d" % n_theta, n_r=151, n_theta=n_theta, dt_over_dx=0.002, steps=12)
        terms = _random_terms(cfg, 2 * cfg.steps + 1, n_theta)
        check_pair(_run_terms(orc, teuk, cfg, cfg.steps, terms, 0, chunks=[1, 11]))
        check_pair(_run_terms(orc, teuk, cfg, cfg.steps, terms, 2))


def test_source_terms_reset_and_errors(orc, teuk):
    cfg = SMALL[3].scaled(steps=16)
    orbit = wl.orbit_table(cfg, n_steps=16)
    g = teuk.Solver.from_config(cfg)
    with pytest.raises(teuk.TeukError):
        g.set_source_terms(_random_terms(cfg, 33, 1))             # no trajectory installed yet
    g.set_source(orbit)
    with pytest.raises(teuk.TeukError):
        g.set_source_terms([(3, 0, np.zeros((cfg.n_modes, 33)))])
    with pytest.raises(teuk.TeukError):
        g.set_source_terms([(0, -1, np.zeros((cfg.n_modes, 33)))])
    g.set_source_terms(_random_terms(cfg, 33, 1))
    for key, val in (("kernel", 1), ("temporal_block", 2), ("coef_mode", 1)):    # single-term variants only
        with pytest.raises(teuk.TeukError):
            g.set_option(key, val)
    g.set_source_terms([])
    # the (0, 0) term with the table's own amplitude is the default deposit; an empty list and a new
    # teuk_set_source both restore it
    mono = orbit["amp_re"] + 1j * orbit["amp_im"]
    out = []
    for mode in ("default", "explicit", "emptied", "reinstalled"):
        g.set_initial()
        if mode == "explicit":
            g.set_source_terms([(0, 0, mono)])
        elif mode == "emptied":
            g.set_source_terms(_random_terms(cfg, 33, 2))
            g.set_source_terms([])
        elif mode == "reinstalled":
            g.set_source_terms(_random_terms(cfg, 33, 3))
            g.set_source(orbit)
        g.step(16)
        out.append(g.get_state())
    g.close()
    for a, b in zip(out[0], out[1]):                              # another kernel instantiation: rounding level
        assert np.allclose(a, b, rtol=1e-12, atol=1e-12 * np.abs(b).max())
    for k in (2, 3):
        for a, b in zip(out[0], out[k]):
            assert np.array_equal(a, b), k
    assert np.abs(out[0][2]).max() > 0


# ---- the wide kernel: a group of ceil(n_theta / 64) warps per row ("wide" = 1) -------------------------------
def _run_gpu(teuk, cfg, steps, options, ini, orbit, observers, chunks=None):
    g = teuk.Solver.from_config(cfg)
    for k, v in options.items():
        g.set_option(k, v)
    g.set_initial(*ini)
    g.set_source(orbit)
    W = wl.observer_weights(cfg)
    for x in observers:
        g.add_observer(x, W)
    for c in (chunks or [steps]):
        g.step(c)
    out = (g.get_state(), [g.extract(x) for x in observers], g.stat("wide"), g.stat("launches"))
    g.close()
    return out


@pytest.mark.parametrize("n_theta", [66, 100, 128, 130, 192, 256, 304, 320])
def test_wide_kernel_is_bitwise_identical(teuk, n_theta):
    """Fields AND waveforms of the group-of-warps kernel equal those of the one-warp-per-row / theta-segment kernels
    bit for bit: 2 .. 5 warps per row, idle lanes in the last warp, source window and observers (one in the first
    cell, one in the last) crossing slab and chunk boundaries, plain launches, graph batches with and without pdl."""
    cfg = SMALL[3].scaled(name="wide%d" % n_theta, n_r=211, n_theta=n_theta, dt_over_dx=0.002, steps=70, modes=(2, 1),
                          rs_min=-30.0, rs_max=45.0)
    dx = cfg.dx
    obs = (30.0, cfg.rs_min + 0.3 * dx, cfg.rs_max - 1.2 * dx)
    ini = wl.random_state(cfg, n_theta)
    orbit = wl.orbit_table(cfg, n_steps=70)
    ref = _run_gpu(teuk, cfg, 70, {"kernel": 0, "wide": 0}, ini, orbit, obs)
    assert ref[2] == 0
    for opt, chunks in (({"kernel": 0, "wide": 1}, None), ({"kernel": 0, "wide": 1, "pdl": 0}, [1, 2, 67]),
                        ({"kernel": 0, "wide": 1, "graph": 0, "slab_rows": 5}, [35, 35]),
                        ({"kernel": 0, "wide": 1, "slab_rows": 40}, None)):
        got = _run_gpu(teuk, cfg, 70, opt, ini, orbit, obs, chunks)
        assert got[2] == 1, "the wide kernel did not run"
        for a, b in zip(ref[0], got[0]):
            assert np.array_equal(a, b), (n_theta, opt)
        for (ta, wa), (tb, wb) in zip(ref[1], got[1]):
            assert len(ta) == 70 and np.array_equal(ta, tb) and np.array_equal(wa, wb), (n_theta, opt)


@pytest.mark.parametrize("cfg", [SMALL[5], SMALL[5].scaled(name="wide_dirichlet_304", n_theta=304, n_r=400, outer_bc=1,
                                                           dt_over_dx=0.01, steps=120)],
                         ids=["kerr099_small_1500x128", "dirichlet_400x304"])
def test_wide_kernel_parity(orc, teuk, cfg):
    res = run_pair(orc, teuk, cfg, min(cfg.steps, 200), options={"kernel": 0, "wide": 1})
    check_pair(res)


def test_wide_option_applicability(teuk):
    cfg = SMALL[3]                                   # n_theta = 64: one warp per row is all there is
    g = teuk.Solver.from_config(cfg)
    with pytest.raises(teuk.TeukError):
        g.set_option("wide", 1)
    g.close()
    cfg = SMALL[5]
    g = teuk.Solver.from_config(cfg)
    g.set_option("kernel", 0)
    g.set_option("wide", 1)
    assert g.stat("wide") == 1
    g.set_option("temporal_block", 2)                # variants the wide kernel does not cover: the setting is ignored
    assert g.stat("wide") == 0
    g.set_option("temporal_block", 1)
    g.set_source(wl.orbit_table(cfg, n_steps=4))
    g.set_source_terms([(1, 0, np.ones((cfg.n_modes, 9), dtype=complex))])
    assert g.stat("wide") == 1                       # the multi-term deposit has its own wide instantiation
    g.close()


def test_wide_kernel_source_terms(orc, teuk):
    """f2 on the paper's 304-column grid and on 128 columns through the group-of-warps kernel."""
    for n_theta in (304, 128):
        cfg = SMALL[3].scaled(name="wterms%d" % n_theta, n_r=151, n_theta=n_theta, dt_over_dx=0.002, steps=12)
        terms = _random_terms(cfg, 2 * cfg.steps + 1, n_theta)
        res = _run_terms(orc, teuk, cfg, cfg.steps, terms, 0, options={"kernel": 0, "wide": 1}, chunks=[1, 11])
        check_pair(res)
        base = _run_terms(orc, teuk, cfg, cfg.steps, terms, 0, options={"kernel": 0, "wide": 0})
        for a, b in zip(base["sg"], res["sg"]):
            assert np.array_equal(a, b), n_theta


def test_fp64_microbenchmark_is_plausible(teuk):
    """teuk_measure_fp64 (the "alu" ceiling of bench.py): every instruction kind within a factor of the nominal
    148 SMs x 64 lanes x 1.965 GHz = 1.86e13 lane-operations per second; bad arguments are refused."""
    rates = [teuk.measure_fp64(k) for k in range(4)]
    for r in rates:
        assert 4e12 < r < 2.5e13, rates
    with pytest.raises(teuk.TeukError):
        teuk.measure_fp64(4)
