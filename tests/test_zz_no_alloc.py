"""teuk_step_noalloc (include/teuk.h): the allocation-free variant of the resident kernel, whose exchange scratch is
a static device array, against the existing path (teuk_set_initial + teuk_step + teuk_get_state) on the same
inputs.  In a file of its own that pytest collects last; passes alone in a fresh process and after the others."""
import numpy as np
import pytest

from paper_1206_0270_b200 import workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-10       # the bar of tests/test_gpu_parity.py (the two paths run the same kernel: equal bit for bit)


def _rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def _existing_path(teuk, cfg, ini, orbit, chunks):
    g = teuk.Solver.from_config(cfg)
    g.set_option("kernel", 2)
    g.set_initial(*ini)
    g.set_source(orbit)
    out = []
    for c in chunks:
        g.step(c)
        out.append(g.get_state())
    g.close()
    return out


@pytest.mark.parametrize("which", [3, 0])
def test_no_alloc_entry_point_matches_the_existing_path_on_two_calls_in_a_row(which):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1206_0270_b200 import teuk
    teuk.load()
    cfg = wl.small_test_configs()[which]            # 1203 x 64 with a circular-orbit source; 512 x 32 source-free
    n1, n2 = 23, 14
    ini = wl.random_state(cfg, 11 + which)
    orbit = wl.orbit_table(cfg, n_steps=n1 + n2)
    ref = _existing_path(teuk, cfg, ini, orbit, [n1, n2])
    g = teuk.Solver.from_config(cfg)
    g.set_source(orbit)
    dev_in = [torch.from_numpy(a).cuda() for a in ini]
    out1 = [torch.empty_like(a) for a in dev_in]
    out2 = [torch.empty_like(a) for a in dev_in]
    g.step_noalloc(dev_in, 0, n1, out1)              # first call
    g.step_noalloc(out1, n1, n2, out2)               # second call in a row: level n1 -> n1 + n2, same scratch
    g.sync()
    for got, want in ((out1, ref[0]), (out2, ref[1])):
        for a, b in zip(got, want):
            a = a.cpu().numpy()
            assert np.all(np.isfinite(a)) and np.linalg.norm(b) > 0
            assert _rel(a, b) <= TOL, _rel(a, b)
            assert np.array_equal(a, b)              # same kernel, same arithmetic
    # the solver's own state is the result, and the ordinary path continues from it
    st = g.get_state()
    for a, b in zip(st, ref[1]):
        assert np.array_equal(a, b)
    assert g.stat("steps") == n1 + n2
    # another solver of another shape shares the static array and finds this one's rows and tags in it
    cfg2 = wl.small_test_configs()[1]                # 301 x 32, ragged
    ini2 = wl.random_state(cfg2, 5)
    ref2 = _existing_path(teuk, cfg2, ini2, None, [17])
    g2 = teuk.Solver.from_config(cfg2)
    d2 = [torch.from_numpy(a).cuda() for a in ini2]
    g2.step_noalloc(d2, 0, 17, d2)                   # in place
    g2.sync()
    for a, b in zip(d2, ref2[0]):
        assert _rel(a.cpu().numpy(), b) <= TOL
    g2.close()
    g.close()


def test_no_alloc_entry_point_rejects_what_it_cannot_run():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1206_0270_b200 import teuk
    big = wl.CONFIGS[3]                              # 16000 x 64: does not fit on chip
    g = teuk.Solver.from_config(big)
    z = [None] * 4
    with pytest.raises(teuk.TeukError) as e:
        g.step_noalloc(z, 0, 1, z)
    assert e.value.code == teuk.TEUK_EINVAL and "fit on chip" in str(e.value)
    g.close()
    cfg = wl.small_test_configs()[0]
    g = teuk.Solver.from_config(cfg)
    with pytest.raises(teuk.TeukError):
        g.step_noalloc(z, 0, 0, z)                   # n < 1
    g.add_observer(30.0, wl.observer_weights(cfg))
    with pytest.raises(teuk.TeukError) as e:
        g.step_noalloc(z, 0, 4, z)
    assert "observers" in str(e.value)
    g.close()
