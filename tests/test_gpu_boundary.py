"""Boundary extensions of SURVEY 8(b): zero-copy device getters / setter, the combined md_get_state, md_measure_peaks."""
import numpy as np
import pytest

from md_workloads import get_config, make_state

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def md():
    import paper_2003_14061_b200 as m
    m.load_library()
    return m


@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_device_getters_and_get_state_equal_the_host_getters(md, precision):
    import torch
    cfg = get_config("wca_4k")
    r, v, _, box = make_state(cfg, 4, jitter_amp=0.1)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", step_mode="split", precision=precision)
    g.set_state(r, v)
    g.step(25)                                                   # several rebuilds: device order differs from id order
    rh, vh, fh = g.positions(), g.velocities(), g.forces()
    rd, vd, fd = g.positions_device(), g.velocities_device(), g.forces_device()
    torch.cuda.synchronize()
    assert np.array_equal(rd.cpu().numpy(), rh) and np.array_equal(vd.cpu().numpy(), vh) and np.array_equal(fd.cpu().numpy(), fh)
    r2, v2 = g.state()
    assert np.array_equal(r2, rh) and np.array_equal(v2, vh)
    both = torch.empty((2, cfg.n_atoms, 3), dtype=torch.float64, pin_memory=True).numpy()      # one transfer
    g.state(both[0], both[1])
    assert np.array_equal(both[0], rh) and np.array_equal(both[1], vh)
    with pytest.raises(md.MDError):                              # a host pointer is refused, not written through
        g._ck(g._L.md_get_positions_device(g._h, rh.ctypes.data))
    # device -> device state hand-off into a second system
    g2 = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", step_mode="split", precision=precision)
    g2.set_state_device(rd, vd)
    assert np.array_equal(g2.positions(), rh) and np.array_equal(g2.velocities(), vh)
    # the same state in another storage order (a fresh system sorts from id order): forces agree to summation rounding
    assert np.abs(g2.forces() - fh).max() <= (1e-11 if precision == "f64" else 64 * 2.0 ** -24 * 4) * np.abs(fh).max()
    bad = rd.clone()
    bad[5, 2] = -0.5
    with pytest.raises(md.MDError):
        g2.set_state_device(bad, vd)
    g.close()
    g2.close()


def test_measure_peaks(md):
    cfg = get_config("wca_4k")
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, density=cfg.density)
    p = g.measure_peaks()
    assert p["sm_count"] >= 100 and p["sm_clock_khz"] > 1e6
    # at most 64 fp64 FMA lanes per SM and clock (the nominal 37-40 TFLOP/s of a B200): 2 x 64 x SMs x clock flops/s
    top64 = 2 * 64 * p["sm_count"] * p["sm_clock_khz"] * 1e3 / 1e12
    assert 5.0 < p["fp64_tflops"] < 1.05 * top64
    assert p["fp32_tflops"] > p["fp64_tflops"]
    g.close()
