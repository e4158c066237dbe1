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


def _pinned(shape):
    import torch
    return torch.empty(shape, dtype=torch.float64, pin_memory=True).numpy()


@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_async_io_equals_the_synchronous_calls(md, precision):
    """md_stage_state + md_commit_state == md_set_state and md_get_state_async + md_wait_io == md_get_state, bit for bit;
    staging a next state leaves the current one and its steps untouched."""
    cfg = get_config("wca_4k")
    r, v, _, box = make_state(cfg, 6, jitter_amp=0.1)
    mk = lambda: md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", precision=precision)
    ga, gb = mk(), mk()
    pin = _pinned((2, cfg.n_atoms, 3))
    pin[0], pin[1] = r, v
    ga.set_state(r, v)
    gb.stage_state(pin[0], pin[1])
    gb.commit_state()
    ga.step(17)
    gb.step(17)
    ra, va = ga.state()
    out = _pinned((2, cfg.n_atoms, 3))
    out[:] = -1.0
    gb.state_async(out[0], out[1])
    gb.wait_io()
    assert np.array_equal(out[0], ra) and np.array_equal(out[1], va)
    # separate (non-adjacent) page-locked arrays: two transfers each way
    r2, v2 = _pinned((cfg.n_atoms, 3)), _pinned((cfg.n_atoms, 3))
    gb.state_async(r2, v2)
    gb.state_async(out[0], out[1])                 # a second request queues behind the first
    gb.wait_io()
    assert np.array_equal(r2, ra) and np.array_equal(v2, va) and np.array_equal(out[0], ra)
    # a staged state does not touch the running one
    nxt = _pinned((2, cfg.n_atoms, 3))
    nxt[0], nxt[1] = np.mod(r + 0.01, box), -v
    gb.stage_state(nxt[0], nxt[1])
    ga.step(9)
    gb.step(9)
    assert np.array_equal(gb.positions(), ga.positions())
    gb.commit_state()
    ga.set_state(nxt[0], nxt[1])
    assert gb.energies().step == 0
    ga.step(5)
    gb.step(5)
    assert np.array_equal(gb.positions(), ga.positions()) and np.array_equal(gb.velocities(), ga.velocities())
    ga.close()
    gb.close()


@pytest.mark.parametrize("name,precision", [("wca_4k", "f64"), ("wca_262k", "f64"), ("wca_262k", "f32")])
def test_async_io_pipeline_over_independent_host_states(md, name, precision):
    """The service loop bench.py's e2e leg times: three independent host-resident trajectories advanced in turn by one
    system, two uploads queued ahead, downloads two deep; a trajectory's buffer goes up again only after its download is
    known complete (wait_io(1): everything but the newest download).  Same results as the serial loop, bit for bit.
    At 262,144 atoms a transfer (12.6 MB each way) outlasts the step it overlaps."""
    cfg = get_config(name)
    n, nt, turns = cfg.n_atoms, 3, 11
    states = [make_state(cfg, seed, jitter_amp=0.1) for seed in (11, 12, 13)]
    box = states[0][3]
    g = md.MDSystem(n, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", precision=precision)
    ser = [np.stack([s[0], s[1]]) for s in states]
    for it in range(turns):
        k = it % nt
        g.set_state(ser[k][0], ser[k][1])
        g.step(3)
        ser[k][0], ser[k][1] = g.state()
    buf = [_pinned((2, n, 3)) for _ in range(nt)]
    for k in range(nt):
        buf[k][0], buf[k][1] = states[k][0], states[k][1]
    g.stage_state(buf[0][0], buf[0][1])
    g.stage_state(buf[1][0], buf[1][1])
    with pytest.raises(md.MDError):
        g.stage_state(buf[2][0], buf[2][1])        # the FIFO holds two
    for it in range(turns):
        k = it % nt
        g.commit_state()                           # the oldest staged state: trajectory k
        g.step(3)
        g.state_async(buf[k][0], buf[k][1])
        if it + 2 < turns:
            g.wait_io(1)                           # trajectory (it + 2) % nt came down one turn ago: complete now
            g.stage_state(buf[(it + 2) % nt][0], buf[(it + 2) % nt][1])
    g.wait_io()
    for k in range(nt):
        assert np.array_equal(buf[k], ser[k])
    with pytest.raises(md.MDError):
        g.wait_io(4)
    g.close()


def test_async_io_rejects_bad_input(md):
    from md_workloads import tetrahedron_body
    cfg = get_config("wca_4k")
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, density=cfg.density)
    pageable = np.zeros((cfg.n_atoms, 3))
    with pytest.raises(md.MDError):
        g.stage_state(pageable, pageable)
    with pytest.raises(md.MDError):
        g.state_async(pageable, pageable)
    with pytest.raises(md.MDError):
        g.commit_state()                           # nothing staged
    g.wait_io()                                    # nothing pending: returns
    bad = _pinned((2, cfg.n_atoms, 3))
    bad[0], bad[1] = g.positions(), g.velocities()
    bad[0][7, 1] = -3.0
    before = g.positions()
    g.stage_state(bad[0], bad[1])
    with pytest.raises(md.MDError):
        g.commit_state()                           # the range check fails on the device; the old state stays
    assert np.array_equal(g.positions(), before)
    g.close()
    body = tetrahedron_body(0.9)
    g = md.MDSystem(4000, cfg.r_cut, 0.4, 0.004, density=0.4, lattice="none")
    g.set_rigid(body)
    with pytest.raises(md.MDError):
        g.stage_state(bad[0][:4000], bad[1][:4000])
    g.close()
