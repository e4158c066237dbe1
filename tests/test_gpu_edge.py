"""GPU edge cases and error behaviour of the C ABI."""
import numpy as np
import pytest

from md_workloads import get_config, make_state, scaled_config
from md_workloads.configs import R_WCA

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def md():
    import paper_2003_14061_b200 as m
    m.load_library()
    return m


def test_invalid_arguments(md):
    with pytest.raises(md.MDError):
        md.MDSystem(0, R_WCA, 0.4, 0.005, density=0.8)
    with pytest.raises(md.MDError):
        md.MDSystem(4096, R_WCA, 0.4, 0.005)                          # neither box nor density
    with pytest.raises(md.MDError):
        md.MDSystem(4096, R_WCA, 0.4, 0.005, density=0.8, box=10.0)   # inconsistent
    with pytest.raises(md.MDError):
        md.MDSystem(27, R_WCA, 0.4, 0.005, density=0.8)               # box < 3 cells
    with pytest.raises(md.MDError):
        md.MDSystem(4097, R_WCA, 0.4, 0.005, density=0.8)             # fits no lattice
    g = md.MDSystem(4096, R_WCA, 0.4, 0.005, density=0.8, lattice="none")
    with pytest.raises(md.MDError):
        g.step(1)                                                     # no state yet
    r, v, _, box = make_state(get_config("wca_4k"), 1)
    bad = r.copy()
    bad[5, 1] = box * 1.5
    with pytest.raises(md.MDError):
        g.set_state(bad, v)
    g.set_state(r, v)
    g.step(0)
    assert g.energies().step == 0


def test_neighbor_overflow_is_reported(md):
    cfg = get_config("wca_4k")
    r, v, _, box = make_state(cfg, 1, jitter_amp=0.12)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", max_neighbors=4)
    with pytest.raises(md.MDError) as ei:
        g.set_state(r, v)
    assert ei.value.code == -2


def test_zero_shell_rebuilds_every_step(md):
    cfg = scaled_config("wca_4k", 4096, r_shell=0.0)
    r, v, _, box = make_state(cfg, 1, jitter_amp=0.1)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, 0.0, cfg.dt, box=box, lattice="none")
    g.set_state(r, v)
    from oracle.md_oracle import OracleMD
    o = OracleMD(cfg.n_atoms, box, cfg.r_cut, 0.0, cfg.dt)
    o.set_state(r, v)
    g.step(20)
    o.step(20)
    e, eo = g.energies(), o.energies()
    assert e.n_rebuilds == eo.n_rebuilds == 20
    assert e.total == pytest.approx(eo.total, rel=1e-9)


def test_broken_bond_is_reported(md):
    cfg = scaled_config("chains_rows_1m", 4096, chain_len=16)
    r, v, bonds, box = make_state(cfg, 1)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
    g.set_state(r, v)
    far = np.array([[0, 2048]], np.int32)                              # beads of different chains, far apart
    with pytest.raises(md.MDError) as ei:
        g.set_bonds(far, cfg.fene_k, cfg.fene_r0)
    assert ei.value.code == -3
    g2 = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
    g2.set_state(r, v)
    with pytest.raises(md.MDError) as ei:
        g2.set_bonds(np.array([[0, 1], [0, 2], [0, 3]], np.int32), 30.0, 1.5)
    assert ei.value.code == -6


def test_info_and_timers(md):
    cfg = get_config("wca_4k")
    g = md.MDSystem.from_config(cfg, seed=1)
    i = g.info()
    assert i["n_atoms"] == 4096 and i["n_pad"] == 4096 and i["cells_per_edge"] == 11 and i["max_neighbors"] == 32
    assert "B200" in i["device_name"] or i["device_name"]
    g.set_profiling(True)
    g.reset_timers()
    k0 = g.info()["kernel_launches"]
    g.step(50)
    t = g.timers()
    assert t["fused_step"]["launches"] == 49 and t["fused_step"]["ms"] > 0
    assert t["decide"]["launches"] == 50
    assert t["nebr"]["launches"] == 50
    # + 1: the status read that ends md_step is a kernel too (k_publish_ctrl writes the control block to mapped host memory)
    assert g.info()["kernel_launches"] - k0 == sum(x["launches"] for x in t.values()) + 1


def test_set_state_keeps_velocities_when_none(md):
    cfg = get_config("wca_4k")
    g = md.MDSystem.from_config(cfg, seed=3)
    g.step(30)
    v = g.velocities()
    r = g.positions()
    g.set_state(r)                                                     # velocities kept, order reset
    assert np.array_equal(g.velocities(), v)
    assert np.array_equal(g.positions(), r)


def test_graph_and_direct_launch_agree_bitwise(md):
    """md_step through the CUDA graph (conditional rebuild node) and with FLAG_NO_GRAPH run the same kernels in the
    same order: states must be identical, rebuild counts too."""
    cfg = get_config("wca_4k")
    r, v, _, box = make_state(cfg, 4, jitter_amp=0.05)
    out = []
    for flags in (md.FLAG_NO_PERSIST, md.FLAG_NO_GRAPH, md.FLAG_TILED_W, md.FLAG_TILED_W | md.FLAG_NO_GRAPH):
        g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", flags=flags)
        g.set_state(r, v)
        g.step(150)
        g.step(1)
        g.step(37)
        e = g.energies()
        assert g.info()["use_graph"] == (0 if flags & md.FLAG_NO_GRAPH else 1)
        out.append((g.positions(), g.velocities(), e.n_rebuilds, g.info()["kernel_launches"]))
        g.close()
    for a, b in ((0, 1), (2, 3)):
        assert np.array_equal(out[a][0], out[b][0]) and np.array_equal(out[a][1], out[b][1])
        assert out[a][2] == out[b][2] > 10
        assert out[a][3] < out[b][3]          # the graph skips the rebuild chain of steps that do not rebuild


def test_pinned_host_buffers_take_the_direct_copy_path(md):
    import torch
    cfg = get_config("wca_4k")
    r, v, _, box = make_state(cfg, 2, jitter_amp=0.05)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
    rp = torch.empty(r.shape, dtype=torch.float64, pin_memory=True).numpy()
    vp = torch.empty(v.shape, dtype=torch.float64, pin_memory=True).numpy()
    rp[:], vp[:] = r, v
    g.set_state(rp, vp)
    g.step(5)
    out = torch.empty(r.shape, dtype=torch.float64, pin_memory=True).numpy()
    g.positions(out)
    assert np.array_equal(out, g.positions())
    g.velocities(out)
    assert np.array_equal(out, g.velocities())
    g2 = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
    g2.set_state(r, v)
    g2.step(5)
    assert np.array_equal(g2.positions(), g.positions())


def test_two_systems_with_different_tiles_coexist(md):
    """The dynamic shared-memory opt-in is a property of the kernels, not of one system: a dense (large tile) and a
    dilute (small tile) system must both keep working when alive at the same time."""
    from oracle.md_oracle import OracleMD
    big = scaled_config("lj_1m", 4 * 12 ** 3)
    small = get_config("wca_4k")
    systems = []
    for cfg in (big, small, big):
        r, v, _, box = make_state(cfg, 1, jitter_amp=0.1)
        g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
        g.set_state(r, v)
        o = OracleMD(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
        o.set_state(r, v)
        systems.append((g, o, box))
    for g, o, box in systems:
        g.step(10)
        o.step(10)
    for g, o, box in systems:
        d = g.positions() - o.positions()
        d -= box * np.round(d / box)
        assert np.abs(d).max() <= 1e-9
        g.close()


@pytest.mark.parametrize("precision", ["f64", "f32"])
def test_set_state_rejects_out_of_range_coordinates_and_keeps_the_old_state(md, precision):
    """The range check of md_set_state runs on the device before anything of the old state is touched."""
    cfg = get_config("wca_4k")
    r, v, _, box = make_state(cfg, 1, jitter_amp=0.1)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", precision=precision)
    g.set_state(r, v)
    g.step(3)
    p0, v0, e0 = g.positions(), g.velocities(), g.energies()
    for bad_value in (box * 1.001, -1e-9, float("nan")):
        bad = r.copy()
        bad[1234, 2] = bad_value
        with pytest.raises(md.MDError) as ei:
            g.set_state(bad, v)
        assert ei.value.code == md.binding.MD_ERR_INVALID and "coordinate" in str(ei.value)
    assert np.array_equal(g.positions(), p0) and np.array_equal(g.velocities(), v0)
    assert g.energies().total == e0.total and g.energies().step == 3
    g.step(2)                                        # still usable
    edge = r.copy()
    edge[0, 0] = box                                 # x = L itself is accepted (wrapped to 0)
    g.set_state(edge, v)
    assert g.positions()[0, 0] == 0.0
    g.close()


@pytest.mark.parametrize("precision", ["f64", "f32"])
@pytest.mark.parametrize("case", ["wca_4k", "ragged_1000", "chains", "batch", "stride_110k", "stride_chains_98k"])
def test_persistent_launch_equals_the_step_graph_bitwise(md, case, precision):
    """Small systems run md_step as ONE cooperative launch (k_persist: blocks resident over all steps, grid-wide barriers,
    the bodies of the same kernels).  With the same W build (the gathering kernel, MD_FLAG_GLOBAL_W) the step graph must
    give bit-identical states, energies and rebuild counts -- across many rebuilds, in one call or several.  The "stride"
    cases are larger than the resident grid holds one atom per thread (~75,000): the high-occupancy instantiation with
    grid-stride loops, several atoms per thread."""
    n_sys = 1
    if case == "wca_4k":
        cfg = get_config("wca_4k")
    elif case == "ragged_1000":
        cfg = scaled_config("wca_4k", 1000)
    elif case == "chains":
        cfg = scaled_config("chains_rows_1m", 4096, chain_len=16)
    elif case == "stride_110k":
        cfg = scaled_config("wca_262k", 110592)
    elif case == "stride_chains_98k":
        cfg = scaled_config("chains_rows_1m", 98304, chain_len=64)
    else:
        cfg, n_sys = scaled_config("wca_4k", 1728), 3
    states = [make_state(cfg, 4 + b, jitter_amp=0.05 if cfg.lattice == "sc" else 0.0) for b in range(n_sys)]
    box = states[0][3]
    r, v = np.concatenate([s[0] for s in states]), np.concatenate([s[1] for s in states])
    bonds = None if states[0][2] is None else np.concatenate([s[2] + b * cfg.n_atoms for b, s in enumerate(states)])
    out = []
    for flags in (0, md.FLAG_GLOBAL_W):
        g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", flags=flags, n_systems=n_sys, precision=precision)
        g.set_state(r, v)
        if bonds is not None:
            g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
        assert g.info()["use_graph"] == (2 if flags == 0 else 0)     # the graph is built at the first md_step
        g.step(150)
        g.step(1)
        g.step(37)
        e = g.energies()
        assert g.info()["use_graph"] == (2 if flags == 0 else 1)
        out.append((g.positions(), g.velocities(), g.forces(), e.n_rebuilds, e.ke, e.pe, g.info()["kernel_launches"]))
        g.close()
    a, b = out
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])
    assert a[3] == b[3] > 10 and a[4] == b[4] and a[5] == b[5]
    assert a[6] < b[6] // 10                      # three launches for the three md_step calls, plus set-up and read-out


def test_bond_list_validation_and_allocators_side_by_side(md):
    """md_set_bonds rejects a bond between two independent systems and a pair listed twice (either order); systems created
    under different allocator hooks coexist and free their memory the way it was allocated."""
    cfg = scaled_config("chains_rows_1m", 1024, chain_len=16)
    r, v, bonds, box = make_state(cfg, 1)
    n = cfg.n_atoms
    g = md.MDSystem(n, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", n_systems=2)
    g.set_state(np.concatenate([r, r]), np.concatenate([v, v]))
    with pytest.raises(md.MDError) as ei:
        g.set_bonds(np.array([[3, n + 3]], np.int32), cfg.fene_k, cfg.fene_r0)          # atoms of two mutually invisible systems
    assert ei.value.code == md.binding.MD_ERR_INVALID
    for dup in ([[0, 1], [0, 1]], [[0, 1], [1, 0]]):
        with pytest.raises(md.MDError) as ei:
            g.set_bonds(np.array(dup, np.int32), cfg.fene_k, cfg.fene_r0)
        assert ei.value.code == md.binding.MD_ERR_INVALID
    g.set_bonds(np.concatenate([bonds, bonds + n]), cfg.fene_k, cfg.fene_r0)                # the valid list still goes in
    g.step(5)
    # one system on cudaMalloc, one on torch's caching allocator, created and destroyed in interleaved order
    a = md.MDSystem(n, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", torch_memory=False)
    b = md.MDSystem(n, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", torch_memory=True)
    c = md.MDSystem(n, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", torch_memory=False)
    for s in (a, b, c):
        s.set_state(r, v)
        s.step(3)
    a.close()
    b.step(3)
    c.step(3)
    assert np.array_equal(b.positions(), c.positions())
    b.close()
    c.close()
    g.close()
