"""GPU parity of the bond-angle terms (md_set_angles, R19) against the oracle, with
north_star's tolerances (forces 1e-10, positions and energies after 10 steps 1e-9)."""
import numpy as np
import pytest

from md_workloads import make_state, scaled_config
from oracle.md_oracle import OracleMD
from parity_util import ENERGY_RTOL, FORCE_RTOL, POS_ATOL, force_rel_err, pos_err, sets_equal

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def md():
    import paper_2003_14061_b200 as m
    m.load_library()
    return m


def make_pair(md, cfg, seed, k_theta, cos0, variant="full", mode="fused", flags=0, thermal=False, **kw):
    r, v, bonds, box = make_state(cfg, seed)
    o = OracleMD(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(r, v)
    assert o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0) == 0
    assert o.set_angles(k_theta, cos0) == 0
    if thermal:
        assert o.step(150) == 0
        r, v = o.positions(), o.velocities()
        o.set_state(r, v)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", force_variant=variant,
                    step_mode=mode, flags=flags, **kw)
    g.set_state(r, v)
    g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    g.set_angles(k_theta, cos0)
    return g, o, box


CASES = {"chains_4096x16": (4096, 16), "chains_ragged_1000x10": (1000, 10), "chains_3000x20": (3000, 20)}


@pytest.mark.parametrize("case", list(CASES))
@pytest.mark.parametrize("variant,mode,flags", [("full", "fused", 0), ("full", "split", 0), ("full", "fused", 2),
                                                ("newton3", "split", 0), ("full", "fused", 32), ("full", "fused", 16 | 8)])
@pytest.mark.parametrize("k_theta,cos0", [(2.0, -1.0), (5.0, -0.5)])
def test_angles_forces_energy_and_ten_steps(md, case, variant, mode, flags, k_theta, cos0):
    n, clen = CASES[case]
    cfg = scaled_config("chains_rows_1m", n, chain_len=clen)
    for seed, thermal in ((1, False), (2, True)):
        g, o, box = make_pair(md, cfg, seed, k_theta, cos0, variant=variant, mode=mode, flags=flags, thermal=thermal)
        counts, lst = g.neighbors()
        assert sets_equal(counts, lst, o)[0] == 0
        assert force_rel_err(g.forces(), o.forces()) <= FORCE_RTOL
        eg, eo = g.energies(), o.energies()
        assert eg.pe_bond == pytest.approx(eo.pe_bond, rel=ENERGY_RTOL)
        assert eg.pe_pair == pytest.approx(eo.pe_pair, rel=ENERGY_RTOL, abs=1e-9)
        assert eg.virial == pytest.approx(eo.virial, rel=ENERGY_RTOL, abs=1e-7)
        g.step(10)
        assert o.step(10) == 0
        assert pos_err(g.positions(), o.positions(), box) <= POS_ATOL
        eg, eo = g.energies(), o.energies()
        assert eg.ke == pytest.approx(eo.ke, rel=ENERGY_RTOL)
        assert eg.pe == pytest.approx(eo.pe, rel=ENERGY_RTOL)
        g.close()


def test_angles_change_the_forces(md):
    """Guard against a silently ignored call: with k_theta > 0 the forces differ from the FENE-only ones."""
    cfg = scaled_config("chains_rows_1m", 1024, chain_len=16)
    r, v, bonds, box = make_state(cfg, 1)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
    g.set_state(r, v)
    g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    f0, e0 = g.forces(), g.energies().pe_bond
    g.set_angles(3.0, -1.0)
    assert np.abs(g.forces() - f0).max() > 1e-2 and g.energies().pe_bond > e0
    g.set_angles(0.0, -1.0)                                   # k = 0 switches the terms off again
    assert np.array_equal(g.forces(), f0)
    g.close()


def test_angles_call_order_and_unsupported(md):
    cfg = scaled_config("chains_rows_1m", 1024, chain_len=16)
    r, v, bonds, box = make_state(cfg, 1)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
    g.set_state(r, v)
    with pytest.raises(md.MDError):                           # no bond list yet
        g.set_angles(2.0, -1.0)
    g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    with pytest.raises(md.MDError):
        g.set_angles(2.0, -1.5)
    g.step(1)
    with pytest.raises(md.MDError):                           # only before the first step
        g.set_angles(2.0, -1.0)
    g.close()
    for kw in (dict(flags=md.FLAG_TILED_W),):
        g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", **kw)
        g.set_state(r, v)
        g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
        with pytest.raises(md.MDError) as ei:
            g.set_angles(2.0, -1.0)
        assert ei.value.code == md.binding.MD_ERR_UNSUPPORTED
        g.close()


@pytest.mark.parametrize("case", list(CASES))
@pytest.mark.parametrize("mode", ["fused", "split"])
def test_angles_single_precision(md, case, mode):
    """Binary32 variant against the binary32 oracle, bounds of tests/test_gpu_sp.py."""
    from oracle.md_oracle import OracleMDSP
    eps = 2.0 ** -24
    n, clen = CASES[case]
    cfg = scaled_config("chains_rows_1m", n, chain_len=clen)
    r, v, bonds, box = make_state(cfg, 1)
    o = OracleMDSP(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(r, v)
    o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    assert o.set_angles(5.0, -0.5) == 0
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", step_mode=mode, precision="f32")
    g.set_state(r, v)
    g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    g.set_angles(5.0, -0.5)
    fo = o.forces()
    assert np.abs(g.forces() - fo).max() <= 64 * eps * 4 * np.abs(fo).max()
    eg, eo = g.energies(), o.energies()
    assert abs(eg.pe_bond - eo.pe_bond) <= 64 * eps * abs(eo.pe_bond)
    g.step(10)
    assert o.step(10) == 0
    assert pos_err(g.positions(), o.positions(), float(np.float32(box))) <= 16 * float(np.spacing(np.float32(box)))
    eg, eo = g.energies(), o.energies()
    assert abs(eg.pe - eo.pe) <= 64 * eps * max(abs(eo.pe), eo.ke) * 4
    g.close()


@pytest.mark.parametrize("case", list(CASES))
@pytest.mark.parametrize("variant,mode,flags", [("full", "fused", 0), ("full", "split", 0), ("full", "fused", 2),
                                                ("newton3", "split", 0), ("full", "fused", 32)])
@pytest.mark.parametrize("with_angles", [False, True])
def test_dihedrals_forces_energy_and_ten_steps(md, case, variant, mode, flags, with_angles):
    """Dihedral terms (md_set_dihedrals, R19), alone and together with the angle terms."""
    n, clen = CASES[case]
    cfg = scaled_config("chains_rows_1m", n, chain_len=clen)
    for seed, thermal in ((1, False), (2, True)):
        r, v, bonds, box = make_state(cfg, seed)
        o = OracleMD(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
        o.set_state(r, v)
        assert o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0) == 0
        if with_angles:
            assert o.set_angles(3.0, -0.8) == 0          # bent equilibrium keeps the chains away from collinear bonds
        assert o.set_dihedrals(1.5, -0.6) == 0
        if thermal:
            assert o.step(150) == 0
            r, v = o.positions(), o.velocities()
            o.set_state(r, v)
        g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", force_variant=variant,
                        step_mode=mode, flags=flags)
        g.set_state(r, v)
        g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
        if with_angles:
            g.set_angles(3.0, -0.8)
        g.set_dihedrals(1.5, -0.6)
        assert force_rel_err(g.forces(), o.forces()) <= FORCE_RTOL
        eg, eo = g.energies(), o.energies()
        assert eg.pe_bond == pytest.approx(eo.pe_bond, rel=ENERGY_RTOL)
        assert eg.virial == pytest.approx(eo.virial, rel=ENERGY_RTOL, abs=1e-7)
        g.step(10)
        assert o.step(10) == 0
        assert pos_err(g.positions(), o.positions(), box) <= POS_ATOL
        eg, eo = g.energies(), o.energies()
        assert eg.ke == pytest.approx(eo.ke, rel=ENERGY_RTOL)
        assert eg.pe == pytest.approx(eo.pe, rel=ENERGY_RTOL)
        g.close()


def test_dihedrals_change_the_forces_and_unsupported(md):
    cfg = scaled_config("chains_rows_1m", 1000, chain_len=10)
    r, v, bonds, box = make_state(cfg, 1)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
    g.set_state(r, v)
    with pytest.raises(md.MDError):
        g.set_dihedrals(1.0, -1.0)                          # no bond list yet
    g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    f0, e0 = g.forces(), g.energies().pe_bond
    g.set_dihedrals(2.0, 0.5)
    assert np.abs(g.forces() - f0).max() > 1e-2 and g.energies().pe_bond > e0
    g.set_dihedrals(0.0, 0.5)
    assert np.array_equal(g.forces(), f0)
    g.close()
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", flags=md.FLAG_TILED_W)
    g.set_state(r, v)
    g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    with pytest.raises(md.MDError) as ei:
        g.set_dihedrals(1.0, -1.0)
    assert ei.value.code == md.binding.MD_ERR_UNSUPPORTED
    g.close()


@pytest.mark.parametrize("case", list(CASES))
@pytest.mark.parametrize("mode", ["fused", "split"])
def test_dihedrals_single_precision(md, case, mode):
    """Binary32 variant with angle + dihedral terms against the binary32 oracle.  Forces: the dihedral gradient divides by
    |b x b'|^2, so its binary32 rounding is bounded relative to the largest force, 1024 eps (the oracle's own pin SP8)."""
    from oracle.md_oracle import OracleMDSP
    eps = 2.0 ** -24
    n, clen = CASES[case]
    cfg = scaled_config("chains_rows_1m", n, chain_len=clen)
    r, v, bonds, box = make_state(cfg, 1)
    o = OracleMDSP(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(r, v)
    o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    assert o.set_angles(3.0, -0.8) == 0 and o.set_dihedrals(1.5, -0.6) == 0
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", step_mode=mode, precision="f32")
    g.set_state(r, v)
    g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    g.set_angles(3.0, -0.8)
    g.set_dihedrals(1.5, -0.6)
    fo = o.forces()
    assert np.abs(g.forces() - fo).max() <= 1024 * eps * np.abs(fo).max()
    eg, eo = g.energies(), o.energies()
    assert abs(eg.pe_bond - eo.pe_bond) <= 256 * eps * abs(eo.pe_bond)
    g.step(10)
    assert o.step(10) == 0
    assert pos_err(g.positions(), o.positions(), float(np.float32(box))) <= 16 * float(np.spacing(np.float32(box)))
    eg, eo = g.energies(), o.energies()
    assert abs(eg.pe - eo.pe) <= 256 * eps * max(abs(eo.pe), eo.ke) * 4
    g.close()
