"""GPU parity at BASELINE.json's FULL sizes against the stepping oracle: every atom, nothing sampled.

For each config at its real N (configs[1]..[4] with both swept shells of configs[2]) the same state is loaded into the
library and into the oracle; then
  neighbor sets of ALL atoms         exact (sorted integer sets)
  forces of ALL atoms                <= 1e-10 (A11 norm), bonds included for the chain workload
  energies, virial, vmax             1e-9 relative
and after md_step(10) / orc_step(10)
  positions                          <= 1e-9 (component-wise, modulo L)
  ke, pe                             1e-9 relative;  momentum 1e-9 sqrt(N) absolute
  n_rebuilds                         equal;  vmax 1e-9 relative
from the seeded start and from a state melted on the GPU and injected into both sides with md_set_state / orc_set_state.
The launch configuration is the one bench.py times (default flags, fused steps, CUDA graph); variant B, the forced W
layouts and the single-precision twin are run once each at full size.
"""
import numpy as np
import pytest

from md_workloads import get_config
from oracle.md_oracle import OracleMD, OracleMDSP
from parity_util import ENERGY_RTOL, FORCE_RTOL, POS_ATOL, force_rel_err, pos_err, sets_equal, prepared_state

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def md():
    import paper_2003_14061_b200 as m
    m.load_library()
    return m


def _pair(md, cfg, seed, melt_steps, oracle_cls=OracleMD, **kw):
    r, v, bonds, box = prepared_state(md, cfg, seed)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", **kw)
    g.set_state(r, v)
    if bonds is not None:
        g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    if melt_steps:
        g.step(melt_steps)
        r, v = g.positions(), g.velocities()
        g.set_state(r, v)                     # resets the step / rebuild counters and the displacement accumulator
    o = oracle_cls(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(r, v)
    if bonds is not None:
        assert o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0) == 0
    return g, o, box


def _check_static(g, o, cfg, lattice_start):
    counts, lst = g.neighbors()
    nbad, first = sets_equal(counts, lst, o)
    assert nbad == 0, f"neighbor sets differ for {nbad} atoms (first: atom {first})"
    del lst
    fo, fg = o.forces(), g.forces()
    if lattice_start and cfg.lattice in ("sc", "fcc"):
        assert np.abs(fg).max() <= 1e-12 * 24.0 * 78 and np.abs(fo).max() <= 1e-12 * 24.0 * 78
    else:
        assert force_rel_err(fg, fo) <= FORCE_RTOL
    eg, eo = g.energies(), o.energies()
    assert eg.pe_pair == pytest.approx(eo.pe_pair, rel=ENERGY_RTOL, abs=1e-9)
    assert eg.pe_bond == pytest.approx(eo.pe_bond, rel=ENERGY_RTOL, abs=1e-9)
    assert eg.virial == pytest.approx(eo.virial, rel=ENERGY_RTOL, abs=1e-7)
    assert eg.ke == pytest.approx(eo.ke, rel=1e-12)
    assert eg.vmax == pytest.approx(eo.vmax, rel=1e-12)
    assert eg.mean_neighbors == pytest.approx(eo.mean_neighbors, rel=1e-12)


def _check_ten_steps(g, o, cfg, box):
    g.step(10)
    assert o.step(10) == 0
    assert pos_err(g.positions(), o.positions(), box) <= POS_ATOL
    assert np.abs(g.velocities() - o.velocities()).max() <= 1e-8
    eg, eo = g.energies(), o.energies()
    assert eg.ke == pytest.approx(eo.ke, rel=ENERGY_RTOL)
    assert eg.pe == pytest.approx(eo.pe, rel=ENERGY_RTOL)
    assert eg.vmax == pytest.approx(eo.vmax, rel=ENERGY_RTOL)
    assert eg.step == eo.step == 10
    assert eg.n_rebuilds == eo.n_rebuilds
    for pg, po in ((eg.px, eo.px), (eg.py, eo.py), (eg.pz, eo.pz)):
        assert abs(pg - po) <= 1e-9 * np.sqrt(cfg.n_atoms)


FULL = ["wca_262k", "wca_2m_dr03", "wca_2m", "wca_2m_dr05", "lj_1m", "chains_1m"]


@pytest.mark.parametrize("name", FULL)
@pytest.mark.parametrize("start", ["seeded", "melted"])
def test_full_size_all_atoms_and_ten_steps(md, name, start):
    cfg = get_config(name)
    g, o, box = _pair(md, cfg, 1, 200 if start == "melted" else 0)
    assert g.info()["n_atoms"] == cfg.n_atoms
    _check_static(g, o, cfg, start == "seeded")
    _check_ten_steps(g, o, cfg, box)
    # the launch configuration bench.py times: one cooperative launch up to 400,000 atoms, the step graph above
    assert g.info()["use_graph"] == (2 if cfg.n_atoms <= 400_000 else 1)
    g.close()


@pytest.mark.parametrize("seed", [2, 3])
def test_full_size_other_seeds(md, seed):
    cfg = get_config("wca_2m_dr05")
    g, o, box = _pair(md, cfg, seed, 60)
    _check_static(g, o, cfg, False)
    _check_ten_steps(g, o, cfg, box)
    g.close()


@pytest.mark.parametrize("name,kw", [
    ("lj_1m", dict(force_variant="newton3", step_mode="split")),       # variant B, half list + fp64 atomics
    ("lj_1m", dict(flags=8)),                                          # MD_FLAG_GATHER_W: long columns through the gathering kernels
    ("lj_1m", dict(flags=4, step_mode="split")),                       # MD_FLAG_TILED_W, split steps
    ("wca_2m", dict(flags=4)),                                         # MD_FLAG_TILED_W forced on short columns
    ("wca_2m", dict(flags=2)),                                         # MD_FLAG_GLOBAL_W: the paper's literal data path
    ("wca_2m", dict(force_variant="newton3", step_mode="split")),
    ("chains_1m", dict(step_mode="split")),
])
def test_full_size_variants(md, name, kw):
    cfg = get_config(name)
    g, o, box = _pair(md, cfg, 1, 100, **kw)
    _check_static(g, o, cfg, False)
    _check_ten_steps(g, o, cfg, box)
    g.close()


@pytest.mark.parametrize("name", ["wca_262k", "wca_2m", "lj_1m", "chains_1m"])
def test_full_size_single_precision(md, name):
    """The single-precision twin against the single-precision oracle at full size (bounds of tests/test_gpu_sp.py).
    wca_262k runs as the persistent launch (k_sp_persist, grid-stride instantiation), the others as the step graph."""
    eps32 = 2.0 ** -24
    cfg = get_config(name)
    g, o, box = _pair(md, cfg, 1, 100, oracle_cls=OracleMDSP, precision="f32")
    counts, lst = g.neighbors()
    nbad, first = sets_equal(counts, lst, o)
    assert nbad == 0, f"neighbor sets differ for {nbad} atoms (first: atom {first})"
    del lst
    fo = o.forces()
    assert np.abs(g.forces() - fo).max() <= 64 * eps32 * 4 * np.abs(fo).max()
    g.step(10)
    assert o.step(10) == 0
    ulp_L = float(np.spacing(np.float32(box)))
    assert pos_err(g.positions(), o.positions(), float(np.float32(box))) <= 16 * ulp_L
    eg, eo = g.energies(), o.energies()
    escale = max(abs(eo.pe), eo.ke)
    assert abs(eg.ke - eo.ke) <= 64 * eps32 * escale
    assert abs(eg.pe - eo.pe) <= 64 * eps32 * escale * 4
    assert eg.n_rebuilds == eo.n_rebuilds
    assert g.info()["use_graph"] == (2 if cfg.n_atoms <= 400_000 else 1)
    g.close()
