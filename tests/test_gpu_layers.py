"""GPU parity of the ablation MD_FLAG_LAYER_H -- the paper's own cell structure (dense cell x layer matrix H filled
from the atomic slots) and sort schedule (atoms re-sorted every `reorder_interval` steps or never,
PAPER.md:80, 159) -- against the same oracle and tolerances as the default path."""
import numpy as np
import pytest

from md_workloads import get_config, make_state, scaled_config
from oracle.md_oracle import OracleMD
from parity_util import ENERGY_RTOL, FORCE_RTOL, POS_ATOL, force_rel_err, pos_err, sets_equal

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def md():
    import paper_2003_14061_b200 as m
    m.load_library()
    return m


def cases():
    return {
        "wca_4k": get_config("wca_4k"),
        "wca_ragged_1000": scaled_config("wca_4k", 1000),
        "lj_6912": scaled_config("lj_1m", 4 * 12 ** 3),
        "chains_4096": scaled_config("chains_rows_1m", 4096, chain_len=16),
    }


def shuffled_state(cfg, seed, shuffle):
    """State of md_workloads, optionally with the atom numbering permuted (a decorrelated storage order: what a long
    run without sorting tends to)."""
    r, v, bonds, box = make_state(cfg, seed, jitter_amp=0.12 if cfg.lattice != "chains" else 0.0)
    if shuffle:
        perm = np.random.default_rng(100 + seed).permutation(cfg.n_atoms)        # new id k holds old atom perm[k]
        inv = np.empty_like(perm)
        inv[perm] = np.arange(cfg.n_atoms)
        r, v = r[perm], v[perm]
        if bonds is not None:
            bonds = inv[bonds].astype(np.int32)
    return r, v, bonds, box


def make_pair(md, cfg, seed, interval, shuffle, mode="fused"):
    r, v, bonds, box = shuffled_state(cfg, seed, shuffle)
    o = OracleMD(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(r, v)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", step_mode=mode,
                    flags=md.FLAG_LAYER_H, reorder_interval=interval)
    g.set_state(r, v)
    if bonds is not None:
        assert o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0) == 0
        g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    return g, o, box


@pytest.mark.parametrize("case", list(cases()))
@pytest.mark.parametrize("interval", [0, 7, -1])
@pytest.mark.parametrize("shuffle", [False, True])
def test_layers_sets_forces_and_ten_steps(md, case, interval, shuffle):
    cfg = cases()[case]
    for seed in (1, 2):
        g, o, box = make_pair(md, cfg, seed, interval, shuffle)
        info = g.info()
        assert info["n_layers"] >= 8 and info["w_layout"] == 0
        counts, lst = g.neighbors()
        nbad, first = sets_equal(counts, lst, o)
        assert nbad == 0, f"neighbor sets differ for {nbad} atoms (first: atom {first})"
        assert force_rel_err(g.forces(), o.forces()) <= FORCE_RTOL
        eg, eo = g.energies(), o.energies()
        assert eg.pe == pytest.approx(eo.pe, rel=ENERGY_RTOL)
        assert eg.max_cell_occupancy == eo.max_cell_occupancy
        g.step(10)
        assert o.step(10) == 0
        assert pos_err(g.positions(), o.positions(), box) <= POS_ATOL
        eg, eo = g.energies(), o.energies()
        assert eg.ke == pytest.approx(eo.ke, rel=ENERGY_RTOL)
        assert eg.pe == pytest.approx(eo.pe, rel=ENERGY_RTOL)
        assert eg.n_rebuilds == eo.n_rebuilds
        g.close()


@pytest.mark.parametrize("interval", [7, 20, -1])
@pytest.mark.parametrize("mode", ["fused", "split"])
def test_layers_later_rebuilds_sorted_and_in_place(md, interval, mode):
    """60 steps: several rebuilds, some with and some without the sort.  Then the matrix rebuilt from the GPU's own
    coordinates equals the definition evaluated by the oracle on those coordinates, and the trajectory has stayed with
    the oracle's (bound for 60 steps: 6 x the 10-step bound)."""
    cfg = get_config("wca_4k")
    g, o, box = make_pair(md, cfg, 3, interval, True, mode=mode)
    g.step(60)
    assert o.step(60) == 0
    assert g.energies().n_rebuilds == o.energies().n_rebuilds >= 4
    assert pos_err(g.positions(), o.positions(), box) <= 6 * POS_ATOL
    r, v = g.positions(), g.velocities()
    g.rebuild_neighbors()
    o2 = OracleMD(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    o2.set_state(r, v)
    counts, lst = g.neighbors()
    nbad, first = sets_equal(counts, lst, o2)
    assert nbad == 0, f"neighbor sets differ for {nbad} atoms (first: atom {first})"
    assert force_rel_err(g.forces(), o2.forces()) <= FORCE_RTOL
    g.close()


def test_layers_reject_unsupported(md):
    cfg = get_config("wca_4k")
    for kw in (dict(precision="f32"), dict(force_variant="newton3"), dict(n_systems=2)):
        with pytest.raises(md.MDError):
            md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, density=cfg.density, flags=md.FLAG_LAYER_H, **kw)


def test_layers_cell_overflow_is_reported(md):
    """More atoms in one cell than N_l: MD_ERR_CELL_OVERFLOW, never a silently short H row."""
    cfg = scaled_config("wca_4k", 1000)
    r, v, _, box = make_state(cfg, 1, jitter_amp=0.05)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", flags=md.FLAG_LAYER_H,
                    max_neighbors=256)
    nl = g.info()["n_layers"]
    w = g.info()["cell_width"]
    r = r.copy()
    rng = np.random.default_rng(0)
    r[: nl + 4] = 0.25 * w + 0.5 * w * rng.random((nl + 4, 3))        # nl + 4 atoms into the first cell
    with pytest.raises(md.MDError) as ei:
        g.set_state(r, v)
    assert ei.value.code == md.binding.MD_ERR_CELL_OVERFLOW
    g.close()
