"""md_pushoff: BASELINE.json configs[4] "chains grown as seeded random walks then pushed apart".

The push-off is initialisation outside the parity-checked path, so it is pinned by invariants only, each checked here
with independent host arithmetic (scipy k-d tree, numpy): every bond in (0.7, 1.3), smallest non-bonded distance above
0.85, zero total momentum, temperature as asked, bonds and ids intact, and the state it loads is the state a plain
md_set_state + md_set_bonds of the same arrays gives (so the oracle can be handed the result as data)."""
import numpy as np
import pytest
from scipy.spatial import cKDTree

from md_workloads import gaussian_velocities, get_config, make_state, scaled_config
from oracle.md_oracle import OracleMD
from parity_util import FORCE_RTOL, force_rel_err, sets_equal

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def md():
    import paper_2003_14061_b200 as m
    m.load_library()
    return m


def invariants(r, v, bonds, box, n, temperature):
    d = r[bonds[:, 0]] - r[bonds[:, 1]]
    d -= box * np.round(d / box)
    bl = np.sqrt((d * d).sum(1))
    pairs = cKDTree(r, boxsize=box).query_pairs(0.85, output_type="ndarray")
    key = set(map(tuple, np.sort(bonds, 1)))
    close = [p for p in map(tuple, np.sort(pairs, 1)) if p not in key]
    return bl.min(), bl.max(), len(close), np.abs(v.sum(0)).max(), (v * v).sum() / (3 * (n - 1))


@pytest.mark.parametrize("n,chain_len,kw", [(4096, 16, {}), (3000, 10, {}), (16384, 64, {}), (4096, 16, dict(precision="f32")),
                                            (4096, 16, dict(flags=4))])
def test_pushoff_invariants(md, n, chain_len, kw):
    cfg = scaled_config("chains_1m", n, chain_len=chain_len)
    for seed in (1, 2):
        r0, _, bonds, box = make_state(cfg, seed)
        assert r0.min() >= 0 and r0.max() < box
        g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", **kw)
        rep = g.pushoff(r0, bonds, cfg.fene_k, cfg.fene_r0, temperature=cfg.temperature, seed=seed)
        assert rep["min_nonbonded_start"] < 0.5 < 0.85 < rep["min_nonbonded"] and rep["max_bond"] < 1.3 and rep["steps"] >= 3000
        r, v = g.positions(), g.velocities()
        bmin, bmax, nclose, pmax, T = invariants(r, v, bonds, box, n, cfg.temperature)
        assert 0.7 < bmin and bmax < 1.3 and nclose == 0
        assert bmax == pytest.approx(rep["max_bond"], abs=1e-6 if kw.get("precision") == "f32" else 1e-12)
        f32 = kw.get("precision") == "f32"              # velocities rounded to binary32 on entry: momentum ~ sqrt(N) eps32 |v|
        assert pmax < (1e-4 if f32 else 1e-9) and T == pytest.approx(cfg.temperature, rel=1e-5 if f32 else 1e-9)
        if not kw.get("precision"):
            assert np.abs(v - gaussian_velocities(n, cfg.temperature, seed)).max() < 1e-12        # fresh velocities, recipe O2
        # the loaded state behaves like any other: it steps, conserves energy, and the bonds hold
        e0 = g.energies()
        g.step(200)
        e1 = g.energies()
        assert abs(e1.total - e0.total) / n < (5e-3 if not kw.get("precision") else 2e-2)
        assert e1.pe_bond > 0 and e1.n_rebuilds > 5
        g.close()


def test_pushoff_result_is_plain_data_for_the_oracle(md):
    """The pushed-off arrays, loaded into a fresh system and into the oracle, agree as any other state does."""
    cfg = scaled_config("chains_1m", 4096, chain_len=16)
    r0, _, bonds, box = make_state(cfg, 3)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
    g.pushoff(r0, bonds, cfg.fene_k, cfg.fene_r0, temperature=cfg.temperature, seed=3)
    r, v = g.positions(), g.velocities()
    f_after_pushoff = g.forces()
    g.close()
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
    g.set_state(r, v)
    g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    assert np.array_equal(g.forces(), f_after_pushoff)
    o = OracleMD(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(r, v)
    assert o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0) == 0
    counts, lst = g.neighbors()
    assert sets_equal(counts, lst, o)[0] == 0
    assert force_rel_err(g.forces(), o.forces()) <= FORCE_RTOL
    g.close()


def test_pushoff_reports_failure_and_bad_arguments(md):
    cfg = scaled_config("chains_1m", 4096, chain_len=16)
    r0, _, bonds, box = make_state(cfg, 1)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
    with pytest.raises(md.MDError) as ei:                        # far too few steps for the criteria
        g.pushoff(r0, bonds, cfg.fene_k, cfg.fene_r0, ramp_steps=50, max_steps=100, check_interval=50)
    assert ei.value.code == md.binding.MD_ERR_UNSUPPORTED
    bad = r0.copy()
    bad[7, 1] = -1.0
    with pytest.raises(md.MDError) as ei:
        g.pushoff(bad, bonds, cfg.fene_k, cfg.fene_r0)
    assert ei.value.code == md.binding.MD_ERR_INVALID
    g.close()


def test_full_size_pushoff_config5(md):
    """configs[4] at its real size: 16,384 walks of 64 beads."""
    cfg = get_config("chains_1m")
    r0, _, bonds, box = make_state(cfg, 1)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
    rep = g.pushoff(r0, bonds, cfg.fene_k, cfg.fene_r0, temperature=cfg.temperature, seed=1)
    r, v = g.positions(), g.velocities()
    bmin, bmax, nclose, pmax, T = invariants(r, v, bonds, box, cfg.n_atoms, cfg.temperature)
    assert 0.7 < bmin and bmax < 1.3 and nclose == 0 and pmax < 1e-8 and T == pytest.approx(1.0, rel=1e-9)
    assert rep["min_nonbonded"] > 0.85
    g.close()
