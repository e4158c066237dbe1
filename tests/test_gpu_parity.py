"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.
Tolerances are BASELINE.json north_star's: neighbor sets exact, forces 1e-10, positions 1e-9 and energies 1e-9
after 10 steps."""
import numpy as np
import pytest

from md_workloads import get_config, make_state, scaled_config
from oracle.md_oracle import OracleMD, brute_forces_sample, brute_neighbors_sample
from parity_util import ENERGY_RTOL, FORCE_RTOL, POS_ATOL, force_rel_err, pos_err, prepared_state, sets_equal

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def md():
    import paper_2003_14061_b200 as m
    m.load_library()
    return m


def small_cases():
    return {
        "wca_4k": (get_config("wca_4k"), {}),
        "wca_ragged_1000": (scaled_config("wca_4k", 1000), {}),                     # N not a multiple of 32/128
        "wca_dr03_13824": (scaled_config("wca_2m_dr03", 24 ** 3), {}),
        "wca_dr05_13824": (scaled_config("wca_2m_dr05", 24 ** 3), {}),
        "lj_6912": (scaled_config("lj_1m", 4 * 12 ** 3), {}),
        "chains_4096": (scaled_config("chains_rows_1m", 4096, chain_len=16), {}),
        # BASELINE.json configs[4] scaled down: seeded random walks pushed apart by the library (md_pushoff)
        "walk_4096": (scaled_config("chains_1m", 4096, chain_len=16), {}),
    }


def make_pair(md, cfg, seed, variant="full", mode="fused", state="jitter", **kw):
    """GPU system and oracle loaded with the SAME state (from md_workloads or evolved by the oracle)."""
    jit = 0.0 if state == "lattice" else (0.12 if cfg.lattice in ("sc", "fcc") else 0.0)
    r, v, bonds, box = prepared_state(md, cfg, seed, jitter_amp=jit)
    o = OracleMD(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(r, v)
    if bonds is not None:
        assert o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0) == 0
    if state == "thermal":
        assert o.step(200) == 0
        r, v = o.positions(), o.velocities()
        o.set_state(r, v)
        if bonds is not None:
            o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    if variant == "full-globalw":          # variant A on the paper's literal data path (global indices, L1/L2 gathers)
        variant, kw = "full", dict(kw, flags=md.FLAG_GLOBAL_W)
    elif variant == "full-gatherw":        # tile-staged build, global W, gathering force kernel (the default for short columns)
        variant, kw = "full", dict(kw, flags=md.FLAG_GATHER_W)
    elif variant == "full-transposed":     # ablation: W stored atom-index-slowest
        variant, kw = "full", dict(kw, flags=md.FLAG_W_TRANSPOSED | md.FLAG_GATHER_W)
    elif variant == "full-tiledw":         # variant A with 16-bit tile-local W entries and shared-memory force kernels
        variant, kw = "full", dict(kw, flags=md.FLAG_TILED_W)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", force_variant=variant,
                    step_mode=mode, **kw)
    g.set_state(r, v)
    if bonds is not None:
        g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    return g, o, box


@pytest.mark.parametrize("case", list(small_cases()))
@pytest.mark.parametrize("variant", ["full", "full-globalw", "full-gatherw", "full-tiledw", "full-transposed", "newton3"])
@pytest.mark.parametrize("state", ["lattice", "jitter", "thermal"])
def test_neighbor_sets_and_forces(md, case, variant, state):
    cfg, _ = small_cases()[case]
    if state == "lattice" and cfg.lattice in ("chains", "walk"):
        pytest.skip("chain start has no separate lattice state")
    for seed in (1, 2, 3) if state != "thermal" else (1,):
        g, o, box = make_pair(md, cfg, seed, variant=variant, mode="split", state=state)
        counts, lst = g.neighbors()
        nbad, first = sets_equal(counts, lst, o)
        assert nbad == 0, f"neighbor sets differ for {nbad} atoms (first: atom {first})"
        fo = o.forces()
        fg = g.forces()
        if state == "lattice" and cfg.lattice in ("sc", "fcc"):
            # every f_i = 0 analytically: only an absolute test makes sense;
            # a single pair force is < 24 and at most 78 pairs contribute
            assert np.abs(fg).max() <= 1e-12 * 24.0 * 78 and np.abs(fo).max() <= 1e-12 * 24.0 * 78
        else:
            assert force_rel_err(fg, fo) <= FORCE_RTOL
        eg, eo = g.energies(), o.energies()
        assert eg.pe_pair == pytest.approx(eo.pe_pair, rel=ENERGY_RTOL, abs=1e-9)
        assert eg.pe_bond == pytest.approx(eo.pe_bond, rel=ENERGY_RTOL, abs=1e-9)
        assert eg.virial == pytest.approx(eo.virial, rel=ENERGY_RTOL, abs=1e-7)
        assert eg.ke == pytest.approx(eo.ke, rel=1e-12)
        if variant != "newton3":                                 # variant B stores (and reports) the half matrix
            assert eg.max_neighbors == eo.max_neighbors
        assert eg.mean_neighbors == pytest.approx(eo.mean_neighbors, rel=1e-12)
        g.close()


@pytest.mark.parametrize("case", list(small_cases()))
@pytest.mark.parametrize("variant,mode", [("full", "fused"), ("full", "split"), ("full-globalw", "fused"),
                                          ("full-globalw", "split"), ("full-tiledw", "fused"), ("full-tiledw", "split"), ("full-transposed", "fused"),
                                          ("newton3", "split")])
def test_ten_steps(md, case, variant, mode):
    cfg, _ = small_cases()[case]
    for seed in (1, 2, 3):
        g, o, box = make_pair(md, cfg, seed, variant=variant, mode=mode, state="jitter")
        g.step(10)
        assert o.step(10) == 0
        assert pos_err(g.positions(), o.positions(), box) <= POS_ATOL
        assert np.abs(g.velocities() - o.velocities()).max() <= 1e-8
        eg, eo = g.energies(), o.energies()
        assert eg.ke == pytest.approx(eo.ke, rel=ENERGY_RTOL)
        assert eg.pe == pytest.approx(eo.pe, rel=ENERGY_RTOL)
        assert eg.step == eo.step == 10
        n = cfg.n_atoms
        for pg, po in ((eg.px, eo.px), (eg.py, eo.py), (eg.pz, eo.pz)):
            assert abs(pg - po) <= 1e-9 * np.sqrt(n)
        assert force_rel_err(g.forces(), o.forces()) <= 1e-8     # after 10 steps positions differ by ~1e-13
        g.close()


def test_steps_one_at_a_time_equal_one_call(md):
    """md_step(1) x 10 (closing/opening half kicks each call) and md_step(10) (fused leapfrog) agree."""
    cfg = get_config("wca_4k")
    g1, o, box = make_pair(md, cfg, 1, mode="fused")
    g2, _, _ = make_pair(md, cfg, 1, mode="fused")
    for _ in range(10):
        g1.step(1)
    g2.step(10)
    assert pos_err(g1.positions(), g2.positions(), box) <= 1e-12
    assert np.abs(g1.velocities() - g2.velocities()).max() <= 1e-12


def test_thermalised_run_with_rebuilds(md):
    """200 steps from the lattice (about 20 rebuilds): the list must stay valid, so energies track the oracle's
    to chaos-limited accuracy and the conserved quantities hold."""
    cfg = get_config("wca_4k")
    g, o, box = make_pair(md, cfg, 1, mode="fused", state="lattice")
    e0 = g.energies()
    g.step(200)
    o.step(200)
    eg, eo = g.energies(), o.energies()
    assert eg.n_rebuilds > 10 and abs(eg.n_rebuilds - eo.n_rebuilds) <= 1
    assert abs(eg.total - e0.total) / cfg.n_atoms < 2e-3
    assert eg.total == pytest.approx(eo.total, rel=1e-7)
    assert max(abs(eg.px), abs(eg.py), abs(eg.pz)) < 1e-9
    # forces on the GPU's own final state against the all-pairs definition (list validity)
    pos = g.positions()
    idx = np.arange(0, cfg.n_atoms, 7)
    fb, _, _ = brute_forces_sample(pos, box, cfg.r_cut, idx)
    assert force_rel_err(g.forces()[idx], fb) <= FORCE_RTOL


def test_md_create_initial_state_matches_generator(md):
    for name in ("wca_4k", "lj_6912"):
        cfg = small_cases()[name][0]
        r, v, _, box = make_state(cfg, 5)
        g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, density=cfg.density, seed=5,
                        temperature=cfg.temperature)
        assert np.abs(g.positions() - r).max() < 1e-12
        assert np.abs(g.velocities() - v).max() < 1e-12
        e = g.energies()
        assert e.ke == pytest.approx(1.5 * (cfg.n_atoms - 1) * cfg.temperature, rel=1e-12)
        g.close()


def test_runs_are_bitwise_reproducible(md):
    cfg = get_config("wca_4k")
    out = []
    for _ in range(2):
        g, _, _ = make_pair(md, cfg, 2, mode="fused")
        g.step(120)
        out.append((g.positions(), g.velocities(), g.forces()))
        g.close()
    for a, b in zip(*out):
        assert np.array_equal(a, b)


def test_medium_system_full_comparison(md):
    """configs[1] size (N = 262,144): spans ~2000 blocks; the oracle's cell search handles it in seconds."""
    cfg = get_config("wca_262k")
    g, o, box = make_pair(md, cfg, 1, mode="fused")
    counts, lst = g.neighbors()
    assert sets_equal(counts, lst, o)[0] == 0
    assert force_rel_err(g.forces(), o.forces()) <= FORCE_RTOL
    g.step(10)
    o.step(10)
    assert pos_err(g.positions(), o.positions(), box) <= POS_ATOL
    eg, eo = g.energies(), o.energies()
    assert eg.ke == pytest.approx(eo.ke, rel=ENERGY_RTOL) and eg.pe == pytest.approx(eo.pe, rel=ENERGY_RTOL)


TILE_GEOMS = [dict(S=1, R=1, RZ=1, THREADS=128), dict(S=2, R=3, RZ=1, THREADS=128), dict(S=3, R=2, RZ=3, THREADS=256),
              dict(S=1000, R=3, RZ=3, THREADS=512), dict(S=4, R=1, RZ=2, THREADS=256), dict(S=5, R=2, RZ=2, THREADS=128)]


@pytest.mark.parametrize("case", ["wca_ragged_1000", "wca_dr05_13824", "lj_6912", "chains_4096", "walk_4096"])
@pytest.mark.parametrize("geom", range(len(TILE_GEOMS)))
@pytest.mark.parametrize("variant", ["full-gatherw", "full-tiledw"])
def test_tile_staging_any_box_shape(md, case, geom, variant):
    """The shared-memory staged build (default) and the tiled W layout must give the same matrix, forces and trajectory for every box shape S x R x RZ and
    block size (boxes cut by the periodic faces, boxes wider than the system, blocks looping over their atoms)."""
    cfg, _ = small_cases()[case]
    G = TILE_GEOMS[geom]
    g, o, box = make_pair(md, cfg, 2, variant=variant, mode="fused", state="jitter", tile_cells=(G["S"], G["R"], G["RZ"]),
                          tile_threads=G["THREADS"], tile_capacity=8192)
    info = g.info()
    assert info["w_layout"] == (1 if variant == "full-tiledw" else 0) and info["tile_cells"][1:] == [TILE_GEOMS[geom]["R"], TILE_GEOMS[geom]["RZ"]]
    counts, lst = g.neighbors()
    nbad, first = sets_equal(counts, lst, o)
    assert nbad == 0, f"neighbor sets differ for {nbad} atoms (first: atom {first})"
    assert force_rel_err(g.forces(), o.forces()) <= FORCE_RTOL
    g.step(10)
    o.step(10)
    assert pos_err(g.positions(), o.positions(), box) <= POS_ATOL
    eg, eo = g.energies(), o.energies()
    assert eg.ke == pytest.approx(eo.ke, rel=ENERGY_RTOL) and eg.pe == pytest.approx(eo.pe, rel=ENERGY_RTOL)
    g.close()


def test_tile_overflow_is_reported(md):
    """A tile that cannot hold the mean cell neighbourhood is refused at create (tiled W) or replaced by the gathering
    build kernel (default layout); a neighbourhood that outgrows its tile at run time is an error code, never a
    truncated matrix."""
    cfg = get_config("wca_4k")
    r, v, _, box = make_state(cfg, 1, jitter_amp=0.0)
    with pytest.raises(md.MDError):
        md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", flags=md.FLAG_TILED_W, tile_capacity=64)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", tile_capacity=64)
    g.set_state(r, v)
    assert g.info()["tile_capacity"] == 0          # fell back to the gathering build kernel
    g.close()
    squeezed = r.copy()
    squeezed[:, 1] *= 0.5                          # density x 2 in half of the box (along y: a tile spans all of x)
    for flags in (md.FLAG_GATHER_W, md.FLAG_TILED_W):
        g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", flags=flags,
                        max_neighbors=64)
        with pytest.raises(md.MDError) as ei:
            g.set_state(squeezed, v)
        assert ei.value.code == md.binding.MD_ERR_TILE_OVERFLOW
        g.close()
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", flags=md.FLAG_GLOBAL_W,
                    max_neighbors=64)
    g.set_state(squeezed, v)                       # the literal path has no tile and takes any density
    g.close()


@pytest.mark.parametrize("name", ["wca_2m", "wca_2m_dr03", "wca_2m_dr05", "lj_1m", "chains_1m"])
def test_full_size_sampled_against_definitions(md, name):
    """BASELINE.json's full sizes in the launch configuration bench.py times (default flags, fused steps, CUDA graph):
    after 40 steps from the seeded start, sampled atoms are checked one by one against the all-pairs definitions
    (neighbor sets exact, forces 1e-10), and the conserved quantities against the start."""
    cfg = get_config(name)
    r, v, bonds, box = prepared_state(md, cfg, 1)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
    g.set_state(r, v)
    if bonds is not None:
        g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    n = cfg.n_atoms
    e0 = g.energies()
    g.step(40)
    e1 = g.energies()
    assert g.info()["use_graph"] == 1 and e1.n_rebuilds >= 2
    assert abs(e1.total - e0.total) / n < 2e-3
    assert max(abs(e1.px), abs(e1.py), abs(e1.pz)) < 1e-9 * np.sqrt(n) * 10
    g.rebuild_neighbors()                       # W and forces for the current (wrapped) positions
    pos = g.positions()
    assert pos.min() >= 0.0 and pos.max() < box
    rng = np.random.default_rng(7)
    idx = np.sort(rng.choice(n, 400, replace=False))
    counts, lst = g.neighbors()
    want = brute_neighbors_sample(pos, box, cfg.r_cut + cfg.r_shell, idx)
    for k, i in enumerate(idx):
        got = np.sort(lst[i, :counts[i]])
        assert np.array_equal(got, want[k]), f"neighbor set of atom {i} differs"
    del lst
    if bonds is None:                           # the all-pairs definition has no bond term
        fb, _, _ = brute_forces_sample(pos, box, cfg.r_cut, idx)
        assert force_rel_err(g.forces()[idx], fb) <= FORCE_RTOL
    g.close()


@pytest.mark.parametrize("case,n_sys", [("wca_ragged_1000", 5), ("wca_4k", 3), ("lj_6912", 2), ("chains_4096", 2)])
@pytest.mark.parametrize("variant", ["full", "full-globalw", "full-tiledw", "newton3"])
def test_batched_independent_systems(md, case, n_sys, variant):
    """n_systems mutually invisible systems in one set of kernel launches: every system must follow its
    own oracle exactly as if it were alone -- neighbor sets exact (global ids), forces 1e-10, 10 steps 1e-9."""
    cfg, _ = small_cases()[case]
    n = cfg.n_atoms
    states = [make_state(cfg, 10 + b, jitter_amp=0.12 if cfg.lattice != "chains" else 0.0) for b in range(n_sys)]
    box = states[0][3]
    kw = {}
    fv = variant
    if variant == "full-globalw":
        fv, kw = "full", dict(flags=md.FLAG_GLOBAL_W)
    elif variant == "full-tiledw":
        fv, kw = "full", dict(flags=md.FLAG_TILED_W)
    g = md.MDSystem(n, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", force_variant=fv,
                    step_mode="fused" if fv == "full" else "split", n_systems=n_sys, **kw)
    g.set_state(np.concatenate([s[0] for s in states]), np.concatenate([s[1] for s in states]))
    oracles = []
    for b, (r, v, bonds, _) in enumerate(states):
        o = OracleMD(n, box, cfg.r_cut, cfg.r_shell, cfg.dt)
        o.set_state(r, v)
        if bonds is not None:
            assert o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0) == 0
        oracles.append(o)
    if states[0][2] is not None:
        g.set_bonds(np.concatenate([s[2] + b * n for b, s in enumerate(states)]), cfg.fene_k, cfg.fene_r0)
    assert g.info()["n_systems"] == n_sys and g.info()["n_atoms"] == n
    counts, lst = g.neighbors()
    fg = g.forces()
    for b, o in enumerate(oracles):
        sl = slice(b * n, (b + 1) * n)
        rows = np.where(lst[sl] >= 0, lst[sl] - b * n, -1)
        assert ((rows < n) | (lst[sl] < 0)).all() and (rows[lst[sl] >= 0] >= 0).all()      # no partner in another system
        nbad, first = sets_equal(counts[sl], rows, o)
        assert nbad == 0, f"system {b}: neighbor sets differ for {nbad} atoms (first: atom {first})"
        assert force_rel_err(fg[sl], o.forces()) <= FORCE_RTOL
    g.step(10)
    pg, eg = g.positions(), g.energies()
    ke = pe = 0.0
    for b, o in enumerate(oracles):
        assert o.step(10) == 0
        assert pos_err(pg[b * n:(b + 1) * n], o.positions(), box) <= POS_ATOL
        eo = o.energies()
        ke, pe = ke + eo.ke, pe + eo.pe
    assert eg.ke == pytest.approx(ke, rel=ENERGY_RTOL) and eg.pe == pytest.approx(pe, rel=ENERGY_RTOL)
    g.close()


def test_batched_systems_created_from_the_lattice(md):
    cfg = get_config("wca_4k")
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, density=cfg.density, seed=5, temperature=1.0, n_systems=4)
    r, v = g.positions(), g.velocities()
    n = cfg.n_atoms
    for b in range(4):
        rb, vb, _, _ = make_state(cfg, 5 + b)
        assert np.abs(r[b * n:(b + 1) * n] - rb).max() < 1e-12 and np.abs(v[b * n:(b + 1) * n] - vb).max() < 1e-12
    e0 = g.energies()
    assert e0.ke == pytest.approx(4 * 1.5 * (n - 1) * 1.0, rel=1e-12)          # every system at exactly T = 1
    g.step(30)
    e1 = g.energies()
    assert abs(e1.total - e0.total) / (4 * n) < 2e-3 and e1.n_rebuilds >= 2
    g.close()


@pytest.mark.parametrize("variant,mode", [("full", "fused"), ("full", "split"), ("full-globalw", "fused"), ("full-tiledw", "fused"),
                                          ("full-tiledw", "split"), ("newton3", "split")])
@pytest.mark.parametrize("hot", [0, 2])
def test_batched_rebuild_follows_the_hottest_system(md, variant, mode, hot):
    """One rebuild decision serves all systems of a batch (include/md_b200.h: "the largest velocity of any system").
    Three systems, one of them hot and the others at rest: the rebuild count must be the HOT system's oracle count
    whichever slot it sits in, and after the run every system's matrix must still hold all its interacting pairs
    (forces against the all-pairs definition)."""
    cfg = scaled_config("wca_4k", 1000)
    n, n_sys = cfg.n_atoms, 3
    states = [make_state(cfg, 20 + b, jitter_amp=0.05) for b in range(n_sys)]
    box = states[0][3]
    vel = [s[1] * (2.0 if b == hot else 0.0) for b, s in enumerate(states)]
    kw, fv = {}, variant
    if variant == "full-globalw":
        fv, kw = "full", dict(flags=md.FLAG_GLOBAL_W)
    elif variant == "full-tiledw":
        fv, kw = "full", dict(flags=md.FLAG_TILED_W)
    g = md.MDSystem(n, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", force_variant=fv, step_mode=mode,
                    n_systems=n_sys, **kw)
    g.set_state(np.concatenate([s[0] for s in states]), np.concatenate(vel))
    o = OracleMD(n, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(states[hot][0], vel[hot])
    steps = 60
    g.step(steps)
    assert o.step(steps) == 0
    eg, eo = g.energies(), o.energies()
    assert eo.n_rebuilds >= 5 and eg.n_rebuilds == eo.n_rebuilds
    pos, fg = g.positions(), g.forces()
    assert pos_err(pos[hot * n:(hot + 1) * n], o.positions(), box) <= 1e-7      # 60 steps: chaos-limited, not 1e-9
    for b in range(n_sys):
        fb, _, _ = brute_forces_sample(pos[b * n:(b + 1) * n], box, cfg.r_cut, np.arange(n))
        assert force_rel_err(fg[b * n:(b + 1) * n], fb) <= FORCE_RTOL
    g.close()
