"""GPU parity of the single-precision variant (md_params.precision = MD_PREC_F32) against the
single-precision oracle (oracle/md_oracle_sp.c) on the same seeded inputs.

Tolerances ("single precision"; eps = 2^-24):
  neighbor sets   exact -- both sides take r2 < r_n^2 on the same binary32 bits (R18)
  forces          per-pair terms are the same binary32 arithmetic; the sum over a column of W runs in another order
                  than the oracle's CSR row: <= 64 eps x (4 x max|f|), the bound the oracle itself is pinned with
  positions       10 steps: a coordinate moves by 1 ulp(L) when a rounding falls the other way (different summation
                  order, coordinates wrapped at rebuilds instead of every step): <= 16 ulp(L)
  velocities      after 10 steps the coordinates of the two sides differ by ulps of L (above); the pair force is stiff,
                  |df/dr| <= K = 624 r^-14 - 168 r^-8 ~ 2400 at the closest approach r ~ 0.9 (3000 used), so a velocity
                  may differ by steps x dt x K x ulp(L)
  energies        binary64 sums of the same binary32 terms: 64 eps relative to max(|PE|, KE)
"""
import numpy as np
import pytest

from md_workloads import get_config, make_state, scaled_config
from oracle.md_oracle import OracleMD, OracleMDSP
from parity_util import pos_err, sets_equal

pytestmark = pytest.mark.gpu
EPS32 = 2.0 ** -24
F_TOL = 64 * EPS32 * 4


@pytest.fixture(scope="module")
def md():
    import paper_2003_14061_b200 as m
    m.load_library()
    return m


def cases():
    return {
        "wca_4k": get_config("wca_4k"),
        "wca_ragged_1000": scaled_config("wca_4k", 1000),
        "wca_dr03_13824": scaled_config("wca_2m_dr03", 24 ** 3),
        "wca_dr05_13824": scaled_config("wca_2m_dr05", 24 ** 3),
        "lj_6912": scaled_config("lj_1m", 4 * 12 ** 3),
        "chains_4096": scaled_config("chains_rows_1m", 4096, chain_len=16),
    }


def make_pair(md, cfg, seed, mode="fused", state="jitter", flags=0, **kw):
    jit = 0.0 if state == "lattice" else (0.12 if cfg.lattice != "chains" else 0.0)
    r, v, bonds, box = make_state(cfg, seed, jitter_amp=jit)
    o = OracleMDSP(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(r, v)
    if bonds is not None:
        assert o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0) == 0
    if state == "thermal":
        assert o.step(200) == 0
        r, v = o.positions(), o.velocities()
        o.set_state(r, v)
        if bonds is not None:
            o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", step_mode=mode,
                    precision="f32", flags=flags, **kw)
    g.set_state(r, v)
    if bonds is not None:
        g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    return g, o, box


@pytest.mark.parametrize("case", list(cases()))
@pytest.mark.parametrize("state", ["lattice", "jitter", "thermal"])
@pytest.mark.parametrize("build_flags", [0, 2])          # tile-staged build (default) / gather build (MD_FLAG_GLOBAL_W)
def test_sp_neighbor_sets_and_forces(md, case, state, build_flags):
    cfg = cases()[case]
    if state == "lattice" and cfg.lattice == "chains":
        pytest.skip("chain start has no separate lattice state")
    for seed in (1, 2, 3) if state != "thermal" else (1,):
        g, o, box = make_pair(md, cfg, seed, mode="split", state=state, flags=build_flags)
        assert g.info()["precision"] == 1 and (g.info()["tile_capacity"] > 0) == (build_flags == 0)
        counts, lst = g.neighbors()
        nbad, first = sets_equal(counts, lst, o)
        assert nbad == 0, f"neighbor sets differ for {nbad} atoms (first: atom {first})"
        fo, fg = o.forces(), g.forces()
        if state == "lattice" and cfg.lattice in ("sc", "fcc"):
            # f_i = 0 analytically; in binary32 the lattice coordinates are rounded, so only an absolute bound holds:
            # 78 pair forces of magnitude < 24 (r_c = 2.5: < 2.4 beyond the first shell), each with a relative error of
            # a few ulp(L)/r from the rounded coordinates
            scale = 24.0 * 78
            ulp_rel = float(np.spacing(np.float32(box))) * 16
            assert np.abs(fg - fo).max() <= scale * ulp_rel
        else:
            assert np.abs(fg - fo).max() <= F_TOL * np.abs(fo).max()
        eg, eo = g.energies(), o.energies()
        escale = max(abs(eo.pe_pair), eo.ke, 1.0)
        assert abs(eg.pe_pair - eo.pe_pair) <= 64 * EPS32 * escale
        assert abs(eg.pe_bond - eo.pe_bond) <= 64 * EPS32 * max(abs(eo.pe_bond), 1.0)
        assert abs(eg.virial - eo.virial) <= 64 * EPS32 * max(abs(eo.virial), escale)
        assert eg.ke == pytest.approx(eo.ke, rel=1e-12)            # binary64 sums of the same binary32 velocities
        assert eg.max_neighbors == eo.max_neighbors
        assert eg.mean_neighbors == pytest.approx(eo.mean_neighbors, rel=1e-12)
        g.close()


@pytest.mark.parametrize("case", list(cases()))
@pytest.mark.parametrize("mode,flags", [("fused", 0), ("split", 0), ("fused", 1), ("fused", 16), ("fused", 2), ("fused", 2 | 16)])
def test_sp_ten_steps(md, case, mode, flags):
    cfg = cases()[case]
    for seed in (1, 2, 3):
        g, o, box = make_pair(md, cfg, seed, mode=mode, flags=flags)
        g.step(10)
        assert o.step(10) == 0
        ulp_L = float(np.spacing(np.float32(box)))
        assert pos_err(g.positions(), o.positions(), float(np.float32(box))) <= 16 * ulp_L
        vo = o.velocities()
        assert np.abs(g.velocities() - vo).max() <= 10 * cfg.dt * 3000.0 * ulp_L + 64 * EPS32 * np.abs(vo).max()
        eg, eo = g.energies(), o.energies()
        escale = max(abs(eo.pe), eo.ke)
        assert abs(eg.ke - eo.ke) <= 64 * EPS32 * escale
        assert abs(eg.pe - eo.pe) <= 64 * EPS32 * escale * 4      # positions differ by ulps: stiff r^-12 terms amplify
        assert eg.step == eo.step == 10 and eg.n_rebuilds == eo.n_rebuilds
        g.close()


def test_sp_tracks_fp64_oracle(md):
    """Accuracy of the variant itself (not parity): from the same state the binary32 GPU path stays within the bound
    the binary32 oracle is pinned with against the fp64 oracle (test_oracle_sp_pins.py sp4)."""
    cfg = get_config("wca_4k")
    r, v, _, box = make_state(cfg, 1, jitter_amp=0.1)
    r32, v32 = np.asarray(r, np.float32).astype(np.float64), np.asarray(v, np.float32).astype(np.float64)
    box32 = float(np.float32(box))
    o = OracleMD(cfg.n_atoms, box32, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(np.mod(r32, box32), v32)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", precision="f32")
    g.set_state(r, v)
    g.step(10)
    o.step(10)
    assert pos_err(g.positions(), o.positions(), box32) <= 16 * float(np.spacing(np.float32(box)))
    eg, eo = g.energies(), o.energies()
    assert abs(eg.total - eo.total) <= 64 * EPS32 * eo.ke * 10
    g.close()


def test_sp_long_run_conserves_energy_like_fp64(md):
    """1000 steps (config 1's length): total energy per atom of the binary32 run stays within 5e-4 of the fp64 GPU run
    from the same start; the rebuild statistics agree."""
    cfg = get_config("wca_4k")
    r, v, _, box = make_state(cfg, 1, jitter_amp=0.1)
    out = []
    for prec in ("f64", "f32"):
        g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", precision=prec)
        g.set_state(r, v)
        g.step(1000)
        out.append(g.energies())
        g.close()
    e64, e32 = out
    # the runs decorrelate (chaos) and each total fluctuates by ~1e-3 per atom (dt^2 truncation): compare at that scale
    assert abs(e64.total - e32.total) / cfg.n_atoms < 5e-4
    assert abs(e64.n_rebuilds - e32.n_rebuilds) <= 3
    assert max(abs(e32.px), abs(e32.py), abs(e32.pz)) < 1e-2


def test_sp_batched_systems(md):
    """n_systems mutually invisible systems in binary32: each equals its own oracle."""
    cfg = scaled_config("wca_4k", 1000)
    B = 3
    states = [make_state(cfg, 10 + b, jitter_amp=0.12) for b in range(B)]
    box = states[0][3]
    r = np.concatenate([s[0] for s in states])
    v = np.concatenate([s[1] for s in states])
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", precision="f32", n_systems=B)
    g.set_state(r, v)
    g.step(10)
    pg, fg = g.positions(), g.forces()
    for b in range(B):
        o = OracleMDSP(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
        o.set_state(states[b][0], states[b][1])
        o.step(10)
        sl = slice(b * cfg.n_atoms, (b + 1) * cfg.n_atoms)
        assert pos_err(pg[sl], o.positions(), float(np.float32(box))) <= 16 * float(np.spacing(np.float32(box)))
        fo = o.forces()
        assert np.abs(fg[sl] - fo).max() <= 1e-3 * np.abs(fo).max()     # after 10 steps positions differ by ulps
    g.close()


def test_sp_rejects_unsupported_combinations(md):
    cfg = get_config("wca_4k")
    with pytest.raises(md.MDError):
        md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, density=cfg.density, precision="f32", force_variant="newton3")
    with pytest.raises(md.MDError):
        md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, density=cfg.density, precision="f32", flags=md.FLAG_TILED_W)


def test_sp_full_size_sampled(md):
    """wca_2m in the launch configuration bench.py times (fused steps, graph): after 20 steps from the lattice start,
    neighbor sets of sampled atoms equal the binary32 definition evaluated by numpy on the GPU's own coordinates, and
    their forces equal the fp64 textbook sum at those coordinates within the binary32 bound."""
    cfg = get_config("wca_2m")
    g = md.MDSystem.from_config(cfg, seed=1, precision="f32")
    g.step(20)
    g.rebuild_neighbors()
    r = g.positions()
    f = g.forces()
    counts, lst = g.neighbors()
    box32 = np.float32(g.info()["box"])
    rng = np.random.default_rng(7)
    idx = rng.integers(0, cfg.n_atoms, 256)
    rf = np.asarray(r, np.float32)
    rn = cfg.r_cut + cfg.r_shell
    rn2, rc2 = np.float32(rn * rn), cfg.r_cut ** 2
    half = np.float32(0.5) * box32
    for i in idx:
        d = rf[i][None, :] - rf                                   # binary32
        d = np.where(d > half, d - box32, np.where(d < -half, d + box32, d)).astype(np.float32)
        dd = d.astype(np.float64)
        t0 = (dd[:, 0] * dd[:, 0]).astype(np.float32).astype(np.float64)
        t1 = (dd[:, 1] * dd[:, 1] + t0).astype(np.float32).astype(np.float64)
        r2 = (dd[:, 2] * dd[:, 2] + t1).astype(np.float32)
        acc = r2 < rn2
        acc[i] = False
        assert np.array_equal(np.sort(lst[i, :counts[i]]), np.nonzero(acc)[0])
        r2d = (dd * dd).sum(1)
        inside = (r2d < rc2) & acc
        s3 = r2d[inside] ** -3
        fc = 48.0 * s3 * (s3 - 0.5) / r2d[inside]
        fref = (fc[:, None] * dd[inside]).sum(0)
        assert np.abs(f[i] - fref).max() <= F_TOL * max(np.abs(fc[:, None] * dd[inside]).sum(), 1.0)
    g.close()
