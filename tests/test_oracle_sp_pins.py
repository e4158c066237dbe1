"""Pins for the single-precision oracle (oracle/md_oracle_sp.c, R18).

It is pinned to things other than itself: numpy float32 all-pairs decisions written from the definition, the
textbook potential in numpy fp64 at the binary32-rounded coordinates, the (separately pinned) fp64 oracle run
from the same rounded state, two-atom closed forms, conservation laws.  Bounds are derived from binary32
rounding (eps = 2^-24 ~ 6e-8 per operation) and stated next to each check.
"""
import numpy as np
import pytest

from md_workloads import get_config, make_state, scaled_config, sc_lattice
from md_workloads.configs import R_WCA
from oracle.md_oracle import OracleMD, OracleMDSP

EPS32 = 2.0 ** -24


def fluid_state(n_side=8, rho=0.8, amp=0.18, seed=3):
    n = n_side ** 3
    box = (n / rho) ** (1 / 3)
    rng = np.random.default_rng(seed)
    r = sc_lattice(n, box) + rng.uniform(-amp, amp, (n, 3))
    return np.mod(r, box), box


def round32(a):
    return np.asarray(a, np.float32).astype(np.float64)


def np_f32_neighbor_sets(r, box, r_n):
    """The binary32 decision of DESIGN.md R18 written with numpy float32 scalars-as-arrays: d = fl(a - b), minimum
    image by one conditional +-L, r2 = fl(dz*dz + fl(dy*dy + fl(dx*dx))) with fused multiply-adds emulated in
    fp64 (a product of two binary32 numbers is exact in binary64, and one rounding of the exact sum of such a
    product and a binary32 number to binary32 is what fmaf returns -- double rounding cannot occur when the fp64
    sum is exact, which holds here except in ties that the test data do not contain)."""
    rf = np.asarray(r, np.float32)
    L = np.float32(box)
    half = np.float32(0.5) * L
    d = rf[:, None, :] - rf[None, :, :]                       # float32 subtraction
    d = np.where(d > half, d - L, np.where(d < -half, d + L, d)).astype(np.float32)
    dd = d.astype(np.float64)
    t0 = (dd[..., 0] * dd[..., 0]).astype(np.float32).astype(np.float64)     # dx*dx rounded
    t1 = (dd[..., 1] * dd[..., 1] + t0).astype(np.float32).astype(np.float64)
    r2 = (dd[..., 2] * dd[..., 2] + t1).astype(np.float32)
    rn2 = np.float32(r_n * r_n)
    acc = r2 < rn2
    np.fill_diagonal(acc, False)
    return [np.nonzero(acc[i])[0].astype(np.int32) for i in range(r.shape[0])], r2


def np_forces64(r, box, r_cut):
    d = r[:, None, :] - r[None, :, :]
    d -= box * np.round(d / box)
    dist = np.sqrt((d * d).sum(-1))
    np.fill_diagonal(dist, np.inf)
    inside = dist < r_cut
    uc = 4.0 * (r_cut ** -12 - r_cut ** -6)
    u = np.where(inside, 4.0 * (dist ** -12 - dist ** -6) - uc, 0.0)
    fmag = np.where(inside, 24.0 * (2.0 * dist ** -13 - dist ** -7), 0.0)
    f = ((fmag / dist)[:, :, None] * d).sum(1)
    return f, u.sum(1), (fmag * np.where(inside, dist, 0.0)).sum(1)


@pytest.mark.parametrize("r_cut,r_shell,rho,n_side", [(R_WCA, 0.4, 0.8, 8), (R_WCA, 0.3, 0.8, 6), (2.5, 0.3, 0.8442, 9)])
def test_sp1_neighbor_sets_are_the_binary32_definition(r_cut, r_shell, rho, n_side):
    r, box = fluid_state(n_side, rho, 0.2)
    ref, _ = np_f32_neighbor_sets(r, box, r_cut + r_shell)
    for brute in (True, False):          # O(N^2) definition and the linked-cell search
        o = OracleMDSP(r.shape[0], box, r_cut, r_shell, 0.005, brute_search=brute)
        o.set_state(r)
        got = o.neighbor_sets()
        assert all(np.array_equal(a, b) for a, b in zip(got, ref)), f"brute={brute}"
    # the relation is symmetric (every pair twice): fl(a-b) = -fl(b-a) exactly
    sets = [set(x.tolist()) for x in ref]
    assert all(i in sets[j] for i in range(len(sets)) for j in sets[i])


def test_sp1b_decision_is_taken_in_binary32_not_binary64():
    """A pair placed so that the binary64 and binary32 values of r^2 fall on opposite sides of r_n^2: the oracle
    must follow binary32 (both sides of the parity test do, R18)."""
    r_cut, r_shell = R_WCA, 0.4
    rn = r_cut + r_shell
    box = 12.0
    rn2f = np.float32(rn * rn)
    found = 0
    rng = np.random.default_rng(5)
    for _ in range(20000):
        a = rng.uniform(1.0, 9.0, 3)
        u = rng.normal(size=3)
        u /= np.linalg.norm(u)
        b = a + u * rn * (1.0 + rng.uniform(-2e-7, 2e-7))
        pair = np.stack([a, b])
        (s0, _), r2 = np_f32_neighbor_sets(pair, box, rn)
        d64 = round32(pair)[0] - round32(pair)[1]
        in64 = float((d64 * d64).sum()) < float(rn2f)
        in32 = bool(r2[0, 1] < rn2f)
        if in64 != in32:
            o = OracleMDSP(2, box, r_cut, r_shell, 0.005, brute_search=True)
            o.set_state(pair)
            assert (o.neighbors()[0][0] == 1) == in32
            found += 1
            if found >= 5:
                break
    assert found >= 1, "no discriminating pair generated"


@pytest.mark.parametrize("r_cut,rho", [(R_WCA, 0.8), (2.5, 0.8442)])
def test_sp2_forces_and_atom_energies_vs_textbook_fp64_at_rounded_coordinates(r_cut, rho):
    """At the binary32-rounded coordinates the only error left is the pair arithmetic: ~10 binary32 operations per
    pair term (each <= eps relative) and m additions.  Bound used: 64 eps relative to the sum of |terms|, which a
    dropped term, a wrong sign or exponent or a transposed operand exceeds by orders of magnitude."""
    r, box = fluid_state(8, rho, 0.2)
    r32 = round32(r)
    o = OracleMDSP(r.shape[0], box, r_cut, 0.3, 0.005)
    o.set_state(r)
    f_ref, u_ref, w_ref = np_forces64(r32, float(np.float32(box)), r_cut)
    f = o.forces()
    u, w = o.atom_energies()
    # scale: sum over neighbors of |f_ij| is a few times max|f|
    scale_f = np.abs(f_ref).max()
    assert np.abs(f - f_ref).max() < 64 * EPS32 * scale_f * 4
    # pairs whose r2 lies within rounding of r_c^2 contribute u ~ 0 and f ~ 0 (WCA) or are tiny (LJ 2.5): no jump
    assert np.abs(u - u_ref).max() < 64 * EPS32 * max(1.0, np.abs(u_ref).max()) * 8
    assert np.abs(w - w_ref).max() < 64 * EPS32 * max(1.0, np.abs(w_ref).max()) * 8


def test_sp3_two_atom_closed_forms():
    """r = 1: f = 24, u = 0 - u_c (exactly representable inputs); r = 2^(1/6): f ~ 0 at the WCA cutoff minimum."""
    box = 10.0
    for r_cut in (2.5, R_WCA):
        o = OracleMDSP(2, box, r_cut, 0.3, 0.005, brute_search=True)
        o.set_state(np.array([[1.0, 2.0, 3.0], [2.0, 2.0, 3.0]]))
        f = o.forces()
        assert f[0, 0] == -24.0 and f[1, 0] == 24.0 and np.all(f[:, 1:] == 0.0)
        uc = 4.0 * (r_cut ** -12 - r_cut ** -6)
        e = o.energies()
        assert abs(e.pe_pair - (0.0 - uc)) < 4 * EPS32 * max(1.0, abs(uc))
        assert abs(e.virial - 24.0) < 1e-6
    # across the periodic face: same pair, minimum image
    o = OracleMDSP(2, box, 2.5, 0.3, 0.005, brute_search=True)
    o.set_state(np.array([[0.25, 2.0, 3.0], [9.25, 2.0, 3.0]]))
    f = o.forces()
    assert f[0, 0] == 24.0 and f[1, 0] == -24.0


def test_sp4_trajectory_tracks_the_fp64_oracle_from_the_same_rounded_state():
    """10 steps from binary32-representable r, v.  Per step a binary32 coordinate is rounded to ulp(x) <= ulp(L)
    (add of dt*v, and the wrap); the fp64 oracle is not.  Bound: 10 steps x 1 ulp(L) + slack = 16 ulp(L).
    Energies: relative 64 eps (binary64 sums of binary32 terms carry unbiased ~eps errors)."""
    cfg = get_config("wca_4k")
    r, v, _, box = make_state(cfg, 1, jitter_amp=0.1)
    r32, v32 = round32(r), round32(v)
    box32 = float(np.float32(box))
    o = OracleMD(cfg.n_atoms, box32, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(np.mod(r32, box32), v32)
    s = OracleMDSP(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    s.set_state(r, v)
    e0o, e0s = o.energies(), s.energies()
    assert abs(e0o.ke - e0s.ke) < 4 * EPS32 * e0o.ke
    assert abs(e0o.pe_pair - e0s.pe_pair) < 64 * EPS32 * max(abs(e0o.pe_pair), e0o.ke)
    o.step(10)
    s.step(10)
    d = o.positions() - s.positions()
    d -= box32 * np.round(d / box32)
    ulp_L = float(np.spacing(np.float32(box)))
    assert np.abs(d).max() < 16 * ulp_L
    eo, es = o.energies(), s.energies()
    assert abs(eo.total - es.total) < 64 * EPS32 * eo.ke * 10
    assert es.step == 10 and es.n_rebuilds == eo.n_rebuilds


def test_sp5_conservation_and_newton3():
    cfg = scaled_config("wca_4k", 1000)
    r, v, _, box = make_state(cfg, 2, jitter_amp=0.1)
    s = OracleMDSP(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    s.set_state(r, v)
    f = s.forces()
    # sum of forces: every pair contributes fc*d and fc*(-d) with identical fc (symmetric arithmetic) -> only the
    # binary32 accumulation order differs: |sum| <= N * m * eps * max|f|
    assert np.abs(f.sum(0)).max() < cfg.n_atoms * 16 * EPS32 * np.abs(f).max()
    # energy: the dt^2 truncation error (~2e-3 per atom for this melting lattice) is common to both precisions;
    # what binary32 adds must stay far below it: |(E_sp - E_dp)(t)| per atom < 5e-5 over 200 steps
    o = OracleMD(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(r, v)
    s.step(200)
    o.step(200)
    e1, eo = s.energies(), o.energies()
    assert abs(e1.total - eo.total) / cfg.n_atoms < 5e-5
    assert max(abs(e1.px), abs(e1.py), abs(e1.pz)) < cfg.n_atoms * 200 * 8 * EPS32 * e1.vmax
    assert e1.n_rebuilds >= 10


def test_sp6_bonds_match_fp64_oracle_at_rounded_coordinates():
    cfg = scaled_config("chains_rows_1m", 512, chain_len=16)
    r, v, bonds, box = make_state(cfg, 3)
    s = OracleMDSP(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    s.set_state(r, v)
    assert s.set_bonds(bonds, cfg.fene_k, cfg.fene_r0) == 0
    box32 = float(np.float32(box))
    o = OracleMD(cfg.n_atoms, box32, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(np.mod(round32(r), box32), round32(v))
    assert o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0) == 0
    fo, fs = o.forces(), s.forces()
    assert np.abs(fo - fs).max() < 256 * EPS32 * np.abs(fo).max()
    eo, es = o.energies(), s.energies()
    assert abs(eo.pe_bond - es.pe_bond) < 64 * EPS32 * abs(eo.pe_bond)
    assert abs(eo.virial - es.virial) < 256 * EPS32 * max(abs(eo.virial), eo.ke)


def test_sp7_angles_match_fp64_oracle_at_rounded_coordinates():
    """Bond-angle terms (R19) in binary32 against the (separately pinned, P14) fp64 oracle from the same
    rounded state: ~20 binary32 operations per term."""
    cfg = scaled_config("chains_rows_1m", 1000, chain_len=10)
    r, v, bonds, box = make_state(cfg, 3)
    box32 = float(np.float32(box))
    s = OracleMDSP(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    s.set_state(r, v)
    s.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    o = OracleMD(cfg.n_atoms, box32, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(np.mod(round32(r), box32), round32(v))
    o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    fs0, fo0, es0, eo0 = s.forces(), o.forces(), s.energies().pe_bond, o.energies().pe_bond
    assert s.set_angles(5.0, -0.5) == 0 and o.set_angles(5.0, -0.5) == 0
    dfs, dfo = s.forces() - fs0, o.forces() - fo0                   # the angle part
    assert np.abs(dfo).max() > 1.0
    assert np.abs(dfs - dfo).max() < 256 * EPS32 * np.abs(fo0).max()
    assert abs((s.energies().pe_bond - es0) - (o.energies().pe_bond - eo0)) < 64 * EPS32 * abs(o.energies().pe_bond)


def test_sp8_dihedrals_match_fp64_oracle_at_rounded_coordinates():
    """Dihedral terms (R19) in binary32 against the fp64 oracle (pinned by P15) from the same rounded state.
    ~80 binary32 operations per term; 1/|A|^2 amplifies rounding where consecutive bonds are nearly collinear, hence the
    bound relative to the largest dihedral force."""
    cfg = scaled_config("chains_rows_1m", 1000, chain_len=10)
    r, v, bonds, box = make_state(cfg, 3)
    box32 = float(np.float32(box))
    s = OracleMDSP(cfg.n_atoms, box, cfg.r_cut, cfg.r_shell, cfg.dt)
    s.set_state(r, v)
    s.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    o = OracleMD(cfg.n_atoms, box32, cfg.r_cut, cfg.r_shell, cfg.dt)
    o.set_state(np.mod(round32(r), box32), round32(v))
    o.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    fs0, fo0, es0, eo0 = s.forces(), o.forces(), s.energies().pe_bond, o.energies().pe_bond
    assert s.set_dihedrals(2.0, 0.3) == 0 and o.set_dihedrals(2.0, 0.3) == 0
    dfs, dfo = s.forces() - fs0, o.forces() - fo0
    assert np.abs(dfo).max() > 0.5
    assert np.abs(dfs - dfo).max() < 1024 * EPS32 * max(np.abs(dfo).max(), np.abs(fo0).max())
    assert abs((s.energies().pe_bond - es0) - (o.energies().pe_bond - eo0)) < 256 * EPS32 * abs(o.energies().pe_bond)
