"""Input generators: geometry and statistics of the seeded synthetic workloads (no MD arithmetic)."""
import math

import numpy as np
import pytest
from scipy.spatial import cKDTree

from md_workloads import (CONFIGS, chain_melt, chain_walks, fcc_lattice, gaussian_velocities, make_state, sc_lattice,
                          scaled_config, splitmix64, uniform01)


def test_counter_generator_reference_values():
    # SplitMix64 finaliser (Steele, Lea, Flood 2014) applied to seed*0xD134..95 + (ctr+1)*0x9E37..15, by hand in Python ints
    def ref(seed, ctr):
        m = (1 << 64) - 1
        z = (seed * 0xD1342543DE82EF95 + (ctr + 1) * 0x9E3779B97F4A7C15) & m
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & m
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & m
        return z ^ (z >> 31)
    ctr = np.array([0, 1, 2, 12345, 2 ** 40 + 5], dtype=np.uint64)
    for seed in (0, 1, 987654321):
        got = splitmix64(seed, ctr)
        assert [int(x) for x in got] == [ref(seed, int(c)) for c in ctr]
    u = uniform01(7, np.arange(200000))
    assert 0.0 < u.min() and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 3e-3 and abs(u.var() - 1 / 12) < 2e-3


def test_velocities_temperature_and_momentum():
    n, T = 4096, 0.72
    v = gaussian_velocities(n, T, 5)
    assert np.abs(v.sum(0)).max() < 1e-10
    assert (v * v).sum() == pytest.approx(3 * (n - 1) * T, rel=1e-13)
    assert abs(np.mean(v ** 4) / np.mean(v ** 2) ** 2 - 3.0) < 0.15      # Gaussian kurtosis
    assert not np.allclose(v, gaussian_velocities(n, T, 6))


def test_lattices():
    box = (4096 / 0.8) ** (1 / 3)
    r = sc_lattice(4096, box)
    assert r.min() > 0 and r.max() < box
    d, _ = cKDTree(r, boxsize=box).query(r, k=2)
    assert np.allclose(d[:, 1], box / 16)
    n = 4 * 6 ** 3
    box = (n / 0.8442) ** (1 / 3)
    r = fcc_lattice(n, box)
    d, _ = cKDTree(r, boxsize=box).query(r, k=13)
    assert np.allclose(d[:, 1:], (box / 6) / math.sqrt(2))               # 12 nearest neighbours


@pytest.mark.parametrize("n_chains,chain_len", [(256, 16), (512, 32), (1024, 64)])
def test_chain_start_is_overlap_free(n_chains, chain_len):
    r, bonds, box = chain_melt(n_chains, chain_len, 0.85, seed=3)
    n = n_chains * chain_len
    assert r.shape == (n, 3) and bonds.shape == (n_chains * (chain_len - 1), 2)
    assert r.min() >= 0 and r.max() < box
    d = r[bonds[:, 0]] - r[bonds[:, 1]]
    d -= box * np.round(d / box)
    bl = np.sqrt((d * d).sum(1))
    assert 0.85 < bl.min() and bl.max() < 1.1                            # FENE R0 = 1.5
    assert np.all(bonds[:, 0] // chain_len == bonds[:, 1] // chain_len)
    pairs = cKDTree(r, boxsize=box).query_pairs(0.9, output_type="ndarray")
    bonded = set(map(tuple, np.sort(bonds, 1)))
    nonbonded = [p for p in map(tuple, np.sort(pairs, 1)) if p not in bonded]
    assert not nonbonded                                                  # min non-bonded distance >= 0.9


def test_make_state_matches_configs():
    for name, cfg in CONFIGS.items():
        assert cfg.box == pytest.approx((cfg.n_atoms / cfg.density) ** (1 / 3))
    cfg = scaled_config("chains_rows_1m", 4096, chain_len=16)
    r, v, bonds, box = make_state(cfg, 1)
    assert r.shape == v.shape == (4096, 3) and bonds is not None
    cfg = scaled_config("wca_2m", 512)
    r, v, bonds, box = make_state(cfg, 1, jitter_amp=0.1)
    assert bonds is None and np.abs(r - sc_lattice(512, box)).max() > 0.01


@pytest.mark.parametrize("n_chains,chain_len", [(256, 16), (300, 10), (2048, 64)])
def test_chain_walks_geometry(n_chains, chain_len):
    """BASELINE.json configs[4] "chains grown as seeded random walks": every bond 0.97 long, next-
    nearest beads of a chain at least 1.02 apart, starts uniform in the box, directions isotropic, reproducible from
    (seed, chain, bead) counters.  The walks ignore one another, so the start overlaps (that is what md_pushoff is for)."""
    r, bonds, box = chain_walks(n_chains, chain_len, 0.85, seed=3)
    n = n_chains * chain_len
    assert box == pytest.approx((n / 0.85) ** (1 / 3))
    assert r.shape == (n, 3) and bonds.shape == (n_chains * (chain_len - 1), 2)
    assert r.min() >= 0 and r.max() < box
    assert np.all(bonds[:, 1] == bonds[:, 0] + 1) and np.all(bonds[:, 0] // chain_len == bonds[:, 1] // chain_len)
    R = r.reshape(n_chains, chain_len, 3)
    b = R[:, 1:] - R[:, :-1]
    b -= box * np.round(b / box)
    assert np.abs(np.sqrt((b * b).sum(-1)) - 0.97).max() < 1e-12
    d2 = R[:, 2:] - R[:, :-2]
    d2 -= box * np.round(d2 / box)
    assert np.sqrt((d2 * d2).sum(-1)).min() >= 1.02 - 1e-12
    # first steps are unconstrained: isotropic; starts uniform
    u = b[:, 0] / 0.97
    assert np.abs(u.mean(0)).max() < 4.0 / math.sqrt(3 * n_chains)
    assert np.abs(R[:, 0].mean(0) / box - 0.5).max() < 4.0 / math.sqrt(12 * n_chains)
    # consecutive bonds: the 1.02 rule removes the sharpest back-folds, cos(angle between bonds) >= 1.02^2/(2 0.97^2) - 1
    cosb = (b[:, 1:] * b[:, :-1]).sum(-1) / 0.97 ** 2
    assert cosb.min() >= 1.02 ** 2 / (2 * 0.97 ** 2) - 1.0 - 1e-12 and cosb.max() > 0.9
    # reproducible, seed-dependent, and chain c does not depend on how many chains there are
    assert np.array_equal(r, chain_walks(n_chains, chain_len, 0.85, seed=3)[0])
    assert not np.array_equal(r, chain_walks(n_chains, chain_len, 0.85, seed=4)[0])
    # it does overlap
    close = cKDTree(r, boxsize=box).query_pairs(0.5, output_type="ndarray")
    assert len(close) > 0


def test_walk_config_is_configs4():
    cfg = CONFIGS["chains_1m"]
    assert (cfg.lattice, cfg.n_chains, cfg.chain_len, cfg.n_atoms) == ("walk", 16384, 64, 1048576)
    assert (cfg.density, cfg.temperature, cfg.dt, cfg.fene_k, cfg.fene_r0) == (0.85, 1.0, 0.005, 30.0, 1.5)
    small = scaled_config("chains_1m", 4096, chain_len=16)
    r, v, bonds, box = make_state(small, 2)
    assert r.shape == (4096, 3) and bonds.shape == (256 * 15, 2) and small.lattice == "walk"
