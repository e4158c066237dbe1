"""Seeded initial-state generators (numpy only; no MD arithmetic).

Random numbers come from a counter-based generator so that any consumer can
re-create the value for (seed, counter) without sequential state:

    h(seed, ctr) = splitmix64_finalise(seed * 0xD1342543DE82EF95
                                       + (ctr + 1) * 0x9E3779B97F4A7C15)   (mod 2^64)
    u(seed, ctr) = ((h >> 11) + 0.5) * 2^-53                               in (0, 1)

Gaussian velocity component k of atom `i` uses counters 2*(3*i + k) and
2*(3*i + k) + 1 through Box-Muller.  The library's own `md_create`
initialiser implements the same recipe in C++; tests compare the two.
"""
from __future__ import annotations

import math

import numpy as np

from .configs import MDConfig

_GOLD = np.uint64(0x9E3779B97F4A7C15)
_SEEDMUL = np.uint64(0xD1342543DE82EF95)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64(seed: int, ctr) -> np.ndarray:
    """h(seed, ctr) for an array of counters (uint64, wrapping arithmetic)."""
    ctr = np.asarray(ctr, dtype=np.uint64)
    s = np.uint64(seed & 0xFFFFFFFFFFFFFFFF)
    with np.errstate(over="ignore"):
        z = s * _SEEDMUL + (ctr + np.uint64(1)) * _GOLD
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, ctr) -> np.ndarray:
    """u(seed, ctr) in the open interval (0, 1), 53 random bits."""
    h = splitmix64(seed, ctr)
    return ((h >> np.uint64(11)).astype(np.float64) + 0.5) * (2.0 ** -53)


def box_edge(n_atoms: int, density: float) -> float:
    return (n_atoms / density) ** (1.0 / 3.0)


def _icbrt(n: int) -> int:
    c = round(n ** (1.0 / 3.0))
    for k in (c - 1, c, c + 1):
        if k > 0 and k * k * k == n:
            return k
    return 0


def sc_lattice(n_atoms: int, box: float) -> np.ndarray:
    """Simple-cubic grid, site (ix,iy,iz) at ((ix+1/2)a, ...), id = ix + Ne*(iy + Ne*iz)."""
    ne = _icbrt(n_atoms)
    if not ne:
        raise ValueError("sc_lattice needs a perfect cube")
    a = box / ne
    idx = np.arange(n_atoms, dtype=np.int64)
    ix, iy, iz = idx % ne, (idx // ne) % ne, idx // (ne * ne)
    r = np.empty((n_atoms, 3), dtype=np.float64)
    r[:, 0] = (ix + 0.5) * a
    r[:, 1] = (iy + 0.5) * a
    r[:, 2] = (iz + 0.5) * a
    return r


_FCC_BASIS = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]])


def fcc_lattice(n_atoms: int, box: float) -> np.ndarray:
    """FCC, n^3 cells x 4-atom basis shifted by (1/4,1/4,1/4), id = 4*cell + b."""
    if n_atoms % 4 or not _icbrt(n_atoms // 4):
        raise ValueError("fcc_lattice needs N = 4 n^3")
    n = _icbrt(n_atoms // 4)
    a = box / n
    idx = np.arange(n_atoms, dtype=np.int64)
    b, cell = idx % 4, idx // 4
    cx, cy, cz = cell % n, (cell // n) % n, cell // (n * n)
    r = np.empty((n_atoms, 3), dtype=np.float64)
    r[:, 0] = (cx + _FCC_BASIS[b, 0] + 0.25) * a
    r[:, 1] = (cy + _FCC_BASIS[b, 1] + 0.25) * a
    r[:, 2] = (cz + _FCC_BASIS[b, 2] + 0.25) * a
    return r


def gaussian_velocities(n_atoms: int, temperature: float, seed: int) -> np.ndarray:
    """N(0,T) components (Box-Muller on the counter generator), mean removed,
    then rescaled so that sum v^2 = 3 (N-1) T exactly (to rounding)."""
    c = 2 * np.arange(3 * n_atoms, dtype=np.uint64)
    u1 = uniform01(seed, c)
    u2 = uniform01(seed, c + np.uint64(1))
    g = np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * math.pi * u2)
    v = g.reshape(n_atoms, 3) * math.sqrt(temperature)
    v -= v.mean(axis=0)
    s2 = float(np.sum(v * v))
    if s2 > 0.0 and n_atoms > 1:
        v *= math.sqrt(3.0 * (n_atoms - 1) * temperature / s2)
    return v


def wrap(r: np.ndarray, box: float) -> np.ndarray:
    r = np.mod(r, box)
    r[r >= box] = 0.0
    return r


def jitter(r: np.ndarray, amplitude: float, seed: int, box: float) -> np.ndarray:
    """Uniform displacement in [-amplitude, amplitude]^3 per atom (separate counter range)."""
    n = r.shape[0]
    c = np.arange(3 * n, dtype=np.uint64) + np.uint64(1 << 40)
    d = (2.0 * uniform01(seed, c) - 1.0).reshape(n, 3) * amplitude
    return wrap(r + d, box)


def _row_grid(n_rows: int) -> tuple[int, int]:
    """ny x nz = n_rows with nz as close to 2*ny as possible, nz even (staggered rows)."""
    best = None
    for ny in range(1, int(math.isqrt(n_rows)) + 2):
        if n_rows % ny:
            continue
        nz = n_rows // ny
        for a, b in ((ny, nz), (nz, ny)):
            if b % 2:
                continue
            score = abs(math.log(b / (2.0 * a)))
            if best is None or score < best[0]:
                best = (score, a, b)
    if best is None:
        raise ValueError("cannot arrange rows on a staggered grid")
    return best[1], best[2]


def chain_melt(n_chains: int, chain_len: int, density: float, seed: int,
               bond: float = 0.97, jitter_amp: float = 0.02):
    """Overlap-free bead-spring start: planar zig-zag chains laid along x.

    Rows of `nx` beads run along x with projected spacing px = L/nx < bond; the
    zig-zag (+-t/2 in y on alternate beads, t = sqrt(bond^2 - px^2)) restores the
    bond length.  Rows sit on a staggered (centred-rectangular) grid in (y, z).
    Each row is cut into nx/chain_len chains starting at a seeded integer
    offset; a seeded jitter breaks the symmetry.  Returns (r, bonds, box) with
    atom id = chain * chain_len + bead and bonds (n_bonds, 2) int32.

    This stands in for "chains grown as seeded random walks then pushed apart"
    (BASELINE.json configs[4]): a push-off needs force evaluations, which this
    module must not contain (reading R12).
    """
    n = n_chains * chain_len
    box = box_edge(n, density)
    target_px = 0.84
    cands = [k * chain_len for k in range(1, n // chain_len + 1)
             if n % (k * chain_len) == 0 and (k * chain_len) % 2 == 0 and box / (k * chain_len) <= 0.9 * bond
             and 2.0 * box / (k * chain_len) >= 1.0]       # next-nearest beads of a chain stay >= 1 apart
    if not cands:
        raise ValueError("cannot lay chains of this length in rows of this box")
    nx = min(cands, key=lambda c: abs(box / c - target_px))
    px = box / nx
    ny, nz = _row_grid(n // nx)
    dy, dz = box / ny, box / nz
    t = math.sqrt(bond * bond - px * px)
    per_row = nx // chain_len

    row = np.arange(n // nx, dtype=np.int64)
    j, k = row % ny, row // ny
    y0 = (j + 0.5 * (k % 2) + 0.25) * dy
    z0 = (k + 0.5) * dz
    off = (splitmix64(seed, row.astype(np.uint64) + np.uint64(1 << 41)) % np.uint64(nx)).astype(np.int64)

    ids = np.arange(n, dtype=np.int64)
    chain, bead = ids // chain_len, ids % chain_len
    crow, cin = chain // per_row, chain % per_row
    site = (off[crow] + cin * chain_len + bead) % nx
    r = np.empty((n, 3), dtype=np.float64)
    r[:, 0] = (site + 0.5) * px
    r[:, 1] = y0[crow] + np.where(site % 2 == 0, 0.5 * t, -0.5 * t)
    r[:, 2] = z0[crow]
    r = wrap(r, box)
    if jitter_amp > 0.0:
        r = jitter(r, jitter_amp, seed, box)

    first = ids[bead < chain_len - 1]
    bonds = np.stack([first, first + 1], axis=1).astype(np.int32)
    return r, bonds, box


def make_state(cfg: MDConfig, seed: int = 1, jitter_amp: float = 0.0):
    """(r, v, bonds, box) for a config.  `jitter_amp` > 0 displaces the lattice
    sites (a cheap non-trivial state for force/neighbor parity at full size)."""
    box = cfg.box
    bonds = None
    if cfg.lattice == "sc":
        r = sc_lattice(cfg.n_atoms, box)
    elif cfg.lattice == "fcc":
        r = fcc_lattice(cfg.n_atoms, box)
    elif cfg.lattice == "chains":
        r, bonds, box = chain_melt(cfg.n_chains, cfg.chain_len, cfg.density, seed)
    else:
        raise ValueError(cfg.lattice)
    if jitter_amp > 0.0:
        r = jitter(r, jitter_amp, seed + 7919, box)
    v = gaussian_velocities(cfg.n_atoms, cfg.temperature, seed)
    return r, v, bonds, box
