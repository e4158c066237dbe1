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

    An extra, crystalline chain input (configs "chains_rows_*"): it needs no push-off, so the CPU-only tests and
    the small parity cases can use it.  BASELINE.json configs[4] itself is `chain_walks` + the library's push-off.
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


_WALK_BASE = 1 << 42          # counter range of the random walks (velocities use [0, 6N), jitter 2^40.., rows 2^41..)
_WALK_ATTEMPTS = 64


def _unit_vectors(seed: int, ctr) -> np.ndarray:
    """Uniform directions on the sphere from counters ctr, ctr + 1: z = 2u1 - 1, phi = 2 pi u2."""
    ctr = np.asarray(ctr, dtype=np.uint64)
    z = 2.0 * uniform01(seed, ctr) - 1.0
    phi = 2.0 * math.pi * uniform01(seed, ctr + np.uint64(1))
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def chain_walks(n_chains: int, chain_len: int, density: float, seed: int,
                bond: float = 0.97, min_second: float = 1.02):
    """Chains "grown as seeded random walks" (BASELINE.json configs[4]).

    Each chain starts at a seeded point uniform in the box and takes chain_len - 1 steps of length `bond` in uniformly
    random directions; a step is redrawn while it would bring bead k+1 closer than `min_second` to bead k-1.  Chains
    ignore one another, so the start OVERLAPS: it must be pushed apart before use (the library's md_pushoff --
    pure geometry here, no forces).  Returns (r wrapped into the box, bonds, box), atom id = chain * chain_len + bead.
    """
    n = n_chains * chain_len
    box = box_edge(n, density)
    chain = np.arange(n_chains, dtype=np.uint64)
    base = np.uint64(_WALK_BASE)
    per_chain = np.uint64(4 + 2 * _WALK_ATTEMPTS * chain_len)
    c0 = base + chain * per_chain
    pos = np.empty((n_chains, chain_len, 3), dtype=np.float64)
    for k in range(3):
        pos[:, 0, k] = uniform01(seed, c0 + np.uint64(k)) * box
    for b in range(1, chain_len):
        pending = np.arange(n_chains)
        for attempt in range(_WALK_ATTEMPTS):
            ctr = c0[pending] + np.uint64(4 + 2 * (_WALK_ATTEMPTS * b + attempt))
            cand = pos[pending, b - 1] + bond * _unit_vectors(seed, ctr)
            if b >= 2:
                d = cand - pos[pending, b - 2]
                ok = (d * d).sum(1) >= min_second * min_second
            else:
                ok = np.ones(len(pending), dtype=bool)
            pos[pending[ok], b] = cand[ok]
            pending = pending[~ok]
            if len(pending) == 0:
                break
        else:
            raise RuntimeError("chain_walks: a step was rejected %d times" % _WALK_ATTEMPTS)
    r = wrap(pos.reshape(n, 3), box)
    ids = np.arange(n, dtype=np.int64)
    first = ids[ids % chain_len < chain_len - 1]
    bonds = np.stack([first, first + 1], axis=1).astype(np.int32)
    return r, bonds, box


# ---- rigid molecules (R20): geometry and seeded random numbers only -----------------------
_ROT_BASE = 1 << 43


def tetrahedron_body(edge: float = 0.9) -> np.ndarray:
    """Four unit-mass sites at the corners of a regular tetrahedron ("four SP spheres in a rigid tetrahedral configuration,
    spaced to overlap slightly"), centre of mass at the origin; the inertia tensor is isotropic (2 edge^2)."""
    a = edge / (2.0 * math.sqrt(2.0))
    return a * np.array([[1.0, 1.0, 1.0], [1.0, -1.0, -1.0], [-1.0, 1.0, -1.0], [-1.0, -1.0, 1.0]])


def cross_body(a: float = 0.55, b: float = 0.4, c: float = 0.25) -> np.ndarray:
    """Six unit-mass sites at (+-a,0,0), (0,+-b,0), (0,0,+-c): an asymmetric top in its principal frame
    (moments 2(b^2+c^2), 2(a^2+c^2), 2(a^2+b^2))."""
    return np.array([[a, 0, 0], [-a, 0, 0], [0, b, 0], [0, -b, 0], [0, 0, c], [0, 0, -c]], dtype=np.float64)


def body_inertia(body: np.ndarray) -> np.ndarray:
    """Principal moments of unit-mass sites given in their principal frame."""
    b2 = (body * body).sum(1)
    return np.array([(b2 - body[:, k] ** 2).sum() for k in range(3)])


def random_rotations(n: int, seed: int) -> np.ndarray:
    """n rotation matrices, uniform on SO(3): unit quaternions from four Gaussians of the counter generator."""
    c = np.uint64(_ROT_BASE) + 2 * np.arange(4 * n, dtype=np.uint64)
    g = (np.sqrt(-2.0 * np.log(uniform01(seed, c))) * np.cos(2.0 * math.pi * uniform01(seed, c + np.uint64(1)))).reshape(n, 4)
    q = g / np.linalg.norm(g, axis=1)[:, None]
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    A = np.empty((n, 3, 3))
    A[:, 0, 0] = 1 - 2 * (y * y + z * z); A[:, 0, 1] = 2 * (x * y - w * z); A[:, 0, 2] = 2 * (x * z + w * y)
    A[:, 1, 0] = 2 * (x * y + w * z); A[:, 1, 1] = 1 - 2 * (x * x + z * z); A[:, 1, 2] = 2 * (y * z - w * x)
    A[:, 2, 0] = 2 * (x * z - w * y); A[:, 2, 1] = 2 * (y * z + w * x); A[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return A


def rigid_state(n_mol: int, body: np.ndarray, mol_density: float, temperature: float, seed: int):
    """Rigid molecules on a simple-cubic grid of centres with seeded random orientations: (R, A, V, pi, box).
    V: Gaussian with variance T / M per component, zero net momentum; body-frame angular momentum pi_k: Gaussian with
    variance I_k T (equipartition)."""
    box = box_edge(n_mol, mol_density)
    R = sc_lattice(n_mol, box)
    A = random_rotations(n_mol, seed)
    M = float(body.shape[0])
    V = gaussian_velocities(n_mol, temperature / M, seed)
    I = body_inertia(body)
    g = gaussian_velocities(n_mol, 1.0, seed + 104729)          # unit-variance Gaussians (mean removed: harmless)
    pi = g * np.sqrt(I * temperature)[None, :]
    return R, A, V, pi, box


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
    elif cfg.lattice == "walk":          # OVERLAPPING: to be pushed apart by the library's md_pushoff before use
        r, bonds, box = chain_walks(cfg.n_chains, cfg.chain_len, cfg.density, seed)
    else:
        raise ValueError(cfg.lattice)
    if jitter_amp > 0.0:
        r = jitter(r, jitter_amp, seed + 7919, box)
    v = gaussian_velocities(cfg.n_atoms, cfg.temperature, seed)
    return r, v, bonds, box
