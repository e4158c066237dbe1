"""Helpers shared by the GPU parity tests: tolerances are north_star's (BASELINE.json) and are written here once."""
import math

import numpy as np

from md_workloads import make_state

FORCE_RTOL = 1e-10      # per-atom max relative force error (SURVEY 8(c) A11 norm)
POS_ATOL = 1e-9         # positions after 10 steps, sigma units, component-wise modulo L
ENERGY_RTOL = 1e-9      # ke, pe separately after 10 steps


def force_rel_err(f, ref):
    frms = math.sqrt(float((ref * ref).sum()) / ref.shape[0])
    den = np.maximum(np.abs(ref).max(1), frms if frms > 0 else 1.0)
    return float((np.abs(f - ref).max(1) / den).max())


def pos_err(a, b, box):
    d = a - b
    d -= box * np.round(d / box)
    return float(np.abs(d).max())


def sets_equal(gpu_counts, gpu_list, oracle):
    """Exact neighbor-set equality, both given per ORIGINAL atom id.  Returns (n_mismatching_atoms, first index)."""
    ocounts, oflat = oracle.neighbors()
    if not np.array_equal(gpu_counts, ocounts):
        bad = np.nonzero(gpu_counts != ocounts)[0]
        return len(bad), int(bad[0])
    n = len(ocounts)
    mmax = gpu_list.shape[1]
    # sort each GPU row (pad -1 -> large), flatten valid entries, compare with the oracle's sorted CSR rows
    g = np.where(gpu_list < 0, np.iinfo(np.int32).max, gpu_list)
    g.sort(axis=1)
    mask = np.arange(mmax)[None, :] < gpu_counts[:, None]
    gflat = g[mask]
    off = np.concatenate([[0], np.cumsum(ocounts, dtype=np.int64)])
    rows = np.repeat(np.arange(n), ocounts)
    order = np.lexsort((oflat, rows))
    oflat_sorted = oflat[order]
    if np.array_equal(gflat, oflat_sorted):
        return 0, -1
    bad_rows = np.unique(rows[gflat != oflat_sorted])
    return len(bad_rows), int(bad_rows[0])


def prepared_state(md, cfg, seed=1, jitter_amp=0.0):
    """(r, v, bonds, box) of a config as BOTH sides receive it.  Lattice starts come straight from md_workloads.  The
    random-walk chain start (cfg.lattice == "walk") overlaps; it is pushed apart by the library's md_pushoff --
    initialisation, outside the parity-checked path -- and the result is handed to the oracle as data."""
    r, v, bonds, box = make_state(cfg, seed, jitter_amp=jitter_amp)
    if cfg.lattice != "walk":
        return r, v, bonds, box
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none")
    rep = g.pushoff(r, bonds, cfg.fene_k, cfg.fene_r0, temperature=cfg.temperature, seed=seed)
    assert rep["min_nonbonded"] > 0.85 and rep["max_bond"] < 1.3, rep
    r, v = g.positions(), g.velocities()
    g.close()
    return r, v, bonds, box
