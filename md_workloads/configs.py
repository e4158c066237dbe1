"""The five BASELINE.json workloads (plus the swept shell widths of config 3).

Every number here is copied from BASELINE.json:configs; nothing is derived from
either implementation.  `scaled_config` keeps the state point of a config and
shrinks N so the CPU oracle can run it in seconds.
"""
from __future__ import annotations

import dataclasses
from dataclasses import dataclass

R_WCA = 2.0 ** (1.0 / 6.0)


@dataclass(frozen=True)
class MDConfig:
    name: str
    n_atoms: int
    lattice: str          # "sc" | "fcc" | "chains" (zig-zag rows) | "walk" (overlapping random walks)
    density: float
    temperature: float
    r_cut: float
    r_shell: float        # the paper's delta (item (5))
    dt: float
    n_steps: int
    chain_len: int = 0
    n_chains: int = 0
    fene_k: float = 0.0
    fene_r0: float = 0.0

    @property
    def box(self) -> float:
        return (self.n_atoms / self.density) ** (1.0 / 3.0)


CONFIGS = {
    # configs[0]
    "wca_4k": MDConfig("wca_4k", 16 ** 3, "sc", 0.8, 1.0, R_WCA, 0.4, 0.005, 1000),
    # configs[1]
    "wca_262k": MDConfig("wca_262k", 64 ** 3, "sc", 0.8, 1.0, R_WCA, 0.4, 0.005, 1000),
    # configs[2]: delta r = 0.3 and 0.5 swept; 0.4 is the mid-point used for the headline
    "wca_2m_dr03": MDConfig("wca_2m_dr03", 128 ** 3, "sc", 0.8, 1.0, R_WCA, 0.3, 0.005, 500),
    "wca_2m": MDConfig("wca_2m", 128 ** 3, "sc", 0.8, 1.0, R_WCA, 0.4, 0.005, 500),
    "wca_2m_dr05": MDConfig("wca_2m_dr05", 128 ** 3, "sc", 0.8, 1.0, R_WCA, 0.5, 0.005, 500),
    # configs[3]
    "lj_1m": MDConfig("lj_1m", 4 * 64 ** 3, "fcc", 0.8442, 0.72, 2.5, 0.3, 0.004, 500),
    # configs[4]: 16,384 chains x 64 beads grown as seeded random walks (md_workloads.chain_walks); the overlapping start
    # is pushed apart by the library (md_pushoff) before any timed or parity-checked step
    "chains_1m": MDConfig("chains_1m", 16384 * 64, "walk", 0.85, 1.0, R_WCA, 0.4, 0.005, 500,
                          chain_len=64, n_chains=16384, fene_k=30.0, fene_r0=1.5),
    # extra input, not a BASELINE.json config: the same melt started from overlap-free zig-zag rows (md_workloads.chain_melt),
    # usable without a push-off (CPU-only tests, small parity cases)
    "chains_rows_1m": MDConfig("chains_rows_1m", 16384 * 64, "chains", 0.85, 1.0, R_WCA, 0.4, 0.005, 500,
                               chain_len=64, n_chains=16384, fene_k=30.0, fene_r0=1.5),
    # Context only (not BASELINE.json configs): the paper's OWN state points and shell at the
    # N = 128^3 row of its Table 1, cubic-grid start, for a line next to that table in BASELINE.md.
    "paper_sp_2m": MDConfig("paper_sp_2m", 128 ** 3, "sc", 0.8, 1.0, R_WCA, 0.6, 0.005, 500),
    "paper_lj_2m": MDConfig("paper_lj_2m", 128 ** 3, "sc", 0.38, 1.2, 2.5, 0.6, 0.005, 500),
}


def get_config(name: str) -> MDConfig:
    return CONFIGS[name]


def scaled_config(name: str, n_atoms: int, **overrides) -> MDConfig:
    """Same state point, smaller system (for parity cases the oracle finishes in seconds)."""
    cfg = CONFIGS[name]
    kw = dict(n_atoms=n_atoms, name=f"{cfg.name}@{n_atoms}")
    if cfg.lattice in ("chains", "walk"):
        chain_len = overrides.pop("chain_len", cfg.chain_len)
        if n_atoms % chain_len:
            raise ValueError("n_atoms must be a multiple of chain_len")
        kw.update(chain_len=chain_len, n_chains=n_atoms // chain_len)
    kw.update(overrides)
    return dataclasses.replace(cfg, **kw)
