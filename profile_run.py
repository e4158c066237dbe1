"""Short, deterministic run of the hot path for profilers (ncu): melt the lattice, then a few steps and forced
rebuilds so that every kernel of the path appears with real work in the last launches.

    python profile_run.py --config wca_2m_dr05 --melt 100 --steps 12 --rebuilds 2 --flags 1

(--flags 1 = MD_FLAG_NO_GRAPH: ncu lists kernels only when they are launched one by one.)  A harness for the commands
quoted in profiles/; not part of the product package.
"""
from __future__ import annotations

import argparse
import os
import sys

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))

from md_workloads import get_config, make_state  # noqa: E402
from paper_2003_14061_b200 import MDSystem  # noqa: E402


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="wca_2m")
    ap.add_argument("--melt", type=int, default=100)
    ap.add_argument("--steps", type=int, default=12)
    ap.add_argument("--rebuilds", type=int, default=2)
    ap.add_argument("--variant", default="full")
    ap.add_argument("--mode", default="fused")
    ap.add_argument("--block", type=int, default=0)
    ap.add_argument("--flags", type=int, default=0, help="md_params.flags (2 = MD_FLAG_GLOBAL_W)")
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"])
    ap.add_argument("--cell-split", type=int, default=0)
    a = ap.parse_args()
    cfg = get_config(a.config)
    r, v, bonds, box = make_state(cfg, 1)
    g = MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", force_variant=a.variant,
                 step_mode=a.mode if a.variant == "full" else "split", block_size=a.block, flags=a.flags, precision=a.precision,
                 cell_split_x=a.cell_split)
    if cfg.lattice == "walk":        # configs[4]: overlapping random walks, pushed apart by the library first
        g.pushoff(r, bonds, cfg.fene_k, cfg.fene_r0, temperature=cfg.temperature, seed=1)
    else:
        g.set_state(r, v)
        if bonds is not None:
            g.set_bonds(bonds, cfg.fene_k, cfg.fene_r0)
    g.step(a.melt)
    e = g.energies()
    print(f"melted: T={e.ke / (1.5 * (cfg.n_atoms - 1)):.4f} mean_nb={e.mean_neighbors:.3f} max_nb={e.max_neighbors} "
          f"rebuilds={e.n_rebuilds} launches={g.info()['kernel_launches']}")
    for _ in range(a.rebuilds):
        g.rebuild_neighbors()
    g.step(a.steps)
    e = g.energies()
    print(f"done: E/N={e.total / cfg.n_atoms:.9f} rebuilds={e.n_rebuilds} launches={g.info()['kernel_launches']}")


if __name__ == "__main__":
    main()
