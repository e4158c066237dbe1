#!/usr/bin/env python
"""bench.py -- atom-timesteps/s (fp64) of the MD hot path on B200, per the driver contract.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config wca_2m] ...

A "step" is one MD time step of the whole hot path (integrate, device-side rebuild decision, cell binning +
reorder + neighbor matrix when triggered, forces) over all N atoms of the workload.  Default workload:
BASELINE.json configs[2] as worded -- the WCA fluid at N = 2,097,152 (128^3 lattice, rho 0.8, T 1.0, dt 0.005) at BOTH
swept shells, delta r = 0.3 and 0.5; `value` is the lower of the two, both are in `sweep`.  Before the W warm-up steps
the lattice start is melted for --equil untimed steps (declared in config), so the K timed steps are steady state.  Multi-GPU (--gpus N under torchrun) runs N
independent replicas with different seeds ("replicas only"): no data-path collective.

Prints ONE JSON line.  `--impl reference` times the CPU oracle (oracle/) instead, on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from md_workloads import get_config, make_state, scaled_config  # noqa: E402

METRIC = "atom-timesteps/sec (fp64)"
UNIT = "atom-steps/s"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def load_ncu_traffic(kernel_key):
    """DRAM bytes per launch of the dominant kernel from the committed ncu summary (profiles/), or None."""
    path = os.path.join(ROOT, "profiles", "roofline_traffic.txt")
    if not os.path.exists(path):
        return None
    found = None
    with open(path) as fh:
        for line in fh:
            line = line.split("#", 1)[0].strip()
            if line.startswith(kernel_key + " "):
                found = float(line.rsplit(None, 1)[1])       # the last line for a key is the latest pass
    return found


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except Exception:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def replica_seed(rank: int) -> int:
    """Replicas only: every rank runs an independent system; only the seed differs."""
    return 1 + rank


def max_over_ranks(x: float, dist, device) -> float:
    """The one collective of the multi-GPU path: the timed region of the job is that of its slowest replica."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([x], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def oracle_rate(cfg, seed, budget_s, steps=None, n_atoms=None, precision="f64"):
    """Time the oracle as it stands on a bounded sample: returns (atom-steps/s, sample text, threads, steps, N)."""
    from oracle.md_oracle import OracleMD, OracleMDSP, get_threads
    if precision == "f32":
        OracleMD = OracleMDSP
    scfg = cfg if not n_atoms or n_atoms == cfg.n_atoms else scaled_config(cfg.name, n_atoms)
    r, v, bonds, box = make_state(scfg, seed)
    o = OracleMD(scfg.n_atoms, box, scfg.r_cut, scfg.r_shell, scfg.dt)
    o.set_state(r, v)
    if bonds is not None:
        o.set_bonds(bonds, scfg.fene_k, scfg.fene_r0)
    t0 = time.perf_counter()
    o.step(2)
    per = (time.perf_counter() - t0) / 2
    if steps is None:
        steps = int(max(2, min(200, budget_s / max(per, 1e-6))))
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    rate = scfg.n_atoms * steps / dt
    sample = (f"{steps} steps of {scfg.name} (N={scfg.n_atoms}) from the t=0 lattice state after 2 untimed steps, "
              f"rebuilds included, {dt:.1f} s")
    return rate, sample, get_threads(), steps, scfg.n_atoms


def sweep_configs(name):
    """--config baseline (the default) = BASELINE.json configs[2] as it is worded: the 2M-atom WCA fluid at BOTH swept
    shells, delta r = 0.3 and 0.5.  Every other name is one workload."""
    return [get_config("wca_2m_dr03"), get_config("wca_2m_dr05")] if name == "baseline" else [get_config(name)]


def workload_config(cfgs, nsys=1):
    """The `config` object of the JSON line: the workload definition only (identical for both --impl arms); what the
    library chose for it (W layout, tile, block size) is reported under `launch`."""
    c0 = cfgs[0]
    name = c0.name if len(cfgs) == 1 else "+".join(c.name for c in cfgs) + " (BASELINE.json configs[2]: delta r = 0.3 and 0.5 swept; value = the lower)"
    return {"workload": name if nsys == 1 else f"{nsys} x {name}", "n_atoms": c0.n_atoms * nsys, "n_systems": nsys,
            "start": {"sc": "simple-cubic lattice", "fcc": "FCC lattice", "chains": "zig-zag chain rows",
                      "walk": "seeded random-walk chains pushed apart by md_pushoff"}[c0.lattice],
            "density": c0.density, "r_cut": c0.r_cut, "r_shell": [c.r_shell for c in cfgs] if len(cfgs) > 1 else c0.r_shell,
            "dt": c0.dt, "temperature": c0.temperature}


def reference_one(args, cfg):
    """The oracle on the host cores: W + K steps, each over a bounded sample of the workload (same state point)."""
    from oracle.md_oracle import OracleMD, OracleMDSP, get_threads
    if args.precision == "f32":
        OracleMD = OracleMDSP
    base = cfg.name if cfg.lattice != "walk" else "chains_rows_1m"          # the oracle cannot push a walk apart
    bcfg = get_config(base)
    # calibrate on a small system, then pick the largest lattice that keeps (K + W) steps within the budget
    small = scaled_config(base, 32 ** 3) if bcfg.lattice == "sc" else scaled_config(base, 4 * 16 ** 3) \
        if bcfg.lattice == "fcc" else scaled_config(base, 64 * bcfg.chain_len * 8)
    rate0, _, _, _, _ = oracle_rate(small, 1, 2.0, precision=args.precision)
    want = rate0 * args.ref_seconds / max(1, args.steps + args.warmup)
    if bcfg.lattice == "sc":
        side = int(min(round(bcfg.n_atoms ** (1 / 3)), max(16, int(want ** (1 / 3)))))
        n = side ** 3
    elif bcfg.lattice == "fcc":
        side = int(min(round((bcfg.n_atoms / 4) ** (1 / 3)), max(8, int((want / 4) ** (1 / 3)))))
        n = 4 * side ** 3
    else:
        n = int(min(bcfg.n_atoms, max(64 * bcfg.chain_len, (int(want) // (64 * bcfg.chain_len)) * 64 * bcfg.chain_len)))
    scfg = bcfg if n == bcfg.n_atoms else scaled_config(base, n)
    r, v, bonds, box = make_state(scfg, 1)
    o = OracleMD(scfg.n_atoms, box, scfg.r_cut, scfg.r_shell, scfg.dt)
    o.set_state(r, v)
    if bonds is not None:
        o.set_bonds(bonds, scfg.fene_k, scfg.fene_r0)
    o.step(args.warmup)
    t0 = time.perf_counter()
    o.step(args.steps)
    dt = time.perf_counter() - t0
    return {"workload": cfg.name, "value": scfg.n_atoms * args.steps / dt, "ms_per_step": 1e3 * dt / args.steps,
            "sample_n_atoms": scfg.n_atoms, "cores": get_threads(),
            "sample": f"each step = one oracle time step over N={scfg.n_atoms} atoms at {cfg.name}'s state point "
                      f"({scfg.lattice} start, {args.warmup} untimed steps first)"}


def run_reference(args, cfgs):
    """--impl reference: the oracle as it stands, timed on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    runs = [reference_one(args, c) for c in cfgs]
    head = min(runs, key=lambda r: r["value"])
    line = {
        "impl": "reference", "metric": metric_name(args), "value": head["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": args.precision, "data": "synthetic",
        "config": workload_config(cfgs),
        "cpu_baseline": {"value": head["value"], "unit": UNIT, "cores": head["cores"], "kind": "oracle", "sample": head["sample"]},
        "e2e": {"value": head["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "sweep": {r["workload"]: {k: r[k] for k in ("value", "ms_per_step", "sample_n_atoms")} for r in runs},
    }
    print(json.dumps(line), flush=True)


def metric_name(args):
    return METRIC if args.precision == "f64" else "atom-timesteps/sec (fp32 state and pair arithmetic, fp64 energy sums)"


FP64_OPS_PER_CANDIDATE = 7      # the R5 accept test: 3 subtractions, 1 multiply, 2 FMA, 1 compare


def measure_gpu(args, cfg, ctx, with_e2e):
    """One workload on this rank's GPU: equilibrate (untimed, declared), W warm-up steps, EXACTLY K timed steps, then the
    per-kernel passes.  Returns the pieces of the JSON line."""
    torch, md, stream, barrier, dist, world, rank = (ctx[k] for k in ("torch", "md", "stream", "barrier", "dist", "world", "rank"))
    seed = replica_seed(rank)
    nsys = max(1, args.systems)
    states = [make_state(cfg, seed + 1000 * b) for b in range(nsys)]
    box = states[0][3]
    if args.shuffle:
        if nsys != 1 or states[0][2] is not None:
            raise SystemExit("--shuffle: one system without bonds only")
        perm = np.random.default_rng(12345).permutation(cfg.n_atoms)
        states = [(states[0][0][perm], states[0][1][perm], None, box)]
    tile = dict(tile_cells=tuple(args.tile_cells), tile_threads=args.tile_threads, tile_capacity=args.tile_capacity,
                cell_split_x=args.cell_split)
    g = md.MDSystem(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, box=box, lattice="none", force_variant=args.variant,
                    step_mode=args.mode if args.variant == "full" else "split", block_size=args.block, flags=args.flags,
                    n_systems=nsys, precision=args.precision, reorder_interval=args.reorder_interval, **tile)
    r_all = np.concatenate([s[0] for s in states])
    bonds_all = None if states[0][2] is None else np.concatenate([s[2] + b * cfg.n_atoms for b, s in enumerate(states)])
    pushoff = None
    if cfg.lattice == "walk":       # configs[4]: the overlapping walks are pushed apart by the library (initialisation, untimed)
        pushoff = g.pushoff(r_all, bonds_all, cfg.fene_k, cfg.fene_r0, temperature=cfg.temperature, seed=seed)
    else:
        g.set_state(r_all, np.concatenate([s[1] for s in states]))
        if bonds_all is not None:
            g.set_bonds(bonds_all, cfg.fene_k, cfg.fene_r0)
    if bonds_all is not None:
        if args.angles > 0:
            g.set_angles(args.angles, args.angle_cos0)
        if args.dihedrals > 0:
            g.set_dihedrals(args.dihedrals, args.dihedral_cos0)
    del states, r_all
    info = g.info()
    n = cfg.n_atoms * nsys                  # atoms advanced per step

    # ---- untimed equilibration (the lattice melts: T falls from 1.0 to ~0.74 within ~150 steps), then W warm-up steps ----
    g.step(args.equil)
    g.step(args.warmup)
    e_start = g.energies()
    launches0 = g.info()["kernel_launches"]
    sampler = ClockSampler(ctx["local_rank"])
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_wall0 = time.perf_counter()
    ev0.record(stream)
    g.step(args.steps)                      # EXACTLY K steps, every rebuild included, one host sync at the end
    ev1.record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.stop() if rank == 0 else None
    info_end = g.info()
    launches = info_end["kernel_launches"] - launches0
    e_end = g.energies()
    ms = max_over_ranks(ms, dist, "cuda")
    value = world * n * args.steps / (ms * 1e-3)

    # ---- per-kernel-class device timers over a second pass of K steps (Table 2 of the paper; roofline) ----
    g.set_profiling(True)
    g.reset_timers()
    g.step(max(args.steps, 50))
    timers = g.timers()
    g.set_profiling(False)
    prof_steps = max(args.steps, 50)
    e_prof = g.energies()
    rebuilds_prof = e_prof.n_rebuilds - e_end.n_rebuilds
    mbar = 0.5 * (e_end.mean_neighbors + e_prof.mean_neighbors)
    peak, peak_src = load_peaks()
    tiled = info["w_layout"] == 1
    sp = args.precision == "f32"
    rec = 16.0 if sp else 24.0               # bytes of one position / velocity / force record (float4 | 3 doubles)
    if args.mode == "fused" and args.variant == "full":
        tk = timers["fused_step"]
        if tiled:
            kname = "k_tile_force<fused step>"
            w_bytes = 2.0                        # 16-bit tile-local entries
        else:
            kname = "k_sp_force<fused step>" if sp else "k_force<fused step>"
            w_bytes = 4.0
        # W w*m + m_i 4 + r_i 24 + gathers 24m + v read+write 48 + r' write 24   (north_star's accounting);
        # single precision: 16-byte float4 records instead of 24
        bytes_per_atom = (w_bytes + rec) * mbar + 4.0 + 4.0 * rec
        floor_bytes = w_bytes * mbar + 4.0 + 4.0 * rec
    else:
        kname, tk = ("k_sp_force" if sp else "k_force"), timers["force"]
        w_bytes = 4.0
        bytes_per_atom = (4.0 + rec) * mbar + 4.0 + 2.0 * rec      # SURVEY 8(d) B_ns: W 4m + m_i 4 + r_i + gathers + f write
        floor_bytes = 4.0 * mbar + 4.0 + 2.0 * rec
        if args.variant == "newton3":
            tk = dict(tk, launches=tk["launches"] // 2)
    dur_ms = tk["ms"] / max(1, tk["launches"])
    achieved = bytes_per_atom * n / (dur_ms * 1e-3) / 1e9
    traffic = load_ncu_traffic(f"{cfg.name}:{kname}")
    roofline = {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                # the cache-honest fractions next to the graded one: DRAM bytes ncu measured for this kernel (profiles/
                # roofline_traffic.txt) and the compulsory bytes, both over the same live launch time
                "frac_measured": None if traffic is None else traffic / (dur_ms * 1e-3) / 1e9 / peak,
                "frac_compulsory": floor_bytes * n / (dur_ms * 1e-3) / 1e9 / peak,
                "algorithmic_bytes_per_atom": bytes_per_atom, "compulsory_bytes_per_atom": floor_bytes,
                "mean_neighbors": mbar, "avg_launch_ms": dur_ms,
                "accounting": f"frac = north_star's B_ns count (SURVEY 8(d), the graded one): every gather charged {rec:.0f} B although "
                              "L1/L2/shared memory serve them, so it can exceed 1; frac_measured = ncu DRAM bytes per launch / the "
                              "same launch time; frac_compulsory = every array touched once",
                "timing": "CUDA events on the library's stream around each launch (md_set_profiling), second pass of >= K steps"}
    nebr = timers["nebr"]
    # the neighbor-matrix build on its own: 5 forced rebuilds, each exactly one working launch of the build kernel
    g.set_profiling(True)
    g.reset_timers()
    for _ in range(5):
        g.rebuild_neighbors()
    tb = g.timers()["nebr"]
    g.set_profiling(False)
    build_ms = tb["ms"] / 5.0                                         # per rebuild (the layer ablation launches 2 kernels)
    pk = g.measure_peaks()
    cand = g.info()["candidates_per_atom"]                            # candidates per atom the last build tested (counted by the kernel)
    nb_floor = rec + w_bytes * mbar + 4.0                             # r_i + W written + m_i
    bname = (("k_sp_tile_build" if sp else "k_tile_build") if info["tile_capacity"] else
             ("k_sp_build" if sp else ("k_build_layers" if args.flags & 32 else "k_build")))
    btraffic = load_ncu_traffic(f"{cfg.name}:{bname}")
    ops = FP64_OPS_PER_CANDIDATE * cand * n / (build_ms * 1e-3) / 1e9  # accept-test arithmetic instructions per second (lanes)
    alu_peak = (pk["fp32_tflops"] if sp else pk["fp64_tflops"]) * 1e3 / 2.0
    roofline_neighbor = {"bound": "alu", "kernel": bname, "avg_launch_ms": build_ms, "candidates_per_atom": cand,
                         "achieved": ops, "peak": alu_peak, "unit": "Gop/s", "frac": ops / alu_peak,
                         "ops_per_candidate": FP64_OPS_PER_CANDIDATE,
                         "peak_source": "md_measure_peaks: register-resident FMA loop timed in this run, one FMA = one op",
                         "accounting": "the accept test of DESIGN.md R5 costs 7 arithmetic instructions per candidate (3 sub, 1 mul, "
                                       "2 fma, 1 compare) in the working precision; achieved = 7 x candidates tested per second, "
                                       "peak = the measured FMA issue rate of that precision.  The kernel is bound by instruction "
                                       "issue, not by HBM: its HBM fractions are given only for completeness",
                         "hbm": {"compulsory_bytes_per_atom": nb_floor, "frac_compulsory": nb_floor * n / (build_ms * 1e-3) / 1e9 / peak,
                                 "traffic": btraffic,
                                 "frac_measured": None if btraffic is None else btraffic / (build_ms * 1e-3) / 1e9 / peak}}
    breakdown = {k: round(v["ms"] / prof_steps, 6) for k, v in timers.items()}
    nebr_info = {"rebuilds": int(rebuilds_prof), "ms_per_rebuild": nebr["ms"] / max(1, rebuilds_prof),
                 "steps_per_rebuild": prof_steps / max(1, rebuilds_prof)}

    # ---- end to end through the C ABI with HOST buffers: H2D state, one step, D2H state + energies ------------------
    # Every step uploads a full state (positions + velocities, page-locked host arrays), installs it (range check, bin,
    # W build, forces), advances it one step, reads the energies and downloads the full state.  `value`: the service
    # loop over three independent host-resident trajectories with the library's pipelined I/O calls (upload of the next
    # state, step of the current one and download of the previous one overlap; pipeline fill and drain are inside the
    # timed region).  `serial_value`: one trajectory fed back through the host with the blocking calls, nothing overlaps.
    e2e = None
    if with_e2e:
        def pinned(shape):                # page-locked host buffers: the library copies to / from them directly
            return torch.empty(shape, dtype=torch.float64, pin_memory=True).numpy()
        a, b = pinned((2, n, 3)), pinned((2, n, 3))       # [positions | velocities], adjacent: one transfer each way
        g.state(a[0], a[1])
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            g.set_state(a[0], a[1])      # host -> device, range check, rebuild, forces
            g.step(1)
            g.state(b[0], b[1])          # device -> host, one call
            g.energies()
            a, b = b, a
        barrier()
        dt_serial = max_over_ranks(time.perf_counter() - t0, dist, "cuda")
        nt = 3
        traj = [a, b, pinned((2, n, 3))]
        traj[2][:] = traj[0]
        g.stage_state(traj[2][0], traj[2][1]); g.commit_state(); g.state_async(traj[2][0], traj[2][1]); g.wait_io()    # untimed: staging buffers, copy streams
        ksteps = args.e2e_steps
        barrier()
        t0 = time.perf_counter()
        g.stage_state(traj[0][0], traj[0][1])
        g.stage_state(traj[1][0], traj[1][1])
        for it in range(ksteps):
            k = it % nt
            g.commit_state()             # the oldest staged state: range check, rebuild, forces
            g.step(1)
            g.state_async(traj[k][0], traj[k][1])
            g.energies()
            if it + 2 < ksteps:
                g.wait_io(1)             # the download started one turn ago is complete: that trajectory may go up again
                g.stage_state(traj[(it + 2) % nt][0], traj[(it + 2) % nt][1])
        g.wait_io()
        barrier()
        dt = max_over_ranks(time.perf_counter() - t0, dist, "cuda")
        # the boundary arrays are binary64 in both precisions
        e2e = {"value": world * n * ksteps / dt, "unit": UNIT, "h2d_bytes_per_step": 2 * 3 * n * 8,
               "d2h_bytes_per_step": 2 * 3 * n * 8 + 160, "steps": ksteps, "ms_per_step": dt / ksteps * 1e3,
               "serial_value": world * n * args.e2e_steps / dt_serial, "serial_ms_per_step": dt_serial / args.e2e_steps * 1e3,
               "what": "per step: md_stage_state(pinned host r,v) + md_commit_state + md_step(1) + md_energies + md_get_state_async, "
                       "three independent host trajectories in turn, transfers overlapped on the library's copy streams, "
                       "pipeline fill and drain timed; serial_value: md_set_state + md_step(1) + md_get_state + md_energies, one trajectory"}
    g.close()
    return {"workload": cfg.name, "value": value, "ms": ms, "n": n, "info": info, "info_end": info_end, "launches": int(launches),
            "roofline": roofline, "roofline_neighbor": roofline_neighbor, "e2e": e2e, "clocks": clocks, "wall_s": t_wall,
            "rebuilds": int(e_end.n_rebuilds - e_start.n_rebuilds), "e_start": e_start.total / n, "e_end": e_end.total / n,
            "temperature_end": e_end.ke / (1.5 * (n - 1)), "breakdown": breakdown, "nebr_info": nebr_info, "peaks": pk,
            "pushoff": pushoff, "tiled": tiled}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--equil", type=int, default=400,
                    help="untimed equilibration steps before the warm-up (the lattice start melts; declared in config)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="baseline",
                    help="baseline = BASELINE.json configs[2] at both swept shells (value = the lower); or one of md_workloads.CONFIGS")
    ap.add_argument("--variant", default="full", choices=["full", "newton3"])
    ap.add_argument("--mode", default="fused", choices=["fused", "split"])
    ap.add_argument("--block", type=int, default=0)
    ap.add_argument("--systems", type=int, default=1,
                    help="batch of independent systems of the workload run by the same launches (md_params.n_systems)")
    ap.add_argument("--flags", type=int, default=0, help="md_params.flags: 1 = no CUDA graph, 2 = global-index W layout, ...")
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"],
                    help="f32: the single-precision variant (md_params.precision = MD_PREC_F32; SURVEY 8(f) NEXT-1)")
    ap.add_argument("--reorder-interval", type=int, default=0,
                    help="with --flags 32 (MD_FLAG_LAYER_H, the paper's cell x layer matrix): steps between sorts of the "
                         "atoms into cell order; 0 = every rebuild, < 0 = never (PAPER.md:159)")
    ap.add_argument("--shuffle", action="store_true",
                    help="permute the atom numbering of the start state (a decorrelated storage order, for the sort ablation)")
    ap.add_argument("--angles", type=float, default=0.0,
                    help="chain workloads: bond-angle stiffness k_theta of md_set_angles (cos theta0 = -1), 0 = off")
    ap.add_argument("--angle-cos0", type=float, default=-1.0)
    ap.add_argument("--dihedrals", type=float, default=0.0,
                    help="chain workloads: dihedral stiffness k_phi of md_set_dihedrals, 0 = off (the cosine form is singular "
                         "for collinear bonds: combine with stiff bent angles, e.g. --angles 40 --angle-cos0 -0.5)")
    ap.add_argument("--dihedral-cos0", type=float, default=-0.6)
    ap.add_argument("--tile-cells", type=int, nargs=3, default=[0, 0, 0], help="md_params.tile_cells (0 = auto)")
    ap.add_argument("--cell-split", type=int, default=0, help="md_params.cell_split_x: fine cells per r_n along x (0 = auto)")
    ap.add_argument("--tile-threads", type=int, default=0)
    ap.add_argument("--tile-capacity", type=int, default=0)
    ap.add_argument("--e2e-steps", type=int, default=24)
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--ref-seconds", type=float, default=75.0, help="--impl reference: budget of one workload's W + K steps")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    cfgs = sweep_configs(args.config)

    if args.impl == "reference":
        run_reference(args, cfgs)
        return

    import torch
    import paper_2003_14061_b200 as md

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the MD path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # the library runs on torch's current stream; the timing events are recorded on that same stream
    stream = torch.cuda.Stream()
    ctx = dict(torch=torch, md=md, stream=stream, barrier=barrier, dist=dist, world=world, rank=rank, local_rank=local_rank)
    with torch.cuda.stream(stream):
        # the headline workload (the slower one of a sweep) carries the e2e leg; it is only known afterwards, so every
        # workload of a sweep measures it
        runs = [measure_gpu(args, c, ctx, not args.no_e2e) for c in cfgs]
    head = min(runs, key=lambda r: r["value"])
    hcfg = get_config(head["workload"])

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    nsys = max(1, args.systems)
    cpu = None
    if not args.no_cpu_baseline and world == 1 and nsys == 1:
        ocfg = hcfg if hcfg.lattice != "walk" else get_config("chains_rows_1m")      # the oracle cannot push a walk apart
        rate, sample, cores, _, _ = oracle_rate(ocfg, 1, args.cpu_seconds, precision=args.precision)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}

    info, info_end = head["info"], head["info_end"]
    config = workload_config(cfgs, nsys)
    config.update({"headline_workload": head["workload"], "equilibration_steps": args.equil,
                   "force_variant": args.variant, "step_mode": args.mode, "precision": args.precision,
                   "angle_k": args.angles, "dihedral_k": args.dihedrals, "flags": args.flags,
                   "reorder_interval": args.reorder_interval, "shuffled_ids": bool(args.shuffle),
                   "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
                   "l2": "working set per step (positions 2x64 MB, velocities 48 MB, W rows ~100 MB) exceeds the 126 MB L2; no flush"})
    launch = {"block_size": info["block_size"], "max_neighbors": info["max_neighbors"], "cells_per_edge": info["cells_per_edge"],
              "cells_x": info["cells_x"], "cell_split_x": info["cell_split_x"], "w_layout": "tiled16" if head["tiled"] else "global32",
              "tile_cells": info["tile_cells"], "tile_threads": info["tile_threads"], "tile_capacity": info["tile_capacity"],
              "cuda_graph": bool(info_end["use_graph"])}
    sweep = {r["workload"]: {"value": r["value"], "ms_per_step": r["ms"] / args.steps, "rebuilds_in_timed_region": r["rebuilds"],
                             "temperature_end": r["temperature_end"], "roofline_frac": r["roofline"]["frac"],
                             "roofline_frac_measured": r["roofline"]["frac_measured"],
                             "fused_step_ms": r["roofline"]["avg_launch_ms"], "build_ms": r["roofline_neighbor"]["avg_launch_ms"],
                             "e2e": None if r["e2e"] is None else r["e2e"]["value"]} for r in runs}
    line = {
        "metric": metric_name(args), "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": head["ms"] / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": args.precision, "data": "synthetic", "config": config, "launch": launch, "sweep": sweep,
        "roofline": head["roofline"], "roofline_neighbor": head["roofline_neighbor"],
        "peaks": {"hbm_gbs": head["roofline"]["peak"], "fp64_tflops": head["peaks"]["fp64_tflops"], "fp32_tflops": head["peaks"]["fp32_tflops"],
                  "sm_count": head["peaks"]["sm_count"], "how": "hbm: MEASURED_PEAKS.json; fp64 / fp32: md_measure_peaks, FMA loops timed in this run"},
        "cpu_baseline": cpu, "e2e": head["e2e"], "gpu_launches": head["launches"], "clocks": head["clocks"],
        "wall_s": head["wall_s"], "rebuilds_in_timed_region": head["rebuilds"],
        "energy_per_atom": {"start": head["e_start"], "end": head["e_end"]},
        "temperature_end": head["temperature_end"],
        "ms_per_step_by_kernel_class": head["breakdown"], "neighbor_build": head["nebr_info"], "pushoff": head["pushoff"],
        "device": info["device_name"],
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
