"""Thin ctypes binding of libmd_b200.so (include/md_b200.h): argument marshalling only.

Every step of the MD path runs in the CUDA kernels of the library.  PyTorch supplies device memory
(its caching allocator, through md_set_allocator) and the stream.  There is no CPU fallback: if the
library is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libmd_b200.so")

MD_OK, MD_ERR_INVALID, MD_ERR_NEBR_OVERFLOW, MD_ERR_BOND_BROKEN = 0, -1, -2, -3
MD_ERR_NONFINITE, MD_ERR_CUDA, MD_ERR_UNSUPPORTED, MD_ERR_NOMEM, MD_ERR_TILE_OVERFLOW, MD_ERR_CELL_OVERFLOW = -4, -5, -6, -7, -8, -9
FLAG_NO_GRAPH, FLAG_GLOBAL_W, FLAG_TILED_W, FLAG_GATHER_W, FLAG_W_TRANSPOSED, FLAG_LAYER_H, FLAG_NO_PERSIST = 1, 2, 4, 8, 16, 32, 64
LATTICE = {"auto": 0, "sc": 1, "fcc": 2, "none": 3}
FORCE_VARIANT = {"full": 0, "newton3": 1}
STEP_MODE = {"fused": 0, "split": 1}
PRECISION = {"f64": 0, "f32": 1}
TIMER_NAMES = ("integrate", "cells", "reorder", "nebr", "force", "energy", "fused_step", "decide")

EXPORTS = ("md_params_default", "md_create", "md_create_ex", "md_destroy", "md_pushoff", "md_set_rigid", "md_set_rigid_state", "md_get_rigid_state", "md_set_bonds", "md_set_angles", "md_set_dihedrals", "md_step", "md_energies",
           "md_get_positions", "md_get_velocities", "md_get_forces", "md_get_state", "md_get_positions_device",
           "md_get_velocities_device", "md_get_forces_device", "md_set_state", "md_set_state_device", "md_stage_state", "md_commit_state", "md_get_state_async", "md_wait_io", "md_measure_peaks",
           "md_rebuild_neighbors",
           "md_get_neighbors", "md_get_info", "md_set_profiling", "md_get_timers", "md_reset_timers",
           "md_set_allocator", "md_velocity_sums_noalloc", "md_last_error", "md_version")


class MDError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"md_b200 error {code}: {msg}")
        self.code = code


class _Params(C.Structure):
    _fields_ = [("n_atoms", C.c_int64), ("box", C.c_double), ("density", C.c_double), ("r_cut", C.c_double),
                ("r_shell", C.c_double), ("dt", C.c_double), ("seed", C.c_uint64), ("temperature", C.c_double),
                ("lattice", C.c_int32), ("force_variant", C.c_int32), ("step_mode", C.c_int32),
                ("max_neighbors", C.c_int32), ("block_size", C.c_int32), ("device", C.c_int32),
                ("stream", C.c_void_p), ("flags", C.c_uint32), ("n_systems", C.c_int32),
                ("precision", C.c_int32), ("reorder_interval", C.c_int32), ("cell_split_x", C.c_int32), ("tile_cells", C.c_int32 * 3),
                ("tile_threads", C.c_int32), ("tile_capacity", C.c_int32)]


class _Energy(C.Structure):
    _fields_ = [("ke", C.c_double), ("pe_pair", C.c_double), ("pe_bond", C.c_double), ("virial", C.c_double),
                ("px", C.c_double), ("py", C.c_double), ("pz", C.c_double), ("vmax", C.c_double),
                ("step", C.c_int64), ("n_rebuilds", C.c_int64),
                ("max_neighbors", C.c_int32), ("max_cell_occupancy", C.c_int32), ("mean_neighbors", C.c_double)]


class _Info(C.Structure):
    _fields_ = [("n_atoms", C.c_int64), ("n_pad", C.c_int64), ("box", C.c_double), ("r_neighbor", C.c_double),
                ("cell_width", C.c_double), ("cells_per_edge", C.c_int32), ("max_neighbors", C.c_int32),
                ("block_size", C.c_int32), ("force_variant", C.c_int32), ("step_mode", C.c_int32),
                ("n_bonds_per_atom_max", C.c_int32), ("device_bytes", C.c_int64), ("kernel_launches", C.c_int64),
                ("device_name", C.c_char * 64), ("w_layout", C.c_int32), ("tile_cells", C.c_int32 * 3),
                ("tile_capacity", C.c_int32), ("tile_threads", C.c_int32), ("use_graph", C.c_int32),
                ("n_systems", C.c_int32), ("precision", C.c_int32), ("n_layers", C.c_int32), ("cells_x", C.c_int32),
                ("cell_split_x", C.c_int32), ("sm_count", C.c_int32), ("candidates_per_atom", C.c_double)]


class _Peaks(C.Structure):
    _fields_ = [("fp64_tflops", C.c_double), ("fp32_tflops", C.c_double), ("sm_count", C.c_int32), ("sm_clock_khz", C.c_int32)]


class _PushoffOpts(C.Structure):
    _fields_ = [("r_cap_start", C.c_double), ("r_cap_end", C.c_double), ("ramp_steps", C.c_int32), ("max_steps", C.c_int32),
                ("check_interval", C.c_int32), ("min_nonbonded", C.c_double), ("max_bond", C.c_double),
                ("max_move", C.c_double), ("temperature", C.c_double), ("seed", C.c_uint64)]


class _PushoffReport(C.Structure):
    _fields_ = [("steps", C.c_int64), ("min_nonbonded", C.c_double), ("max_bond", C.c_double),
                ("min_nonbonded_start", C.c_double)]


@dataclass
class Energies:
    ke: float
    pe_pair: float
    pe_bond: float
    virial: float
    px: float
    py: float
    pz: float
    vmax: float
    step: int
    n_rebuilds: int
    max_neighbors: int
    max_cell_occupancy: int
    mean_neighbors: float

    @property
    def pe(self) -> float:
        return self.pe_pair + self.pe_bond

    @property
    def total(self) -> float:
        return self.ke + self.pe


_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p)
_FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)
_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_ip = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")

_lib = None
_keep = []          # callback objects must outlive the library's use of them


def load_library(path: str = LIB_PATH):
    """dlopen the C-ABI library and declare signatures.  Needs no GPU."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise MDError(MD_ERR_CUDA, f"{path} not built: run `python -m paper_2003_14061_b200.build` "
                                   "(there is no CPU fallback)")
    L = C.CDLL(path)
    L.md_params_default.argtypes = [C.POINTER(_Params)]
    L.md_create.restype = C.c_void_p
    L.md_create.argtypes = [C.c_int64, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double, C.c_uint64]
    L.md_create_ex.restype = C.c_void_p
    L.md_create_ex.argtypes = [C.POINTER(_Params)]
    L.md_destroy.argtypes = [C.c_void_p]
    L.md_set_bonds.argtypes = [C.c_void_p, C.c_int64, _ip, C.c_double, C.c_double]
    L.md_pushoff.argtypes = [C.c_void_p, _dp, C.c_int64, _ip, C.c_double, C.c_double, C.POINTER(_PushoffOpts),
                             C.POINTER(_PushoffReport)]
    L.md_set_rigid.argtypes = [C.c_void_p, C.c_int32, _dp]
    L.md_set_rigid_state.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
    L.md_get_rigid_state.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
    L.md_set_angles.argtypes = [C.c_void_p, C.c_double, C.c_double]
    L.md_set_dihedrals.argtypes = [C.c_void_p, C.c_double, C.c_double]
    L.md_step.argtypes = [C.c_void_p, C.c_int64]
    L.md_energies.argtypes = [C.c_void_p, C.POINTER(_Energy)]
    for n in ("md_get_positions", "md_get_velocities", "md_get_forces"):
        getattr(L, n).argtypes = [C.c_void_p, _dp]
    L.md_set_state.argtypes = [C.c_void_p, _dp, C.c_void_p]
    L.md_get_state.argtypes = [C.c_void_p, _dp, _dp]
    for n in ("md_get_positions_device", "md_get_velocities_device", "md_get_forces_device"):
        getattr(L, n).argtypes = [C.c_void_p, C.c_void_p]
    L.md_set_state_device.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.md_stage_state.argtypes = [C.c_void_p, _dp, _dp]
    L.md_commit_state.argtypes = [C.c_void_p]
    L.md_get_state_async.argtypes = [C.c_void_p, _dp, _dp]
    L.md_wait_io.argtypes = [C.c_void_p, C.c_int32]
    L.md_measure_peaks.argtypes = [C.c_void_p, C.POINTER(_Peaks)]
    L.md_velocity_sums_noalloc.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
    L.md_rebuild_neighbors.argtypes = [C.c_void_p]
    L.md_get_neighbors.argtypes = [C.c_void_p, _ip, C.c_void_p, C.POINTER(C.c_int32)]
    L.md_get_info.argtypes = [C.c_void_p, C.POINTER(_Info)]
    L.md_set_profiling.argtypes = [C.c_void_p, C.c_int]
    L.md_get_timers.argtypes = [C.c_void_p, _dp, np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")]
    L.md_reset_timers.argtypes = [C.c_void_p]
    L.md_set_allocator.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    L.md_last_error.restype = C.c_char_p
    L.md_version.restype = C.c_char_p
    _lib = L
    return L


def use_torch_allocator():
    """Route the library's device allocations to torch's caching allocator."""
    import torch
    L = load_library()

    def _alloc(nbytes, stream, _user):
        try:
            return torch.cuda.caching_allocator_alloc(int(nbytes), stream=int(stream or 0))
        except Exception:
            return None

    def _free(ptr, _user):
        try:
            torch.cuda.caching_allocator_delete(int(ptr))
        except Exception:
            pass

    if not _keep:
        _keep.extend([_ALLOC_FN(_alloc), _FREE_FN(_free)])
    L.md_set_allocator(C.cast(_keep[0], C.c_void_p), C.cast(_keep[1], C.c_void_p), None)


def use_cuda_allocator():
    """Back to cudaMalloc / cudaFree for systems created from now on (existing systems keep the hooks they were created with)."""
    load_library().md_set_allocator(None, None, None)


def _err(L):
    return (L.md_last_error() or b"").decode()


NOALLOC_MAX_ATOMS = 16777216       # MD_NOALLOC_MAX_ATOMS


def velocity_sums_noalloc(v, out=None, stream=None):
    """md_velocity_sums_noalloc: ke, px, py, pz, vmax of a float64 CUDA tensor of velocities (N, 3) into a float64 CUDA
    tensor of 5 elements, on torch's current stream (or `stream`, a cudaStream_t value).  The library allocates nothing;
    pass `out` to make the whole call allocation-free.  Not synchronised.  Calls that overlap on the GPU race."""
    import torch
    L = load_library()
    if out is None:
        out = torch.empty(5, dtype=torch.float64, device=v.device)
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    rc = L.md_velocity_sums_noalloc(C.c_void_p(v.data_ptr()), v.numel() // 3, C.c_void_p(out.data_ptr()), C.c_void_p(stream))
    if rc != MD_OK:
        raise MDError(rc, _err(L))
    return out


class MDSystem:
    """One MD system on one GPU (the handle of md_create_ex)."""

    def __init__(self, n_atoms, r_cut, r_shell, dt, box=0.0, density=0.0, seed=1, temperature=1.0, lattice="auto",
                 force_variant="full", step_mode="fused", max_neighbors=0, block_size=0, device=-1,
                 torch_memory=True, flags=0, n_systems=1, precision="f64", reorder_interval=0,
                 tile_cells=(0, 0, 0), tile_threads=0, tile_capacity=0, cell_split_x=0):
        import torch
        if not torch.cuda.is_available():
            raise MDError(MD_ERR_CUDA, "no CUDA device: the MD path has no CPU fallback")
        L = load_library()
        # the library records the hooks in force at creation inside the handle, so systems of either kind can coexist
        if torch_memory:
            use_torch_allocator()
        else:
            use_cuda_allocator()
        p = _Params()
        L.md_params_default(C.byref(p))
        p.n_atoms, p.box, p.density, p.r_cut, p.r_shell, p.dt = int(n_atoms), box, density, r_cut, r_shell, dt
        p.seed, p.temperature = int(seed), temperature
        p.lattice, p.force_variant, p.step_mode = LATTICE[lattice], FORCE_VARIANT[force_variant], STEP_MODE[step_mode]
        p.max_neighbors, p.block_size, p.device, p.flags = max_neighbors, block_size, device, flags
        p.n_systems = int(n_systems)
        p.precision = PRECISION[precision]
        p.reorder_interval = int(reorder_interval)
        p.tile_cells[0], p.tile_cells[1], p.tile_cells[2] = (int(x) for x in tile_cells)
        p.tile_threads, p.tile_capacity = int(tile_threads), int(tile_capacity)
        p.cell_split_x = int(cell_split_x)
        p.stream = torch.cuda.current_stream().cuda_stream or None
        self._L = L
        self._h = L.md_create_ex(C.byref(p))
        if not self._h:
            raise MDError(MD_ERR_INVALID, _err(L))
        self.n = int(n_atoms) * int(n_systems)          # rows of every per-atom array at the boundary

    @classmethod
    def from_config(cls, cfg, **kw):
        lattice = kw.pop("lattice", cfg.lattice if cfg.lattice in ("sc", "fcc") else "none")
        return cls(cfg.n_atoms, cfg.r_cut, cfg.r_shell, cfg.dt, density=cfg.density, temperature=cfg.temperature,
                   lattice=lattice, **kw)

    def close(self):
        if getattr(self, "_h", None):
            self._L.md_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc):
        if rc != MD_OK:
            raise MDError(rc, _err(self._L))

    def set_state(self, r, v=None):
        r = np.ascontiguousarray(r, np.float64)
        vp = None
        if v is not None:
            v = np.ascontiguousarray(v, np.float64)
            vp = v.ctypes.data_as(C.c_void_p)
        self._ck(self._L.md_set_state(self._h, r, vp))

    def set_bonds(self, bonds, k, r0):
        b = np.ascontiguousarray(bonds, np.int32).reshape(-1, 2)
        self._ck(self._L.md_set_bonds(self._h, b.shape[0], b, float(k), float(r0)))

    def pushoff(self, r, bonds, k, r0, temperature=1.0, seed=1, **opts) -> dict:
        """md_pushoff: push an overlapping chain start apart inside the library and load the result (fresh velocities,
        bonds) into this system.  opts: fields of md_pushoff_opts.  Returns the report as a dict."""
        r = np.ascontiguousarray(r, np.float64)
        b = np.ascontiguousarray(bonds, np.int32).reshape(-1, 2)
        o = _PushoffOpts()
        o.temperature, o.seed = float(temperature), int(seed)
        for key, val in opts.items():
            setattr(o, key, val)
        rep = _PushoffReport()
        self._ck(self._L.md_pushoff(self._h, r, b.shape[0], b, float(k), float(r0), C.byref(o), C.byref(rep)))
        return {key: getattr(rep, key) for key, _ in _PushoffReport._fields_}

    def set_rigid(self, body):
        """md_set_rigid: the atoms become the sites of rigid molecules of len(body) sites (body: (n_sites, 3), principal frame)."""
        b = np.ascontiguousarray(body, np.float64).reshape(-1, 3)
        self._ck(self._L.md_set_rigid(self._h, b.shape[0], b))
        self._n_sites = b.shape[0]

    def set_rigid_state(self, com, rot, vcom, angmom_body):
        nm = self.n // self._n_sites
        a = [np.ascontiguousarray(x, np.float64).reshape(nm, k) for x, k in ((com, 3), (rot, 9), (vcom, 3), (angmom_body, 3))]
        self._ck(self._L.md_set_rigid_state(self._h, *a))

    def rigid_state(self):
        nm = self.n // self._n_sites
        R, A, V, pi = np.empty((nm, 3)), np.empty((nm, 9)), np.empty((nm, 3)), np.empty((nm, 3))
        self._ck(self._L.md_get_rigid_state(self._h, R, A, V, pi))
        return R, A.reshape(nm, 3, 3), V, pi

    def set_angles(self, k_theta, cos_theta0):
        self._ck(self._L.md_set_angles(self._h, float(k_theta), float(cos_theta0)))

    def set_dihedrals(self, k_phi, cos_phi0):
        self._ck(self._L.md_set_dihedrals(self._h, float(k_phi), float(cos_phi0)))

    def step(self, n=1):
        self._ck(self._L.md_step(self._h, int(n)))

    def rebuild_neighbors(self):
        self._ck(self._L.md_rebuild_neighbors(self._h))

    def energies(self) -> Energies:
        e = _Energy()
        self._ck(self._L.md_energies(self._h, C.byref(e)))
        return Energies(**{k: getattr(e, k) for k, _ in _Energy._fields_})

    def _get(self, name, out=None):
        if out is None:
            out = np.empty((self.n, 3))
        self._ck(getattr(self._L, name)(self._h, out))
        return out

    def positions(self, out=None):
        return self._get("md_get_positions", out)

    def velocities(self, out=None):
        return self._get("md_get_velocities", out)

    def forces(self, out=None):
        return self._get("md_get_forces", out)

    def state(self, r_out=None, v_out=None):
        """md_get_state: positions and velocities with one synchronisation.  Pass the two halves of ONE page-locked
        (2, N, 3) array to get a single device-to-host transfer."""
        if r_out is None or v_out is None:
            both = np.empty((2, self.n, 3))
            r_out, v_out = both[0], both[1]
        self._ck(self._L.md_get_state(self._h, r_out, v_out))
        return r_out, v_out

    def _device_out(self, name, out):
        import torch
        if out is None:
            out = torch.empty((self.n, 3), dtype=torch.float64, device="cuda")
        if not (out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == 3 * self.n):
            raise MDError(MD_ERR_INVALID, "need a contiguous float64 CUDA tensor of 3 N elements")
        self._ck(getattr(self._L, name)(self._h, C.c_void_p(out.data_ptr())))
        return out

    def positions_device(self, out=None):
        """Zero-copy read-out into a torch CUDA tensor (N, 3), original-id order; enqueued on the system's stream."""
        return self._device_out("md_get_positions_device", out)

    def velocities_device(self, out=None):
        return self._device_out("md_get_velocities_device", out)

    def forces_device(self, out=None):
        return self._device_out("md_get_forces_device", out)

    def set_state_device(self, r, v=None):
        """md_set_state from torch CUDA tensors (float64, contiguous): no host transfer."""
        import torch
        for t in (r, v):
            if t is not None and not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == 3 * self.n):
                raise MDError(MD_ERR_INVALID, "need contiguous float64 CUDA tensors of 3 N elements")
        self._ck(self._L.md_set_state_device(self._h, C.c_void_p(r.data_ptr()), C.c_void_p(v.data_ptr()) if v is not None else None))

    # double-buffered host I/O on the library's copy streams; all arrays page-locked float64 (N, 3), kept alive and
    # untouched by the caller until wait_io() (or, for a staged state, commit_state()) has returned
    def stage_state(self, r, v):
        """md_stage_state: start the upload of a next state; returns at once.  Up to two states can be staged (FIFO)."""
        self._ck(self._L.md_stage_state(self._h, r, v))

    def commit_state(self):
        """md_commit_state: install the oldest staged state as md_set_state would."""
        self._ck(self._L.md_commit_state(self._h))

    def state_async(self, r_out, v_out):
        """md_get_state_async: start the download of the current state; complete after wait_io()."""
        self._ck(self._L.md_get_state_async(self._h, r_out, v_out))

    def wait_io(self, max_pending=0):
        """md_wait_io: 0 = every transfer complete; 1..3 = all but that many of the newest downloads."""
        self._ck(self._L.md_wait_io(self._h, int(max_pending)))

    def measure_peaks(self) -> dict:
        p = _Peaks()
        self._ck(self._L.md_measure_peaks(self._h, C.byref(p)))
        return {k: getattr(p, k) for k, _ in _Peaks._fields_}

    def neighbors(self, with_list=True):
        """(counts[N], list[N, Mmax] of original ids, -1 padded)."""
        info = self.info()
        counts = np.empty(self.n, np.int32)
        lst = np.empty((self.n, info["max_neighbors"]), np.int32) if with_list else None
        mm = C.c_int32(0)
        self._ck(self._L.md_get_neighbors(self._h, counts, lst.ctypes.data_as(C.c_void_p) if with_list else None,
                                          C.byref(mm)))
        return counts, lst

    def neighbor_sets(self):
        counts, lst = self.neighbors()
        return [np.sort(lst[i, :counts[i]]) for i in range(self.n)]

    def info(self) -> dict:
        i = _Info()
        self._ck(self._L.md_get_info(self._h, C.byref(i)))
        d = {k: getattr(i, k) for k, _ in _Info._fields_}
        d["device_name"] = d["device_name"].decode()
        d["tile_cells"] = list(d["tile_cells"])

        return d

    def set_profiling(self, on: bool):
        self._ck(self._L.md_set_profiling(self._h, int(bool(on))))

    def reset_timers(self):
        self._ck(self._L.md_reset_timers(self._h))

    def timers(self) -> dict:
        ms = np.zeros(8)
        n = np.zeros(8, np.int64)
        self._ck(self._L.md_get_timers(self._h, ms, n))
        return {name: {"ms": float(ms[k]), "launches": int(n[k])} for k, name in enumerate(TIMER_NAMES) if name != "reserved"}
