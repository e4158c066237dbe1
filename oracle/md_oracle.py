"""ctypes front end of the CPU oracles (oracle/md_oracle.c, fp64; oracle/md_oracle_sp.c, the single-precision
variant of SURVEY.md 8(f) NEXT-1).  TEST INFRASTRUCTURE ONLY.

Imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` legs -- never by the product package.  Shares nothing with
paper_2003_14061_b200/.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "md_oracle.c")
_LIB = os.path.join(_HERE, "libmd_oracle.so")
_SRC_SP = os.path.join(_HERE, "md_oracle_sp.c")
_LIB_SP = os.path.join(_HERE, "libmd_oracle_sp.so")
_SRC_RIGID = os.path.join(_HERE, "md_oracle_rigid.c")
_LIB_RIGID = os.path.join(_HERE, "libmd_oracle_rigid.so")


def build(force: bool = False) -> str:
    """gcc -O2 build of the oracle (fp contraction off: every a*b+c rounds twice unless written fma())."""
    for src, out in ((_SRC, _LIB), (_SRC_SP, _LIB_SP), (_SRC_RIGID, _LIB_RIGID)):
        if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
            cmd = ["gcc", "-std=c11", "-O2", "-march=native", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
                   "-fPIC", "-shared", "-o", out, src, "-lm"]
            subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


class _Energy(C.Structure):
    _fields_ = [("ke", C.c_double), ("pe_pair", C.c_double), ("pe_bond", C.c_double), ("virial", C.c_double),
                ("px", C.c_double), ("py", C.c_double), ("pz", C.c_double), ("vmax", C.c_double),
                ("step", C.c_int64), ("n_rebuilds", C.c_int64),
                ("max_neighbors", C.c_int32), ("max_cell_occupancy", C.c_int32),
                ("mean_neighbors", C.c_double)]


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


_lib = None
_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_ip = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_lp = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")


class _Prefixed:
    """The functions of one oracle library under prefix-free names (orc_* / orcs_* share one signature set)."""

    def __init__(self, L, prefix):
        self._L, self._p = L, prefix

    def __getattr__(self, name):
        return getattr(self._L, self._p + name)


def _declare_system_api(L, p):
    f = lambda n: getattr(L, p + n)
    f("create").restype = C.c_void_p
    f("create").argtypes = [C.c_int64, C.c_double, C.c_double, C.c_double, C.c_double]
    f("destroy").argtypes = [C.c_void_p]
    f("force_brute_search").argtypes = [C.c_void_p, C.c_int]
    f("set_state").argtypes = [C.c_void_p, _dp, C.c_void_p]
    f("set_bonds").argtypes = [C.c_void_p, C.c_int64, _ip, C.c_double, C.c_double]
    f("set_bonds").restype = C.c_int
    f("rebuild_neighbors").argtypes = [C.c_void_p]
    f("step").argtypes = [C.c_void_p, C.c_int64]
    f("step").restype = C.c_int
    f("energies").argtypes = [C.c_void_p, C.POINTER(_Energy)]
    for name in ("get_positions", "get_velocities", "get_forces", "set_velocities"):
        f(name).argtypes = [C.c_void_p, _dp]
    f("get_atom_energies").argtypes = [C.c_void_p, _dp, _dp]
    f("neighbor_total").argtypes = [C.c_void_p]
    f("neighbor_total").restype = C.c_int64
    f("get_neighbors").argtypes = [C.c_void_p, _ip, _ip]
    f("set_threads").argtypes = [C.c_int]
    f("get_threads").restype = C.c_int


_lib_sp = None


def lib_sp():
    global _lib_sp
    if _lib_sp is None:
        build()
        L = C.CDLL(_LIB_SP)
        _declare_system_api(L, "orcs_")
        L.orcs_set_angles.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.orcs_set_angles.restype = C.c_int
        L.orcs_set_dihedrals.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.orcs_set_dihedrals.restype = C.c_int
        _lib_sp = L
    return _lib_sp


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        _declare_system_api(L, "orc_")
        L.orc_set_angles.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.orc_set_angles.restype = C.c_int
        L.orc_set_dihedrals.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.orc_set_dihedrals.restype = C.c_int
        L.orc_brute_forces.argtypes = [C.c_int64, C.c_double, _dp, C.c_double, _dp, _dp, _dp]
        L.orc_brute_forces_sample.argtypes = [C.c_int64, C.c_double, _dp, C.c_double, C.c_int64, _lp, _dp, _dp, _dp]
        L.orc_brute_neighbors_sample.argtypes = [C.c_int64, C.c_double, _dp, C.c_double, C.c_int64, _lp,
                                                 C.c_int32, _ip, _ip]
        L.orc_brute_neighbors_sample.restype = C.c_int32
        _lib = L
    return _lib


def set_threads(n: int) -> None:
    lib().orc_set_threads(int(n))
    lib_sp().orcs_set_threads(int(n))


def get_threads() -> int:
    return int(lib().orc_get_threads())


def _c(a, dtype=np.float64):
    return np.ascontiguousarray(a, dtype=dtype)


def brute_forces(r, box, r_cut):
    """All-pairs minimum-image truncated LJ: (f[N,3], u[N], w[N]); u, w double counted per atom."""
    r = _c(r)
    n = r.shape[0]
    f, u, w = np.empty((n, 3)), np.empty(n), np.empty(n)
    lib().orc_brute_forces(n, float(box), r, float(r_cut), f, u, w)
    return f, u, w


def brute_forces_sample(r, box, r_cut, idx):
    r, idx = _c(r), _c(idx, np.int64)
    ns = idx.shape[0]
    f, u, w = np.empty((ns, 3)), np.empty(ns), np.empty(ns)
    lib().orc_brute_forces_sample(r.shape[0], float(box), r, float(r_cut), ns, idx, f, u, w)
    return f, u, w


def brute_neighbors_sample(r, box, r_n, idx, cap=256):
    """Neighbor sets by definition for the atoms in idx: list of sorted int arrays."""
    r, idx = _c(r), _c(idx, np.int64)
    ns = idx.shape[0]
    counts = np.empty(ns, np.int32)
    out = np.empty((ns, cap), np.int32)
    mx = lib().orc_brute_neighbors_sample(r.shape[0], float(box), r, float(r_n), ns, idx, cap, counts, out)
    if mx > cap:
        return brute_neighbors_sample(r, box, r_n, idx, cap=int(mx))
    return [out[k, :counts[k]].copy() for k in range(ns)]


class OracleMD:
    """Plain CPU MD of the same model (see md_oracle.c header for the passages followed)."""

    _prefix = "orc_"

    def _load(self):
        return lib()

    def __init__(self, n_atoms, box, r_cut, r_shell, dt, brute_search=False):
        self._L = _Prefixed(self._load(), self._prefix)
        self.n = int(n_atoms)
        self.box, self.r_cut, self.r_shell, self.dt = float(box), float(r_cut), float(r_shell), float(dt)
        self._h = self._L.create(self.n, self.box, self.r_cut, self.r_shell, self.dt)
        if not self._h:
            raise ValueError("orc_create failed")
        if brute_search:
            self._L.force_brute_search(self._h, 1)

    def close(self):
        if self._h:
            self._L.destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_state(self, r, v=None):
        r = _c(r)
        assert r.shape == (self.n, 3)
        vp = None
        if v is not None:
            v = _c(v)
            vp = v.ctypes.data_as(C.c_void_p)
        self._L.set_state(self._h, r, vp)

    def set_velocities(self, v):
        self._L.set_velocities(self._h, _c(v))

    def set_bonds(self, bonds, k, r0):
        b = _c(bonds, np.int32).reshape(-1, 2)
        return self._L.set_bonds(self._h, b.shape[0], b, float(k), float(r0))

    def set_angles(self, k, cos0):
        """Cosine-harmonic bond-angle terms; after set_bonds."""
        return self._L.set_angles(self._h, float(k), float(cos0))

    def set_dihedrals(self, k, cos0):
        """Cosine-harmonic dihedral terms; after set_bonds."""
        return self._L.set_dihedrals(self._h, float(k), float(cos0))

    def rebuild_neighbors(self):
        self._L.rebuild_neighbors(self._h)

    def step(self, n=1):
        return self._L.step(self._h, int(n))

    def energies(self) -> Energies:
        e = _Energy()
        self._L.energies(self._h, C.byref(e))
        return Energies(**{k: getattr(e, k) for k, _ in _Energy._fields_})

    def _get(self, name):
        out = np.empty((self.n, 3))
        getattr(self._L, name)(self._h, out)
        return out

    def positions(self):
        return self._get("get_positions")

    def velocities(self):
        return self._get("get_velocities")

    def forces(self):
        return self._get("get_forces")

    def atom_energies(self):
        u, w = np.empty(self.n), np.empty(self.n)
        self._L.get_atom_energies(self._h, u, w)
        return u, w

    def neighbors(self):
        """(counts[N], flat list in CSR order)."""
        tot = self._L.neighbor_total(self._h)
        counts = np.empty(self.n, np.int32)
        flat = np.empty(max(tot, 1), np.int32)
        self._L.get_neighbors(self._h, counts, flat)
        return counts, flat[:tot]

    def neighbor_sets(self):
        counts, flat = self.neighbors()
        off = np.concatenate([[0], np.cumsum(counts, dtype=np.int64)])
        return [np.sort(flat[off[i]:off[i + 1]]) for i in range(self.n)]


class OracleMDSP(OracleMD):
    """The single-precision variant (md_oracle_sp.c): binary32 state and pair arithmetic, binary64 energy sums.
    Same interface; boundary arrays are float64 holding binary32 values."""
    _prefix = "orcs_"

    def _load(self):
        return lib_sp()


# ---- rigid molecules (oracle/md_oracle_rigid.c; R20) ----------------------------------------------------
class _RigidEnergy(C.Structure):
    _fields_ = [("ke_trans", C.c_double), ("ke_rot", C.c_double), ("pe", C.c_double), ("virial", C.c_double),
                ("px", C.c_double), ("py", C.c_double), ("pz", C.c_double), ("vbound", C.c_double),
                ("lx", C.c_double), ("ly", C.c_double), ("lz", C.c_double),
                ("step", C.c_int64), ("n_rebuilds", C.c_int64), ("max_neighbors", C.c_int32), ("mean_neighbors", C.c_double)]


@dataclass
class RigidEnergies:
    ke_trans: float
    ke_rot: float
    pe: float
    virial: float
    px: float
    py: float
    pz: float
    vbound: float
    lx: float
    ly: float
    lz: float
    step: int
    n_rebuilds: int
    max_neighbors: int
    mean_neighbors: float

    @property
    def ke(self) -> float:
        return self.ke_trans + self.ke_rot

    @property
    def total(self) -> float:
        return self.ke_trans + self.ke_rot + self.pe


_lib_rigid = None


def lib_rigid():
    global _lib_rigid
    if _lib_rigid is None:
        build()
        L = C.CDLL(_LIB_RIGID)
        L.orr_create.restype = C.c_void_p
        L.orr_create.argtypes = [C.c_int64, C.c_int, _dp, C.c_double, C.c_double, C.c_double, C.c_double]
        L.orr_destroy.argtypes = [C.c_void_p]
        L.orr_set_state.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
        L.orr_get_state.argtypes = [C.c_void_p, _dp, _dp, _dp, _dp]
        L.orr_step.argtypes = [C.c_void_p, C.c_int64]
        L.orr_step.restype = C.c_int
        L.orr_energies.argtypes = [C.c_void_p, C.POINTER(_RigidEnergy)]
        for name in ("orr_get_sites", "orr_get_site_forces", "orr_get_inertia"):
            getattr(L, name).argtypes = [C.c_void_p, _dp]
        L.orr_get_force_torque.argtypes = [C.c_void_p, _dp, _dp]
        L.orr_neighbor_total.argtypes = [C.c_void_p]
        L.orr_neighbor_total.restype = C.c_int64
        L.orr_get_neighbors.argtypes = [C.c_void_p, _ip, _ip]
        _lib_rigid = L
    return _lib_rigid


class OracleRigid:
    """Rigid molecules of n_sites unit-mass sites each (md_oracle_rigid.c header for the model and its sources)."""

    def __init__(self, n_mol, body, box, r_cut, r_shell, dt):
        self._L = lib_rigid()
        body = _c(body).reshape(-1, 3)
        self.nm, self.ns = int(n_mol), body.shape[0]
        self._h = self._L.orr_create(self.nm, self.ns, body, float(box), float(r_cut), float(r_shell), float(dt))
        if not self._h:
            raise ValueError("orr_create failed: body frame must be the principal frame about the centre of mass, moments > 0")

    def close(self):
        if self._h:
            self._L.orr_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_state(self, R, A, V, pi):
        self._L.orr_set_state(self._h, _c(R), _c(A).reshape(self.nm, 9), _c(V), _c(pi))

    def state(self):
        R, A, V, pi = np.empty((self.nm, 3)), np.empty((self.nm, 9)), np.empty((self.nm, 3)), np.empty((self.nm, 3))
        self._L.orr_get_state(self._h, R, A, V, pi)
        return R, A.reshape(self.nm, 3, 3), V, pi

    def step(self, n=1):
        return self._L.orr_step(self._h, int(n))

    def energies(self) -> RigidEnergies:
        e = _RigidEnergy()
        self._L.orr_energies(self._h, C.byref(e))
        return RigidEnergies(**{k: getattr(e, k) for k, _ in _RigidEnergy._fields_})

    def sites(self):
        out = np.empty((self.nm * self.ns, 3))
        self._L.orr_get_sites(self._h, out)
        return out

    def site_forces(self):
        out = np.empty((self.nm * self.ns, 3))
        self._L.orr_get_site_forces(self._h, out)
        return out

    def force_torque(self):
        F, T = np.empty((self.nm, 3)), np.empty((self.nm, 3))
        self._L.orr_get_force_torque(self._h, F, T)
        return F, T

    def inertia(self):
        out = np.empty(3)
        self._L.orr_get_inertia(self._h, out)
        return out

    def neighbors(self):
        tot = self._L.orr_neighbor_total(self._h)
        counts = np.empty(self.nm * self.ns, np.int32)
        flat = np.empty(max(tot, 1), np.int32)
        self._L.orr_get_neighbors(self._h, counts, flat)
        return counts, flat[:tot]
