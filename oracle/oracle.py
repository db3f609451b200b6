"""ctypes front end of the fp64 CPU oracle (oracle/sph_oracle.c).

TEST INFRASTRUCTURE ONLY.  Importers allowed: tests/, __graft_entry__.smoke(), and bench.py's
cpu_baseline / --impl reference legs.  Nothing here imports, links or calls the CUDA path
(paper_2512_09904_b200); the two share only the input generators.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sph_oracle.c")
_LIB = os.path.join(_HERE, "libsph_oracle.so")
MAX_BODIES = 8

FIELDS = {
    "POS": 0, "VEL": 1, "RHO": 2, "P": 3, "T": 4, "ACC": 5, "DRHO_DT": 6, "DT_DT": 7,
    "ACC_P": 8, "ACC_V": 9, "ACC_WP": 10, "ACC_WV": 11, "WALL_POS": 12, "WALL_NORMAL": 13,
    "WALL_FORCE": 14, "DRHO_SAVED": 15, "WALL_T": 16, "WALL_DT_DT": 17,
}
_VEC_FIELDS = {"POS", "VEL", "ACC", "ACC_P", "ACC_V", "ACC_WP", "ACC_WV", "WALL_POS", "WALL_NORMAL",
               "WALL_FORCE"}
_WALL_FIELDS = {"WALL_POS", "WALL_NORMAL", "WALL_FORCE", "WALL_T", "WALL_DT_DT"}


class OrcParams(C.Structure):
    _fields_ = [
        ("flags", C.c_uint32), ("rebuild_every", C.c_int32), ("n_bodies", C.c_int32),
        ("neigh_backend", C.c_int32),
        ("dx", C.c_double), ("h", C.c_double), ("rho0", C.c_double), ("c0", C.c_double),
        ("nu", C.c_double), ("g", C.c_double * 3), ("k_f", C.c_double), ("cp_f", C.c_double),
        ("cfl_ac", C.c_double), ("cfl_ad", C.c_double), ("u_ref", C.c_double),
        ("dt_fixed", C.c_double), ("domain_min", C.c_double * 3), ("domain_max", C.c_double * 3),
        ("body_k", C.c_double * MAX_BODIES),
        ("body_rho", C.c_double * MAX_BODIES), ("body_cp", C.c_double * MAX_BODIES),
        ("body_mode", C.c_int32 * MAX_BODIES),
        ("dim", C.c_int32),
        ("fs_threshold", C.c_double),
    ]


def build(force: bool = False) -> str:
    """compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-Wall",
               _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(OrcParams)]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_load.argtypes = [C.c_void_p, C.c_int64] + [C.c_void_p] * 4 + [C.c_int64] + [C.c_void_p] * 4
        L.orc_set_materials.argtypes = [C.c_void_p] + [C.c_void_p] * 3
        L.orc_set_state.argtypes = [C.c_void_p] + [C.c_void_p] * 5
        L.orc_set_kinematics.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_double]
        L.orc_set_time.argtypes = [C.c_void_p, C.c_double]
        L.orc_keep_config.argtypes = [C.c_void_p]
        L.orc_relax.restype = C.c_double
        L.orc_relax.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.orc_step.argtypes = [C.c_void_p, C.c_int]
        L.orc_rebuild.argtypes = [C.c_void_p]
        L.orc_eval_rates.argtypes = [C.c_void_p]
        L.orc_get_f64.restype = C.c_int64
        L.orc_get_f64.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.orc_get_cells.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_get_neigh.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_get_fs_region.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_get_csr.restype = C.c_int64
        L.orc_get_csr.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.orc_contact_factor.argtypes = [C.c_void_p, C.c_void_p]
        L.orc_get_torque.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_get_stats.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.orc_grid_dims.argtypes = [C.POINTER(OrcParams), C.POINTER(C.c_int)]
        for f in ("orc_W", "orc_dWdr", "orc_W2d", "orc_dWdr2d", "orc_sigma0_2d"):
            getattr(L, f).restype = C.c_double
            getattr(L, f).argtypes = [C.c_double, C.c_double]
        L.orc_sigma0.restype = C.c_double
        L.orc_sigma0.argtypes = [C.c_double, C.c_double]
        L.orc_riemann.argtypes = [C.c_double] * 7 + [C.POINTER(C.c_double)] * 3
        L.orc_dt_ad.restype = C.c_double
        L.orc_dt_ad.argtypes = [C.c_double] * 4
        L.orc_dt_ac.restype = C.c_double
        L.orc_dt_ac.argtypes = [C.c_double] * 4
        L.orc_dt_thermal.restype = C.c_double
        L.orc_dt_thermal.argtypes = [C.c_double] * 4
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def W(r: float, h: float) -> float:
    return lib().orc_W(r, h)


def dWdr(r: float, h: float) -> float:
    return lib().orc_dWdr(r, h)


def W2d(r: float, h: float) -> float:
    return float(lib().orc_W2d(float(r), float(h)))


def dWdr2d(r: float, h: float) -> float:
    return float(lib().orc_dWdr2d(float(r), float(h)))


def sigma0_2d(dx: float, h: float) -> float:
    return float(lib().orc_sigma0_2d(float(dx), float(h)))


def sigma0(dx: float, h: float) -> float:
    return lib().orc_sigma0(dx, h)


def riemann(rhoL, UL, pL, rhoR, UR, pR, c0):
    us, ps, ub = C.c_double(), C.c_double(), C.c_double()
    lib().orc_riemann(rhoL, UL, pL, rhoR, UR, pR, c0, C.byref(us), C.byref(ps), C.byref(ub))
    return us.value, ps.value, ub.value


def dt_ad(h, vmax, nu, cfl=0.25):
    return lib().orc_dt_ad(h, vmax, nu, cfl)


def dt_ac(h, c0, vmax, cfl=0.6):
    return lib().orc_dt_ac(h, c0, vmax, cfl)


def dt_thermal(rho, cp, h, k):
    return lib().orc_dt_thermal(rho, cp, h, k)


def num_threads() -> int:
    return lib().orc_num_threads()


def _params_struct(params: Dict[str, object], body_k, neigh_backend: int, bodies=None) -> OrcParams:
    p = OrcParams()
    p.flags = int(params["flags"])
    p.rebuild_every = int(params.get("rebuild_every", 0))
    p.n_bodies = len(body_k)
    p.neigh_backend = int(neigh_backend)
    for name in ("dx", "h", "rho0", "c0", "nu", "k_f", "cp_f", "cfl_ac", "cfl_ad", "u_ref", "dt_fixed"):
        setattr(p, name, float(params[name]))
    for d in range(3):
        p.g[d] = float(params["g"][d])
        p.domain_min[d] = float(params["domain_min"][d])
        p.domain_max[d] = float(params["domain_max"][d])
    for b, k in enumerate(body_k):
        p.body_k[b] = float(k)
    p.dim = int(params.get("dim", 3))
    p.fs_threshold = float(params.get("fs_threshold", 0.0))
    for b, body in enumerate(bodies or []):
        p.body_rho[b] = float(getattr(body, "rho_s", 0.0))
        p.body_cp[b] = float(getattr(body, "cp_s", 0.0))
        p.body_mode[b] = int(getattr(body, "thermal_mode", 0))
    return p


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Oracle:
    """one oracle simulation; mirrors the six calls of the C ABI (create, load, kinematics,
    step, fields, torque) plus the read-outs the pins need."""

    def __init__(self, params: Dict[str, object], bodies=None, neigh_backend: int = 0):
        body_k = [b.k_s for b in bodies] if bodies else [0.0]
        self._p = _params_struct(params, body_k, neigh_backend, bodies)
        self._h = lib().orc_create(C.byref(self._p))
        self.n_f = self.n_w = 0
        if bodies:
            for b, body in enumerate(bodies):
                self.set_gear_kinematics(b, body.origin, body.axis, body.omega)

    @classmethod
    def from_workload(cls, wl, neigh_backend: int = 0, **param_over) -> "Oracle":
        params = dict(wl.params)
        params.update(param_over)
        o = cls(params, wl.bodies, neigh_backend)
        o.load_particles(wl.pos_f, wl.vel_f, wl.rho_f, wl.T_f, wl.pos_w, wl.normal_w, wl.body_w, wl.T_w)
        return o

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def grid_dims(self):
        n = (C.c_int * 3)()
        lib().orc_grid_dims(C.byref(self._p), n)
        return tuple(n)

    def load_particles(self, pos_f, vel_f, rho_f, T_f, pos_w=None, normal_w=None, body_w=None, T_w=None):
        f32 = lambda a: None if a is None else np.ascontiguousarray(a, np.float32)
        pos_f, vel_f, rho_f, T_f = f32(pos_f), f32(vel_f), f32(rho_f), f32(T_f)
        pos_w = np.zeros((0, 3), np.float32) if pos_w is None else f32(pos_w)
        normal_w = np.zeros((0, 3), np.float32) if normal_w is None else f32(normal_w)
        body_w = np.zeros(len(pos_w), np.int32) if body_w is None else np.ascontiguousarray(body_w, np.int32)
        T_w = np.zeros(len(pos_w), np.float32) if T_w is None else f32(T_w)
        self.n_f, self.n_w = len(pos_f), len(pos_w)
        rc = lib().orc_load(self._h, self.n_f, _ptr(pos_f), _ptr(vel_f), _ptr(rho_f), _ptr(T_f),
                            self.n_w, _ptr(pos_w), _ptr(normal_w), _ptr(body_w), _ptr(T_w))
        assert rc == 0
        return rc

    def set_materials(self, mass=None, k=None, cp=None):
        f64 = lambda a: None if a is None else np.ascontiguousarray(a, np.float64)
        mass, k, cp = f64(mass), f64(k), f64(cp)
        lib().orc_set_materials(self._h, _ptr(mass), _ptr(k), _ptr(cp))

    def set_state(self, r=None, v=None, rho=None, T=None, drho_saved=None):
        f64 = lambda a: None if a is None else np.ascontiguousarray(a, np.float64)
        a = [f64(x) for x in (r, v, rho, T, drho_saved)]
        lib().orc_set_state(self._h, *[_ptr(x) for x in a])

    def keep_config(self) -> None:
        """after set_state between two rebuilds: keep the configuration and the held viscous sums (R26) of the last rebuild."""
        assert lib().orc_keep_config(self._h) == 0

    def set_time(self, t: float) -> None:
        """move the clock to t (the bodies follow at the next rebuild); used with set_state for shared-state steps."""
        lib().orc_set_time(self._h, float(t))

    def set_gear_kinematics(self, body, origin, axis, omega):
        o = (C.c_double * 3)(*[float(x) for x in origin])
        a = (C.c_double * 3)(*[float(x) for x in axis])
        rc = lib().orc_set_kinematics(self._h, int(body), o, a, float(omega))
        assert rc == 0

    def relax(self, n: int, p0: float) -> float:
        """n steps of the background-pressure particle relaxation (Eq. 6-9; reading R24)."""
        return float(lib().orc_relax(self._h, int(n), float(p0)))

    def step(self, n: int = 1) -> int:
        return lib().orc_step(self._h, int(n))

    def rebuild(self) -> int:
        return lib().orc_rebuild(self._h)

    def eval_rates(self) -> int:
        return lib().orc_eval_rates(self._h)

    def get(self, name: str) -> np.ndarray:
        n = self.n_w if name in _WALL_FIELDS else self.n_f
        shape = (n, 3) if name in _VEC_FIELDS else (n,)
        out = np.zeros(shape, np.float64)
        got = lib().orc_get_f64(self._h, FIELDS[name], _ptr(out))
        assert got == out.size, (name, got, out.size)
        return out

    def cells(self):
        cf = np.zeros((self.n_f, 3), np.int32)
        cw = np.zeros((self.n_w, 3), np.int32)
        lib().orc_get_cells(self._h, _ptr(cf), _ptr(cw))
        return cf, cw

    def neigh(self):
        cff = np.zeros(self.n_f, np.uint32)
        cfw = np.zeros(self.n_f, np.uint32)
        dg = np.zeros(self.n_f, np.uint64)
        lib().orc_get_neigh(self._h, _ptr(cff), _ptr(cfw), _ptr(dg))
        return cff, cfw, dg

    def fs_region(self) -> np.ndarray:
        """1 where the last density re-initialisation took the max form of Eq. 14 (free-surface region, R27 / R12), else 0."""
        out = np.zeros(max(self.n_f, 1), np.uint8)
        lib().orc_get_fs_region(self._h, _ptr(out))
        return out[:self.n_f]

    def csr(self, which: int = 0):
        start = np.zeros(self.n_f + 1, np.int64)
        total = lib().orc_get_csr(self._h, which, _ptr(start), None)
        idx = np.zeros(max(int(total), 1), np.int32)
        lib().orc_get_csr(self._h, which, _ptr(start), _ptr(idx))
        return start, idx[: int(total)]

    def contact_factor(self) -> np.ndarray:
        """zeta_C of every wall particle (Eq. 24; reading R22), original wall order."""
        out = np.zeros(max(self.n_w, 1), np.float64)
        rc = lib().orc_contact_factor(self._h, out.ctypes.data_as(C.c_void_p))
        if rc != 0:
            raise RuntimeError("contact_factor needs a neighbour configuration (rebuild or step first)")
        return out[:self.n_w]

    def torque(self, body: int):
        t = (C.c_double * 3)()
        ax = C.c_double()
        lib().orc_get_torque(self._h, int(body), t, C.byref(ax))
        return np.array(list(t)), ax.value

    def stats(self) -> Dict[str, float]:
        s = (C.c_double * 8)()
        lib().orc_get_stats(self._h, s)
        keys = ("t", "dt", "dt_ad", "elapsed", "vmax", "steps", "rebuilds", "sigma0")
        return dict(zip(keys, list(s)))
