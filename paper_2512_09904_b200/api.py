"""Thin ctypes binding of libsph_b200.so (include/sph.h): argument marshalling only.

The functions carry the names of the C ABI (sph_create, sph_load_particles,
sph_set_gear_kinematics, sph_step, sph_get_fields, sph_get_torque, ...) and every step of the
path runs in the CUDA kernels behind them.  There is no CPU fallback: if the shared library is
missing or no CUDA device is present, the calls raise.  PyTorch is used by callers for device
memory and streams only (a tensor's `data_ptr()` may be handed in with SPH_MEM_DEVICE).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsph_b200.so")

SPH_MAX_BODIES = 8
SPH_OK, SPH_EINVAL, SPH_ENOMEM, SPH_ECUDA, SPH_EDOMAIN, SPH_ENAN, SPH_ESTATE, SPH_ENEIGH = 0, -1, -2, -3, -4, -5, -6, -7
SPH_MEM_HOST, SPH_MEM_DEVICE = 0, 1

# enum sph_field
FIELDS = {
    "POS": 0, "VEL": 1, "RHO": 2, "P": 3, "T": 4, "ACC": 5, "DRHO_DT": 6, "DT_DT": 7, "CELL": 8,
    "NEIGH_COUNT": 9, "NEIGH_DIGEST": 10, "DRHO": 11, "WALL_POS": 12, "WALL_NORMAL": 13, "STATS": 14,
    "NEIGH_CSR_FLUID": 15, "NEIGH_CSR_WALL": 16, "DRHO_SAVED": 17, "THETA": 18, "CONTACT_FACTOR": 19, "WALL_T": 20, "WALL_DT_DT": 21, "FS_REGION": 22,
    "SORT_CELL_COUNT": 23, "SORT_CELL_START": 24,
}
# numpy dtype and trailing shape of each field
_FIELD_LAYOUT = {
    "POS": (np.float32, (3,)), "VEL": (np.float32, (3,)), "RHO": (np.float32, ()), "P": (np.float32, ()),
    "T": (np.float32, ()), "ACC": (np.float32, (3,)), "DRHO_DT": (np.float32, ()), "DT_DT": (np.float32, ()),
    "CELL": (np.int32, (3,)), "NEIGH_COUNT": (np.uint32, (2,)), "NEIGH_DIGEST": (np.uint64, ()),
    "DRHO": (np.float32, ()), "WALL_POS": (np.float32, (3,)), "WALL_NORMAL": (np.float32, (3,)),
    "STATS": (np.float64, ()), "NEIGH_CSR_FLUID": (np.int32, ()), "NEIGH_CSR_WALL": (np.int32, ()),
    "DRHO_SAVED": (np.float32, ()), "THETA": (np.float32, ()), "CONTACT_FACTOR": (np.float32, ()), "WALL_T": (np.float32, ()), "WALL_DT_DT": (np.float32, ()),
    "FS_REGION": (np.uint32, ()), "SORT_CELL_COUNT": (np.uint32, ()), "SORT_CELL_START": (np.uint32, ()),
}
STATS = ("t", "dt", "dt_ad", "elapsed", "vmax", "steps", "rebuilds", "sigma0", "ncell_x", "ncell_y",
         "ncell_z", "error_bits", "launches", "device_bytes", "max_neigh_fluid", "max_neigh_wall", "tiles",
         "direct_tiles", "split_tiles", "t_mean", "split4_tiles")
KERNEL_CLASSES = ("control", "wall_kinematics", "hash", "scan", "scatter", "reorder", "build_lists",
                  "reinit", "pre", "sweep_A", "sweep_B", "finish", "other")


class sph_body_params(C.Structure):
    _fields_ = [("k_s", C.c_double), ("rho_s", C.c_double), ("cp_s", C.c_double),
                ("thermal_mode", C.c_int32), ("reserved", C.c_int32)]


class sph_params(C.Structure):
    _fields_ = [
        ("struct_size", C.c_uint32), ("flags", C.c_uint32),
        ("dx", C.c_double), ("h", C.c_double), ("rho0", C.c_double), ("c0", C.c_double), ("nu", C.c_double),
        ("g", C.c_double * 3), ("k_f", C.c_double), ("cp_f", C.c_double), ("T_ref", C.c_double),
        ("cfl_ac", C.c_double), ("cfl_ad", C.c_double), ("u_ref", C.c_double), ("dt_fixed", C.c_double),
        ("rebuild_every", C.c_int32), ("n_bodies", C.c_int32),
        ("domain_min", C.c_double * 3), ("domain_max", C.c_double * 3),
        ("max_fluid", C.c_uint64), ("max_wall", C.c_uint64),
        ("max_neigh_fluid", C.c_uint32), ("max_neigh_wall", C.c_uint32),
        ("body", sph_body_params * SPH_MAX_BODIES),
        ("device", C.c_int32), ("dim", C.c_int32), ("cuda_stream", C.c_void_p),
        ("fs_threshold", C.c_double),
    ]


class SphError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"libsph_b200 error {code}: {text}")
        self.code = code


_lib = None


def lib() -> C.CDLL:
    """load libsph_b200.so (built in-tree by build.py); fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2512_09904_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, u32, u64 = C.c_void_p, C.c_int, C.c_uint32, C.c_uint64
        L.sph_create.argtypes = [C.POINTER(sph_params), C.POINTER(vp)]
        L.sph_destroy.argtypes = [vp]
        L.sph_load_particles.argtypes = [vp, u64, vp, vp, vp, vp, u64, vp, vp, vp, vp, i32]
        L.sph_set_state.argtypes = [vp, vp, vp, vp, vp, i32]
        L.sph_set_materials.argtypes = [vp, vp, vp, vp, i32]
        L.sph_set_gear_kinematics.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_double]
        L.sph_step.argtypes = [vp, i32]
        L.sph_relax.argtypes = [vp, i32, C.c_double]
        L.sph_get_fields.argtypes = [vp, u32, vp, u64, i32]
        L.sph_field_bytes.argtypes = [vp, u32, C.POINTER(u64)]
        L.sph_get_torque.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.sph_synchronize.argtypes = [vp]
        L.sph_profile.argtypes = [vp, i32]
        L.sph_get_profile.argtypes = [vp, i32, C.POINTER(C.c_double), C.POINTER(u64)]
        L.sph_last_error.argtypes = [vp]
        L.sph_last_error.restype = C.c_char_p
        L.sph_cell_scan_static.argtypes = [i32, vp, vp, u32, u32, vp]
        L.sph_measure_fma_peak.argtypes = [i32, C.POINTER(C.c_double), vp]
        for f in ("sph_create", "sph_destroy", "sph_load_particles", "sph_set_gear_kinematics", "sph_step",
                  "sph_get_fields", "sph_field_bytes", "sph_get_torque", "sph_synchronize", "sph_profile",
                  "sph_get_profile", "sph_relax", "sph_set_state", "sph_set_materials", "sph_cell_scan_static", "sph_measure_fma_peak"):
            getattr(L, f).restype = C.c_int
        _lib = L
    return _lib


def _check(rc: int, ctx) -> int:
    if rc != SPH_OK:
        raise SphError(rc, (lib().sph_last_error(ctx) or b"").decode())
    return rc


def make_params(params: Dict[str, object], bodies: Optional[Sequence[object]] = None, device: int = 0,
                cuda_stream: int = 0, max_fluid: int = 0, max_wall: int = 0,
                max_neigh_fluid: int = 0, max_neigh_wall: int = 0) -> sph_params:
    """fill the POD struct from a workload-style dict (paper_2512_09904_b200.workloads.default_params)."""
    p = sph_params()
    p.struct_size = C.sizeof(sph_params)
    p.flags = int(params["flags"])
    for name in ("dx", "h", "rho0", "c0", "nu", "k_f", "cp_f", "T_ref", "cfl_ac", "cfl_ad", "u_ref", "dt_fixed"):
        setattr(p, name, float(params[name]))
    p.rebuild_every = int(params.get("rebuild_every", 0))
    for d in range(3):
        p.g[d] = float(params["g"][d])
        p.domain_min[d] = float(params["domain_min"][d])
        p.domain_max[d] = float(params["domain_max"][d])
    nb = len(bodies) if bodies else 1
    p.n_bodies = nb
    for b in range(nb):
        if bodies:
            p.body[b].k_s = float(bodies[b].k_s)
            p.body[b].rho_s = float(bodies[b].rho_s)
            p.body[b].cp_s = float(bodies[b].cp_s)
            p.body[b].thermal_mode = int(getattr(bodies[b], "thermal_mode", 0))
    p.max_fluid, p.max_wall = int(max_fluid), int(max_wall)
    p.max_neigh_fluid, p.max_neigh_wall = int(max_neigh_fluid), int(max_neigh_wall)
    p.device = int(device)
    p.dim = int(params.get("dim", 3))
    p.cuda_stream = cuda_stream or None
    p.fs_threshold = float(params.get("fs_threshold", 0.0))
    return p


# ------------------------------------------------------------------------------------------------
# the C ABI, one Python function per call (ctx is an opaque c_void_p)
# ------------------------------------------------------------------------------------------------
def sph_create(p: sph_params) -> C.c_void_p:
    ctx = C.c_void_p()
    _check(lib().sph_create(C.byref(p), C.byref(ctx)), None)
    return ctx


def sph_destroy(ctx) -> None:
    lib().sph_destroy(ctx)


def _as_ptr(a, dtype, mem_kind):
    """numpy array (HOST) or an int / object with data_ptr() (DEVICE) -> (void*, keep-alive)."""
    if a is None:
        return None, None
    if mem_kind == SPH_MEM_DEVICE:
        return C.c_void_p(int(a.data_ptr() if hasattr(a, "data_ptr") else a)), a
    arr = np.ascontiguousarray(a, dtype)
    return arr.ctypes.data_as(C.c_void_p), arr


def sph_load_particles(ctx, n_f, pos_f, vel_f, rho_f, T_f, n_w=0, pos_w=None, normal_w=None, body_w=None,
                       T_w=None, mem_kind=SPH_MEM_HOST) -> None:
    keep = []
    ptrs = []
    for a, dt in ((pos_f, np.float32), (vel_f, np.float32), (rho_f, np.float32), (T_f, np.float32)):
        p, k = _as_ptr(a, dt, mem_kind)
        ptrs.append(p); keep.append(k)
    wptrs = []
    for a, dt in ((pos_w, np.float32), (normal_w, np.float32), (body_w, np.int32), (T_w, np.float32)):
        p, k = _as_ptr(a if n_w else None, dt, mem_kind)
        wptrs.append(p); keep.append(k)
    _check(lib().sph_load_particles(ctx, int(n_f), *ptrs, int(n_w), *wptrs, int(mem_kind)), ctx)


def sph_set_materials(ctx, mass_f=None, k_f=None, cp_f=None, mem_kind=SPH_MEM_HOST) -> None:
    keep, ptrs = [], []
    for a in (mass_f, k_f, cp_f):
        p, k = _as_ptr(a, np.float32, mem_kind)
        ptrs.append(p); keep.append(k)
    _check(lib().sph_set_materials(ctx, *ptrs, int(mem_kind)), ctx)


def sph_set_state(ctx, pos_f=None, vel_f=None, rho_f=None, T_f=None, mem_kind=SPH_MEM_HOST) -> None:
    keep, ptrs = [], []
    for a in (pos_f, vel_f, rho_f, T_f):
        p, k = _as_ptr(a, np.float32, mem_kind)
        ptrs.append(p); keep.append(k)
    _check(lib().sph_set_state(ctx, *ptrs, int(mem_kind)), ctx)


def sph_set_gear_kinematics(ctx, body: int, origin, axis, omega: float) -> None:
    o = (C.c_double * 3)(*[float(x) for x in origin])
    a = (C.c_double * 3)(*[float(x) for x in axis])
    _check(lib().sph_set_gear_kinematics(ctx, int(body), o, a, float(omega)), ctx)


def sph_step(ctx, n: int = 1) -> None:
    _check(lib().sph_step(ctx, int(n)), ctx)


def sph_relax(ctx, n: int, p0: float) -> None:
    _check(lib().sph_relax(ctx, int(n), C.c_double(float(p0))), ctx)


def sph_synchronize(ctx) -> None:
    _check(lib().sph_synchronize(ctx), ctx)


def sph_field_bytes(ctx, field) -> int:
    b = C.c_uint64()
    _check(lib().sph_field_bytes(ctx, int(FIELDS[field] if isinstance(field, str) else field), C.byref(b)), ctx)
    return int(b.value)


def sph_get_fields(ctx, field: str, dst=None, mem_kind=SPH_MEM_HOST):
    """HOST: returns a numpy array (allocated here unless `dst` is given).  DEVICE: `dst` is a
    torch tensor / pointer owner with data_ptr() and nbytes; it is filled and returned."""
    fid = FIELDS[field]
    nbytes = sph_field_bytes(ctx, field)
    dtype, tail = _FIELD_LAYOUT[field]
    if mem_kind == SPH_MEM_DEVICE:
        cap = int(dst.numel() * dst.element_size())
        _check(lib().sph_get_fields(ctx, fid, C.c_void_p(int(dst.data_ptr())), cap, SPH_MEM_DEVICE), ctx)
        return dst
    if dst is None:
        n = nbytes // np.dtype(dtype).itemsize
        dst = np.empty(max(n, 1), dtype)[:n]
    if nbytes:
        _check(lib().sph_get_fields(ctx, fid, dst.ctypes.data_as(C.c_void_p), dst.nbytes, SPH_MEM_HOST), ctx)
    return dst.reshape((-1,) + tail) if tail else dst


SCAN_STATIC_MAX_CELLS = 1 << 24


def sph_cell_scan_static(device: int, counts_dev, starts_dev, n_cells: int, n_items: int, cuda_stream: int = 0) -> None:
    """row a3's exclusive scan on the library's static device scratch (include/sph.h): allocates nothing.  `counts_dev`
    (uint32 [n_cells]) and `starts_dev` (uint32 [n_cells + 1]) are DEVICE pointers or objects with data_ptr()."""
    ptr = lambda x: C.c_void_p(int(x.data_ptr()) if hasattr(x, "data_ptr") else int(x))
    _check(lib().sph_cell_scan_static(int(device), ptr(counts_dev), ptr(starts_dev), int(n_cells), int(n_items),
                                      C.c_void_p(int(cuda_stream))), None)


def sph_measure_fma_peak(device: int = 0, cuda_stream: int = 0) -> float:
    """measured plain fp32 FMA rate of the device in TFLOP/s (include/sph.h); a measurement helper of bench.py."""
    t = C.c_double()
    _check(lib().sph_measure_fma_peak(int(device), C.byref(t), C.c_void_p(int(cuda_stream))), None)
    return float(t.value)


def sph_get_torque(ctx, body: int):
    t = (C.c_double * 3)()
    ax = C.c_double()
    _check(lib().sph_get_torque(ctx, int(body), t, C.byref(ax)), ctx)
    return np.array(list(t)), float(ax.value)


def sph_profile(ctx, enable: bool) -> None:
    _check(lib().sph_profile(ctx, int(bool(enable))), ctx)


def sph_get_profile(ctx) -> Dict[str, tuple]:
    out = {}
    for k, name in enumerate(KERNEL_CLASSES):
        ms, n = C.c_double(), C.c_uint64()
        _check(lib().sph_get_profile(ctx, k, C.byref(ms), C.byref(n)), ctx)
        out[name] = (float(ms.value), int(n.value))
    return out


def sph_stats(ctx) -> Dict[str, float]:
    return dict(zip(STATS, sph_get_fields(ctx, "STATS").tolist()))


class Simulation:
    """convenience owner of one context: create + kinematics + load from a workloads.Workload."""

    def __init__(self, wl, device: int = 0, cuda_stream: int = 0, **param_over):
        params = dict(wl.params)
        caps = {k: int(param_over.pop(k)) for k in ("max_neigh_fluid", "max_neigh_wall") if k in param_over}
        params.update(param_over)
        self.params = params
        self.n_f, self.n_w = wl.n_f, wl.n_w
        self.ctx = sph_create(make_params(params, wl.bodies, device=device, cuda_stream=cuda_stream, **caps))
        for b, body in enumerate(wl.bodies):
            sph_set_gear_kinematics(self.ctx, b, body.origin, body.axis, body.omega)
        self.load(wl)

    def load(self, wl) -> None:
        sph_load_particles(self.ctx, wl.n_f, wl.pos_f, wl.vel_f, wl.rho_f, wl.T_f, wl.n_w, wl.pos_w,
                           wl.normal_w, wl.body_w, wl.T_w, SPH_MEM_HOST)

    def step(self, n: int = 1) -> None:
        sph_step(self.ctx, n)

    def relax(self, n: int, p0: float) -> None:
        sph_relax(self.ctx, n, p0)

    def sync(self) -> None:
        sph_synchronize(self.ctx)

    def get(self, field: str) -> np.ndarray:
        return sph_get_fields(self.ctx, field)

    def torque(self, body: int):
        return sph_get_torque(self.ctx, body)

    def stats(self) -> Dict[str, float]:
        return sph_stats(self.ctx)

    def close(self) -> None:
        if self.ctx is not None:
            sph_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
