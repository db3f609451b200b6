"""Seeded synthetic inputs shaped like the paper's cases (oil bath, dummy-particle walls, gears).

This module holds NONE of the method's arithmetic (no kernel function, no pair sums, no
integrator): it only places particles on a lattice, marks solids, and fills a parameter
dictionary.  It is the one module that serves both the CUDA path and the fp64 oracle
(`oracle/`), so that both see bit-identical fp32 input arrays.

The paper's own workloads (FZG rig; bevel-helical reducer CAD,
PAPER.md:276-308) are not available; BASELINE.json's five configs stand in for them and are
generated here.  Common structure, after PAPER.md:137 (dummy wall particles)
(c0 = 10 U_max) and Table 6 (oil / steel property scale):

  * fluid and solids are sampled on ONE cubic lattice of spacing dx (sites at (i+1/2) dx),
  * fluid sites get a seeded jitter U(-jitter*dx, +jitter*dx) per coordinate (Philox, counter
    based; the seed is part of the workload name),
  * every solid is a 3-site-thick shell of wall particles with an outward unit normal,
  * body 0 is the static adiabatic housing; heated faces / gears are bodies >= 1.

Every generator returns a `Workload` with fp32 arrays in caller ("original") order.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional

import numpy as np

# flag bits of `sph_params.flags` (values are part of the C ABI, include/sph.h)
FLAG_FREE_SURFACE = 1
FLAG_DENSITY_REINIT = 2
FLAG_THERMAL = 4
FLAG_VISCOUS = 8
FLAG_HYDRO = 16
FLAG_DUAL_CRITERIA = 32
FLAG_PRESSURE = 64
FLAG_VISCOUS_HELD = 128     # viscous sums evaluated once per advection step and held (ref [45]; R26)
FLAG_FREE_SURFACE_LOCAL = 256   # Eq. 14 only in the identified free-surface region, Eq. 15 elsewhere (R27)
FLAGS_ALL_PHYSICS = FLAG_THERMAL | FLAG_VISCOUS | FLAG_HYDRO | FLAG_PRESSURE

WALL_LAYERS = 3


@dataclasses.dataclass
class Body:
    k_s: float = 0.0          # thermal conductivity seen by the fluid (0 = adiabatic)
    rho_s: float = 7850.0
    cp_s: float = 460.0
    origin: tuple = (0.0, 0.0, 0.0)
    axis: tuple = (0.0, 0.0, 1.0)
    omega: float = 0.0
    thermal_mode: int = 0     # 0: temperature held; 1: evolving solid temperature (Eq. 20)


@dataclasses.dataclass
class Workload:
    name: str
    params: Dict[str, object]          # plain python scalars / lists, see `default_params`
    pos_f: np.ndarray                  # [n_f,3] f32
    vel_f: np.ndarray                  # [n_f,3] f32
    rho_f: Optional[np.ndarray]        # [n_f] f32 or None (-> rho0)
    T_f: np.ndarray                    # [n_f] f32
    pos_w: np.ndarray                  # [n_w,3] f32
    normal_w: np.ndarray               # [n_w,3] f32, unit, solid -> fluid
    body_w: np.ndarray                 # [n_w] i32
    T_w: np.ndarray                    # [n_w] f32
    bodies: List[Body]

    @property
    def n_f(self) -> int:
        return int(self.pos_f.shape[0])

    @property
    def n_w(self) -> int:
        return int(self.pos_w.shape[0])


def default_params(dx: float, **kw) -> Dict[str, object]:
    p = dict(
        flags=FLAGS_ALL_PHYSICS | FLAG_FREE_SURFACE_LOCAL | FLAG_DENSITY_REINIT,   # Eq. 14 in the free-surface region, Eq. 15 elsewhere (R27)
        dx=dx, h=1.3 * dx, rho0=870.0, c0=20.0, nu=1.0e-4, g=[0.0, 0.0, -9.81],
        k_f=0.13, cp_f=2000.0, T_ref=313.0,
        cfl_ac=0.6, cfl_ad=0.25, u_ref=-1.0,      # u_ref < 0 -> c0/10
        dt_fixed=0.0, rebuild_every=0,
        domain_min=[0.0, 0.0, 0.0], domain_max=[1.0, 1.0, 1.0],
    )
    p.update(kw)
    return p


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(seed))


def _sites(lo, hi) -> np.ndarray:
    """integer lattice sites lo <= (i,j,k) < hi as an [n,3] int32 array, x fastest."""
    ax = [np.arange(lo[d], hi[d], dtype=np.int32) for d in range(3)]
    k, j, i = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    return np.stack([i.ravel(), j.ravel(), k.ravel()], axis=1)


def _to_pos(sites: np.ndarray, dx: float, origin=(0.0, 0.0, 0.0)) -> np.ndarray:
    return ((sites.astype(np.float64) + 0.5) * dx + np.asarray(origin, np.float64))


def _box_shell(n_in, layers=WALL_LAYERS, open_top=False):
    """sites of a `layers`-thick shell around the cavity 0 <= i < n_in, and inward normals."""
    lo = [-layers] * 3
    hi = [n_in[d] + layers for d in range(3)]
    if open_top:
        hi[2] = n_in[2]
    s = _sites(lo, hi)
    below = s < 0
    above = s >= np.asarray(n_in, np.int32)[None, :]
    if open_top:
        above[:, 2] = False
    keep = (below | above).any(axis=1)
    s, below, above = s[keep], below[keep], above[keep]
    nrm = below.astype(np.float64) - above.astype(np.float64)   # points into the cavity
    nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
    return s, nrm, below, above


def _finish(name, params, dx, f_sites, w_pos, w_nrm, w_body, w_T, bodies, T_f, seed,
            jitter, origin=(0.0, 0.0, 0.0), pad_cells=0.5, rho_f=None, vel_f=None):
    rng = _rng(seed)
    pos_f = _to_pos(f_sites, dx, origin)
    if jitter > 0:
        pos_f = pos_f + rng.uniform(-jitter * dx, jitter * dx, size=pos_f.shape)
    allp = [pos_f] + ([w_pos] if len(w_pos) else [])
    lo = np.min([a.min(axis=0) for a in allp], axis=0)
    hi = np.max([a.max(axis=0) for a in allp], axis=0)
    pad = pad_cells * 2.0 * float(params["h"])
    params["domain_min"] = [float(x) for x in (lo - pad)]
    params["domain_max"] = [float(x) for x in (hi + pad)]
    n_f = pos_f.shape[0]
    return Workload(
        name=name, params=params,
        pos_f=np.ascontiguousarray(pos_f, np.float32),
        vel_f=np.zeros((n_f, 3), np.float32) if vel_f is None else np.ascontiguousarray(vel_f, np.float32),
        rho_f=None if rho_f is None else np.ascontiguousarray(rho_f, np.float32),
        T_f=np.full(n_f, T_f, np.float32),
        pos_w=np.ascontiguousarray(w_pos, np.float32).reshape(-1, 3),
        normal_w=np.ascontiguousarray(w_nrm, np.float32).reshape(-1, 3),
        body_w=np.ascontiguousarray(w_body, np.int32),
        T_w=np.ascontiguousarray(w_T, np.float32),
        bodies=bodies,
    )


# ----------------------------------------------------------------------------------------------
# config 0: still oil tank (BASELINE.json configs[0])
# ----------------------------------------------------------------------------------------------
def still_tank(n: int = 24, dx: float = 2.0e-3, seed: int = 0, jitter: float = 0.01,
               fill: float = 1.0, c0: float = 20.0, **over) -> Workload:
    """n^3 cavity enclosed by 3 wall layers; the x_min face (body 1) is held at 353 K with
    k = k_f, the other five faces (body 0) are adiabatic.  `fill` < 1 leaves a free surface."""
    nz_f = max(1, int(round(fill * n)))
    f_sites = _sites((0, 0, 0), (n, n, nz_f))
    w_sites, w_nrm, below, _ = _box_shell((n, n, n))
    body = np.where(below[:, 0], 1, 0).astype(np.int32)
    params = default_params(dx, c0=c0)
    params.update(over)
    bodies = [Body(k_s=0.0), Body(k_s=float(params["k_f"]))]
    T_w = np.where(body == 1, 353.0, 313.0)
    return _finish(f"still_tank_n{n}_seed{seed}", params, dx, f_sites, _to_pos(w_sites, dx),
                   w_nrm, body, T_w, bodies, 313.0, seed, jitter)


# ----------------------------------------------------------------------------------------------
# config 1: dam break with a heated floor (BASELINE.json configs[1])
# ----------------------------------------------------------------------------------------------
def dam_break(dx: float = 3.0e-3, seed: int = 1, jitter: float = 0.01, box=(1.2, 0.3, 0.6),
              column=(0.3, 0.3, 0.6), c0: float = 40.0, scale: float = 1.0, **over) -> Workload:
    """oil column in a closed box; floor (body 1) at 353 K, everything else adiabatic.
    `scale` multiplies all lengths except dx (particle count ~ scale^3)."""
    nb = [int(round(scale * b / dx)) for b in box]
    nc = [min(int(round(scale * c / dx)), nb[d]) for d, c in enumerate(column)]
    f_sites = _sites((0, 0, 0), nc)
    w_sites, w_nrm, below, _ = _box_shell(nb)
    body = np.where(below[:, 2], 1, 0).astype(np.int32)
    params = default_params(dx, c0=c0)
    params.update(over)
    bodies = [Body(k_s=0.0), Body(k_s=float(params["k_f"]))]
    T_w = np.where(body == 1, 353.0, 313.0)
    return _finish(f"dam_break_dx{dx:g}_s{scale:g}_seed{seed}", params, dx, f_sites,
                   _to_pos(w_sites, dx), w_nrm, body, T_w, bodies, 313.0, seed, jitter)


# ----------------------------------------------------------------------------------------------
# solids sampled on the lattice: shell extraction + normals (reading R16 in DESIGN.md)
# ----------------------------------------------------------------------------------------------
def _shell_and_normals(solid: np.ndarray, layers: int = WALL_LAYERS):
    """solid: bool [nx,ny,nz].  Returns (mask of shell sites, normals [nx,ny,nz,3]).
    shell  = solid sites with a non-solid site within `layers` sites (Euclidean);
    normal = normalised sum of (r_empty - r_site) over those non-solid sites."""
    from scipy import ndimage

    r = layers
    ax = np.arange(-r, r + 1)
    ox, oy, oz = np.meshgrid(ax, ax, ax, indexing="ij")
    ball = (ox * ox + oy * oy + oz * oz) <= r * r
    empty = (~solid).astype(np.float32)
    cnt = ndimage.correlate(empty, ball.astype(np.float32), mode="constant", cval=1.0)
    shell = solid & (cnt > 0.5)
    nrm = np.zeros(solid.shape + (3,), np.float32)
    for d, off in enumerate((ox, oy, oz)):
        w = (ball * off).astype(np.float32)
        nrm[..., d] = ndimage.correlate(empty, w, mode="constant", cval=0.0)
    norm = np.linalg.norm(nrm, axis=-1, keepdims=True)
    nrm = np.where(norm > 0, nrm / np.maximum(norm, 1e-30), 0.0)
    return shell, nrm


def _inv(a):
    return np.tan(a) - a


def _spur_profile_inside(rad, ang, z: int, module: float, alpha=math.radians(20.0)):
    """textbook involute spur gear cross-section: inside(r, theta) for arrays rad, ang.
    tooth half-angle at radius r >= r_b: pi/(2z) + inv(alpha) - inv(acos(r_b / r))."""
    r_p = 0.5 * module * z
    r_b = r_p * math.cos(alpha)
    r_tip = r_p + module
    r_root = r_p - 1.25 * module
    pitch = 2.0 * math.pi / z
    rr = np.clip(rad, max(r_b, 1e-12), None)
    half = math.pi / (2 * z) + _inv(alpha) - _inv(np.arccos(np.clip(r_b / rr, -1.0, 1.0)))
    a = np.mod(ang + 0.5 * pitch, pitch) - 0.5 * pitch
    tooth = (np.abs(a) <= half) & (rad <= r_tip)
    return (rad <= r_root) | tooth


def _gear_solid(shape, dx, centre, axis: int, z: int, module: float, width: float,
                helix: float = 0.0, phase: float = 0.0, cone: float = 0.0, bore: float = 0.0):
    """bool grid of lattice sites inside a (helical / straight-bevel) involute gear.
    axis: 0/1/2 lattice axis of rotation; helix: helix angle (rad) at the pitch radius;
    cone: half pitch-cone angle (rad), 0 = cylindrical; profile scales linearly along the axis."""
    idx = np.indices(shape, dtype=np.float32)
    p = [(idx[d] + 0.5) * dx - centre[d] for d in range(3)]
    a = p[axis]
    u, v = [p[d] for d in range(3) if d != axis]
    rad = np.sqrt(u * u + v * v)
    ang = np.arctan2(v, u)
    r_p = 0.5 * module * z
    s = np.ones_like(a)
    if cone > 0.0:
        s = np.clip(1.0 - a * math.tan(cone) / r_p, 0.05, None)   # taper towards the apex
    tw = phase + (a * math.tan(helix) / r_p if helix != 0.0 else 0.0)
    inside = _spur_profile_inside(rad / s, ang - tw, z, module)
    inside &= np.abs(a) <= 0.5 * width
    if bore > 0.0:
        inside &= rad >= bore
    return inside


# ----------------------------------------------------------------------------------------------
# body-fitted solids (section 2.2: the paper's gears carry "body-fitted" particles from a level-set /
# relaxation pre-processor, not lattice samples).  A lattice-sampled (stair-step) surface that turns against the fluid lattice
# lets single fluid particles slip into its notches, from where they are shot out at several times the tip speed (measured
# with the oracle on a plain rotating cylinder).  OPTIONAL generator (`fitted=True`; the five configs keep
# the lattice-sampled solids: on the gear workloads the body-fitted shell did not remove the fast particles, DESIGN.md
# section 3).  Here the three dummy-particle layers of a gear
# follow its surface: layer k lies on the inward offset curve of the cross-section at depth (k + 1/2) dx, sampled at
# arc-length spacing dx, stacked along the axis at spacing dx (twisted / tapered per station for helical / bevel gears);
# the two flat faces are closed by three lattice layers of the cross-section interior.  Normals are the outline's.
# ----------------------------------------------------------------------------------------------
def _outline(z: int, module: float, n_theta: int = 36000):
    """closed outline of the involute cross-section (star-shaped about the centre) as a dense CCW polyline with outward unit
    normals: boundary radius per polar ray by bisection on `_spur_profile_inside`, then arc-length resampling."""
    th = np.linspace(0.0, 2.0 * math.pi, n_theta, endpoint=False)
    lo = np.zeros_like(th)
    hi = np.full_like(th, 0.5 * module * z + 1.5 * module)
    for _ in range(44):
        mid = 0.5 * (lo + hi)
        ins = _spur_profile_inside(mid, th, z, module)
        lo = np.where(ins, mid, lo)
        hi = np.where(ins, hi, mid)
    pts = np.stack([lo * np.cos(th), lo * np.sin(th)], axis=1)
    seg = np.linalg.norm(np.roll(pts, -1, axis=0) - pts, axis=1)
    arc = np.concatenate([[0.0], np.cumsum(seg)])
    total = arc[-1]
    n = int(total / (module / 200.0))
    sq = np.linspace(0.0, total, n, endpoint=False)
    closed = np.vstack([pts, pts[:1]])
    P = np.stack([np.interp(sq, arc, closed[:, d]) for d in range(2)], axis=1)
    tan = np.roll(P, -1, axis=0) - np.roll(P, 1, axis=0)
    tan /= np.linalg.norm(tan, axis=1, keepdims=True)
    nrm = np.stack([tan[:, 1], -tan[:, 0]], axis=1)                 # CCW polyline: outward = tangent turned by -90 degrees
    return P, nrm


def _offset_layer(P, nrm, depth: float, spacing: float, tree):
    """points of the inward offset curve at `depth`, thinned to arc-length `spacing`; offsets that come closer than `depth` to
    another part of the outline (concave roots, thin tips) are dropped."""
    Q = P - depth * nrm
    dist, _ = tree.query(Q)
    ok = dist >= depth * (1.0 - 2.0e-3)
    idx = np.nonzero(ok)[0]
    if len(idx) == 0:
        return np.zeros((0, 2)), np.zeros((0, 2))
    Qk = Q[idx]
    step = np.linalg.norm(np.diff(Qk, axis=0), axis=1)
    step = np.minimum(step, spacing)                                # a dropped stretch counts as one spacing
    acc = np.concatenate([[0.0], np.cumsum(step)])
    n = max(int(round(acc[-1] / spacing)), 1)
    pick = np.searchsorted(acc, (np.arange(n) + 0.5) * acc[-1] / n)
    pick = np.unique(np.clip(pick, 0, len(idx) - 1))
    return Qk[pick], nrm[idx[pick]]


def _thin(q, n, kept, dmin):
    """drop points of q (in order) that lie within dmin of a point of `kept` or of an earlier point of q"""
    from scipy.spatial import cKDTree
    if len(q) == 0:
        return q, n
    ok = np.ones(len(q), bool)
    if len(kept):
        d, _ = cKDTree(kept).query(q)
        ok &= d >= dmin
    for i, j in sorted(cKDTree(q).query_pairs(dmin)):
        if ok[i] and ok[j]:
            ok[j] = False
    return q[ok], n[ok]


def _fitted_gear(dx, centre, axis: int, z: int, module: float, width: float, helix: float = 0.0, phase: float = 0.0,
                 cone: float = 0.0, layers: int = WALL_LAYERS):
    """body-fitted dummy particles of one gear: positions [n,3], outward normals [n,3] (world frame, gear at rest angle)."""
    from scipy.spatial import cKDTree
    P0, N0 = _outline(z, module)
    r_p = 0.5 * module * z
    nst = max(int(round(width / dx)), 1)
    stations = (np.arange(nst) + 0.5) * (width / nst) - 0.5 * width
    others = [d for d in range(3) if d != axis]
    pos, nrm = [], []
    cache = {}
    for j, a in enumerate(stations):
        sc = max(1.0 - a * math.tan(cone) / r_p, 0.05) if cone > 0.0 else 1.0
        key = round(sc, 9)
        if key not in cache:
            P = P0 * sc
            tree = cKDTree(P)
            lay, kept = [], np.zeros((0, 2))
            for k in range(layers):                                  # thin tips / concave roots: no two particles closer than 0.6 dx
                q, n = _offset_layer(P, N0, (k + 0.5) * dx, dx, tree)
                q, n = _thin(q, n, kept, 0.6 * dx)
                lay.append((q, n)); kept = np.vstack([kept, q])
            # interior of the cross-section deeper than the shell, on a lattice: closes the flat faces
            rmax = float(np.linalg.norm(P, axis=1).max())
            g = (np.arange(-int(rmax / dx) - 1, int(rmax / dx) + 2) + 0.5) * dx
            U, V = np.meshgrid(g, g, indexing="ij")
            cand = np.stack([U.ravel(), V.ravel()], axis=1)
            rad, ang = np.linalg.norm(cand, axis=1), np.arctan2(cand[:, 1], cand[:, 0])
            ins = _spur_profile_inside(rad / sc, ang, z, module)
            dist, _ = tree.query(cand)
            core = cand[ins & (dist >= layers * dx)]
            core, _ = _thin(core, core, kept, 0.6 * dx)
            cache[key] = (lay, core)
        lay, core = cache[key]
        tw = phase + (a * math.tan(helix) / r_p if helix != 0.0 else 0.0)
        c, s_ = math.cos(tw), math.sin(tw)
        rot = np.array([[c, -s_], [s_, c]])
        cap = min(j, nst - 1 - j) < layers                           # station within three layers of a flat face
        parts = [(q @ rot.T, n @ rot.T, None) for q, n in lay]
        if cap and len(core):
            sign = -1.0 if j < nst - 1 - j else 1.0
            parts.append((core @ rot.T, None, sign))
        for q, n, sign in parts:
            p3 = np.zeros((len(q), 3)); n3 = np.zeros((len(q), 3))
            p3[:, others[0]], p3[:, others[1]], p3[:, axis] = q[:, 0], q[:, 1], a
            if n is not None:
                n3[:, others[0]], n3[:, others[1]] = n[:, 0], n[:, 1]
            else:
                n3[:, axis] = sign
            pos.append(p3 + np.asarray(centre)[None, :]); nrm.append(n3)
    return np.concatenate(pos), np.concatenate(nrm)


def _assemble_gearbox(name, dx, box, gears, fill_height, params, seed, jitter, T_oil, T_gear, fitted=False):
    """housing = closed box of `box` metres (body 0); gears = list of dicts for `_gear_solid`
    plus 'omega', 'k_s'.  Fluid fills non-solid sites below fill_height (metres, lattice z)."""
    nb = [int(round(b / dx)) for b in box]
    solid_any = np.zeros(nb, bool)
    w_pos, w_nrm, w_body, w_T, bodies = [], [], [], [], [Body(k_s=0.0)]
    hs, hn, _, _ = _box_shell(nb)
    w_pos.append(_to_pos(hs, dx)); w_nrm.append(hn)
    w_body.append(np.zeros(len(hs), np.int32)); w_T.append(np.full(len(hs), T_oil))
    for b, gd in enumerate(gears, start=1):
        g = dict(gd)
        omega = g.pop("omega"); k_s = g.pop("k_s")
        solid = _gear_solid(nb, dx, **g)
        solid_any |= solid
        if fitted:
            gp, gn = _fitted_gear(dx, **{k: v for k, v in g.items() if k != "bore"})
            w_pos.append(gp); w_nrm.append(gn)
            w_body.append(np.full(len(gp), b, np.int32)); w_T.append(np.full(len(gp), T_gear))
        else:
            shell, nrm = _shell_and_normals(solid)
            ii = np.argwhere(shell).astype(np.int32)
            w_pos.append(_to_pos(ii, dx)); w_nrm.append(nrm[shell])
            w_body.append(np.full(len(ii), b, np.int32)); w_T.append(np.full(len(ii), T_gear))
        ax = [0.0, 0.0, 0.0]; ax[g["axis"]] = 1.0
        bodies.append(Body(k_s=k_s, origin=tuple(float(c) for c in g["centre"]), axis=tuple(ax),
                           omega=float(omega)))
    nzf = int(round(fill_height / dx))
    fl = ~solid_any
    fl[:, :, nzf:] = False
    f_sites = np.argwhere(fl).astype(np.int32)
    if fitted and len(w_pos) > 1:
        # oil sites closer than 0.8 dx to a body-fitted gear particle would overlap its first layer (which lies half a spacing
        # under the surface): leave them out
        from scipy.spatial import cKDTree
        d, _ = cKDTree(np.concatenate(w_pos[1:])).query(_to_pos(f_sites, dx), distance_upper_bound=dx)
        f_sites = f_sites[d >= 0.8 * dx]
    return _finish(name, params, dx, f_sites, np.concatenate(w_pos), np.concatenate(w_nrm),
                   np.concatenate(w_body), np.concatenate(w_T), bodies, T_oil, seed, jitter)


# ----------------------------------------------------------------------------------------------
# configs 2 / 3: single spur gear in an oil bath (BASELINE.json configs[2], configs[3])
# ----------------------------------------------------------------------------------------------
def spur_gear(dx: float = 1.5e-3, omega: float = 150.0, thermal: bool = False, seed: int = 2,
              jitter: float = 0.01, box=(0.2, 0.1, 0.2), z: int = 30, module: float = 4.0e-3,
              width: float = 40.0e-3, **over) -> Workload:
    r_tip = 0.5 * module * z + module
    centre = (0.5 * box[0], 0.5 * box[1], 0.5 * box[2])
    c0 = 10.0 * omega * r_tip                                   # PAPER.md:48, c0 = 10 U_max
    params = default_params(dx, c0=c0, nu=2.0e-4 if thermal else 1.0e-4)
    if not thermal:
        params["flags"] = int(params["flags"]) & ~FLAG_THERMAL
    params.update(over)
    gears = [dict(centre=centre, axis=1, z=z, module=module, width=width, omega=omega,
                  k_s=45.0 if thermal else 0.0)]
    return _assemble_gearbox(f"spur_gear_dx{dx:g}_w{omega:g}_seed{seed}", dx, box, gears,
                             centre[2], params, seed, jitter, 313.0, 353.0)


# ----------------------------------------------------------------------------------------------
# config 4: synthetic bevel-helical reducer (BASELINE.json configs[4])
# ----------------------------------------------------------------------------------------------
def reducer(dx: float = 1.0e-3, omega_in: float = 300.0, seed: int = 4, jitter: float = 0.01,
            box=(0.35, 0.25, 0.3), **over) -> Workload:
    """helical pair 20/60 (module 3 mm, helix 15 deg) on shafts along y; straight bevel pair 18/36
    (module 3 mm), pinion along x driving a wheel along y.  Ratios: bevel 18/36, helical 20/60."""
    m = 3.0e-3
    hx = math.radians(15.0)
    r20, r60 = 0.5 * m * 20 / math.cos(hx), 0.5 * m * 60 / math.cos(hx)
    r18, r36 = 0.5 * m * 18, 0.5 * m * 36
    zc = 0.5 * box[2]
    w_in = omega_in
    w_mid = -w_in * 18.0 / 36.0
    w_out = -w_mid * 20.0 / 60.0
    x_big = box[0] - r60 - 0.03
    x_small = x_big - (r60 + r20)
    y_hel = 0.30 * box[1]
    y_bev = 0.70 * box[1]
    d18, d36 = math.atan2(18.0, 36.0), math.atan2(36.0, 18.0)
    gears = [
        dict(centre=(x_big, y_hel, zc), axis=1, z=60, module=m / math.cos(hx), width=0.03,
             helix=-hx, omega=w_out, k_s=45.0),
        dict(centre=(x_small, y_hel, zc), axis=1, z=20, module=m / math.cos(hx), width=0.03,
             helix=hx, phase=math.pi / 20, omega=w_mid, k_s=45.0),
        dict(centre=(x_small, y_bev, zc), axis=1, z=36, module=m, width=0.018, cone=d36,
             omega=w_mid, k_s=45.0),
        dict(centre=(x_small - r36 - 0.004, y_bev + r18 + 0.004, zc), axis=0, z=18, module=m,
             width=0.018, cone=d18, phase=math.pi / 18, omega=w_in, k_s=45.0),
    ]
    c0 = 10.0 * abs(w_out) * (r60 + m)
    params = default_params(dx, c0=max(c0, 10.0 * abs(w_in) * (r18 + m)), nu=1.0e-4)
    params.update(over)
    fill = zc - r60 - m + 0.30 * 2.0 * (r60 + m)            # 30 % of the large gear's diameter
    return _assemble_gearbox(f"reducer_dx{dx:g}_w{omega_in:g}_seed{seed}", dx, box, gears, fill,
                             params, seed, jitter, 313.0, 353.0)


# ----------------------------------------------------------------------------------------------
# small random clouds for neighbour-search tests (face / corner / empty-cell cases)
# ----------------------------------------------------------------------------------------------
def random_cloud(n_f: int, n_w: int, dx: float = 2.0e-3, extent=(8, 8, 8), seed: int = 7,
                 snap_fraction: float = 0.2, **over) -> Workload:
    """uniform random points in a box of `extent` cells; a fraction is snapped onto multiples of
    the cell edge (faces, edges, corners of the grid) to stress the cell predicate."""
    rng = _rng(seed)
    params = default_params(dx)
    params.update(over)
    ell = 2.0 * float(params["h"])
    ext = np.asarray(extent, np.float64) * ell

    def cloud(n):
        p = rng.uniform(0.0, 1.0, size=(n, 3)) * ext
        snap = rng.uniform(size=(n, 3)) < snap_fraction
        p = np.where(snap, np.round(p / ell) * ell, p)
        return np.clip(p, 0.0, ext)

    pos_f, pos_w = cloud(n_f), cloud(n_w)
    nrm = rng.normal(size=(n_w, 3))
    nrm /= np.linalg.norm(nrm, axis=1, keepdims=True) if n_w else 1.0
    params["domain_min"] = [0.0, 0.0, 0.0]
    params["domain_max"] = [float(e) for e in ext]
    wl = Workload(
        name=f"cloud_{n_f}_{n_w}_seed{seed}", params=params,
        pos_f=pos_f.astype(np.float32), vel_f=rng.normal(scale=0.5, size=(n_f, 3)).astype(np.float32),
        rho_f=(float(params["rho0"]) * (1.0 + 1e-3 * rng.normal(size=n_f))).astype(np.float32),
        T_f=(313.0 + 5.0 * rng.normal(size=n_f)).astype(np.float32),
        pos_w=pos_w.astype(np.float32).reshape(-1, 3), normal_w=nrm.astype(np.float32).reshape(-1, 3),
        body_w=(np.arange(n_w) % 2).astype(np.int32), T_w=np.full(n_w, 353.0, np.float32),
        bodies=[Body(k_s=0.0), Body(k_s=0.13)],
    )
    return wl


def perturb_state(wl: Workload, seed: int = 11, v_scale: float = 0.2, rho_rel: float = 5e-4,
                  T_scale: float = 3.0) -> Workload:
    """give a lattice workload a non-trivial (seeded, smooth-free random) v, rho, T state so that
    every pair term is exercised in single-step parity tests."""
    rng = _rng(seed)
    n = wl.n_f
    rho0 = float(wl.params["rho0"])
    return dataclasses.replace(
        wl,
        vel_f=(v_scale * rng.normal(size=(n, 3))).astype(np.float32),
        rho_f=(rho0 * (1.0 + rho_rel * rng.normal(size=n))).astype(np.float32),
        T_f=(wl.T_f.astype(np.float64) + T_scale * rng.normal(size=n)).astype(np.float32),
    )


def by_name(name: str, **kw) -> Workload:
    table = {
        "cfg0": still_tank, "still_tank": still_tank,
        "cfg1": dam_break, "dam_break": dam_break,
        "cfg2": lambda **k: spur_gear(dx=1.5e-3, omega=150.0, thermal=False, **k),
        "cfg3": lambda **k: spur_gear(dx=1.2e-3, omega=600.0, thermal=True, seed=3, **k),
        "cfg4": reducer, "reducer": reducer,
    }
    return table[name](**kw)
