"""Pins of reading R27: which fluid particles take Eq. 14 and which Eq. 15 in the density
re-initialisation ("the fluid density in regions identified as free-surface flow is reinitialized according to [Eq. 14]
... In the absence of a free surface [Eq. 15]").  -m "not gpu".

  F1  closed, fully wetted box: no surface particle, Eq. 15 for every particle (a density ABOVE rho0 comes back to rho0,
      which the max form of Eq. 14 would keep);
  F2  open tank on the unjittered lattice: exactly the top three particle layers form the free-surface region (first
      layer: truncated support, sigma / sigma0 = 0.789 < theta; layers two and three: fluid neighbours of the first), all
      deeper layers take Eq. 15; the densities follow in closed form;
  F3  region == its definition evaluated by brute force in numpy on a random cloud (independent O(N^2) evaluation);
  F4  the flags: R12 (max form everywhere) and "no free surface" (Eq. 15 everywhere) are unchanged, R27 wins when both
      free-surface flags are set;
  F5  the purpose of the reading: in a closed, fully wetted box on the jittered lattice the max form applied everywhere
      (R12) ratchets the density up and the motion grows; under R27 the motion decays.
"""
import math

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2512_09904_b200 import workloads as wl

REINIT_LOCAL = wl.FLAGS_ALL_PHYSICS | wl.FLAG_DENSITY_REINIT | wl.FLAG_FREE_SURFACE_LOCAL

# sigma / sigma0 of a particle k layers under a flat free surface of the cubic lattice, Wendland C2, h = 1.3 dx: direct
# lattice sums over the half space (the definition, evaluated here in numpy in _flat_surface_ratio and compared below)
FLAT_RATIO = {0: 0.7887393895, 1: 0.9964973954, 2: 1.0}


def _W(r, h):
    q = r / h
    return np.where(q < 2.0, 21.0 / (16.0 * math.pi * h ** 3) * (1.0 - 0.5 * q) ** 4 * (1.0 + 2.0 * q), 0.0)


def _flat_surface_ratio(k, hod=1.3, m=4):
    a = np.arange(-m, m + 1)
    X, Y, Z = np.meshgrid(a, a, a, indexing="ij")
    w = _W(np.sqrt(X * X + Y * Y + Z * Z).astype(np.float64), hod)
    return float(w[Z <= k].sum() / w.sum())


def test_F2_flat_surface_ratios_are_the_lattice_sums():
    for k, v in FLAT_RATIO.items():
        assert _flat_surface_ratio(k) == pytest.approx(v, abs=5e-10)
    assert FLAT_RATIO[0] < 0.9 < FLAT_RATIO[1]              # the default theta separates the first layer from the second


def test_F1_closed_wetted_box_takes_eq15_everywhere():
    """Fails when orc_density_reinit marks every particle under ORC_FREE_SURFACE_LOCAL (`memset(region, 1, ...)` taken for
    both flags), or when the test `sig[i] < theta * o->sigma0` is inverted."""
    w = wl.still_tank(n=8, jitter=0.0, flags=REINIT_LOCAL)
    rho_in = np.where(np.arange(w.n_f) % 3 == 0, 876.0, 864.0).astype(np.float32)
    o = orc.Oracle.from_workload(wl.dataclasses.replace(w, rho_f=rho_in))
    o.rebuild()
    assert not o.fs_region().any()
    np.testing.assert_allclose(o.get("RHO"), 870.0, rtol=1e-6, atol=0)


@pytest.mark.parametrize("rho_start", [875.0, 860.0])
def test_F2_open_tank_top_three_layers_take_the_max_form(rho_start):
    """Fails when the region is the surface particles only (`region[o->ff_idx[q]] = 1` dropped: layers two and three then
    take Eq. 15, 866.95 / 870 instead of 875), when wall neighbours are left out of sigma (the particles along the side
    walls all turn into surface particles) and when theta is applied to sigma instead of sigma / sigma0."""
    n, fill = 10, 0.6
    w = wl.still_tank(n=n, jitter=0.0, fill=fill, flags=REINIT_LOCAL)
    dx = w.params["dx"]
    layer_from_top = (int(round(fill * n)) - 1) - np.floor(w.pos_f[:, 2] / dx).astype(int)       # 0 = surface layer
    o = orc.Oracle.from_workload(wl.dataclasses.replace(w, rho_f=np.full(w.n_f, rho_start, np.float32)))
    o.rebuild()
    reg = o.fs_region().astype(bool)
    np.testing.assert_array_equal(reg, layer_from_top <= 2)
    rho = o.get("RHO")
    want = np.full(w.n_f, 870.0)                                                                 # Eq. 15 below the region
    for k in (0, 1, 2):
        want[layer_from_top == k] = max(rho_start, 870.0 * FLAT_RATIO[k])                        # Eq. 14 in the region
    # columns next to the side walls see wall particles ABOVE the surface level, so their sums exceed the flat-surface ones
    ij = np.floor(w.pos_f[:, :2] / dx).astype(int)
    inner = ((ij >= 3) & (ij <= n - 4)).all(axis=1)
    np.testing.assert_allclose(rho[inner], want[inner], rtol=2e-6, atol=0)
    assert np.all(rho[~inner] >= want[~inner] * (1 - 2e-6))


def test_F3_region_equals_brute_force_definition():
    """independent O(N^2) numpy evaluation of the definition on a random cloud with walls: sigma from all pairs inside the
    cut-off, surface = sigma < theta sigma0, region = surface particles and their fluid neighbours.  Fails when the
    neighbour marking uses the wall lists, or when sigma leaves out the self term."""
    w = wl.random_cloud(1400, 500, extent=(4, 3, 3), seed=31, snap_fraction=0.0, flags=REINIT_LOCAL)
    h = w.params["h"]
    rc2 = float(np.float32(np.float32(2.0 * h) ** 2))
    pf, pw = w.pos_f.astype(np.float64), w.pos_w.astype(np.float64)
    d2ff = ((pf[:, None, :] - pf[None, :, :]) ** 2).sum(-1)
    d2fw = ((pf[:, None, :] - pw[None, :, :]) ** 2).sum(-1)
    band = min(np.abs(d2ff - rc2).min(), np.abs(d2fw - rc2).min())
    assert band > 5e-7 * rc2                                     # no pair sits in the fp32 rounding band of the cut-off
    nb = (d2ff < rc2) & ~np.eye(len(pf), dtype=bool)
    sig = _W(0.0, h) + (_W(np.sqrt(d2ff), h) * nb).sum(1) + (_W(np.sqrt(d2fw), h) * (d2fw < rc2)).sum(1)
    sigma0 = orc.sigma0(w.params["dx"], h)
    ratio = np.sort(sig / sigma0)
    k = int(0.15 * len(ratio))
    theta = 0.5 * (ratio[k] + ratio[k + 1])                      # the cloud is denser than the lattice: put theta inside its spread
    assert ratio[k + 1] - ratio[k] > 1e-9                        # nobody sits on the threshold
    surf = sig < theta * sigma0
    region = surf | (nb & surf[None, :]).any(axis=1)
    assert region.sum() > surf.sum() > 0 and not region.all()
    o = orc.Oracle.from_workload(w, neigh_backend=1, fs_threshold=theta)
    rho_before = o.get("RHO").copy()
    o.rebuild()
    assert o.stats()["sigma0"] == pytest.approx(sigma0, rel=1e-14)
    np.testing.assert_array_equal(o.fs_region().astype(bool), region)
    rn = w.params["rho0"] * sig / sigma0
    np.testing.assert_allclose(o.get("RHO"), np.where(region, np.maximum(rho_before, rn), rn), rtol=1e-12)


def test_F4_flag_semantics():
    w = wl.still_tank(n=8, jitter=0.0, fill=0.5)
    base = wl.FLAGS_ALL_PHYSICS | wl.FLAG_DENSITY_REINIT
    rho_in = np.full(w.n_f, 878.0, np.float32)
    res = {}
    for name, fl in (("none", base), ("global", base | wl.FLAG_FREE_SURFACE), ("local", base | wl.FLAG_FREE_SURFACE_LOCAL),
                     ("both", base | wl.FLAG_FREE_SURFACE | wl.FLAG_FREE_SURFACE_LOCAL)):
        o = orc.Oracle.from_workload(wl.dataclasses.replace(w, rho_f=rho_in), flags=fl)
        o.rebuild()
        res[name] = (o.get("RHO"), o.fs_region().astype(bool))
    assert not res["none"][1].any() and res["none"][0].max() <= 870.0 * (1 + 1e-6)          # Eq. 15 everywhere
    assert res["global"][1].all() and np.all(res["global"][0] == 878.0)                      # R12: Eq. 14 everywhere
    assert res["local"][1].any() and not res["local"][1].all()
    np.testing.assert_array_equal(res["both"][0], res["local"][0])                           # R27 wins


def test_F5_closed_box_ratchet_of_the_global_max_form_is_gone_under_R27():
    """on the jittered lattice sigma_i / sigma0 scatters by +-0.3 %; Eq. 14 applied to EVERY particle
    (R12) keeps only the upward part of that noise at every rebuild, so in a closed, fully wetted box the density is pumped
    up everywhere and the motion it drives grows; under R27 the box has no surface particle, every particle takes Eq. 15,
    the density follows the kernel sum and the motion decays."""
    def run(flag):
        w = wl.still_tank(n=12, g=[0.0, 0.0, 0.0], c0=40.0, dx=4e-3)
        flags = (int(w.params["flags"]) & ~(wl.FLAG_FREE_SURFACE | wl.FLAG_FREE_SURFACE_LOCAL)) | flag
        o = orc.Oracle.from_workload(w, flags=flags)
        vmax, dmean = [], []
        for _ in range(6):
            o.step(100)
            vmax.append(float(np.linalg.norm(o.get("VEL"), axis=1).max()))
            dmean.append(float((o.get("RHO") - 870.0).mean()))
        return np.array(vmax), np.array(dmean), o
    v27, d27, o27 = run(wl.FLAG_FREE_SURFACE_LOCAL)
    assert not o27.fs_region().any()
    assert v27[-1] < 0.5 * v27[0] and abs(d27[-1]) < 0.05                 # decays, mean density at rho0
    v12, d12, o12 = run(wl.FLAG_FREE_SURFACE)
    assert o12.fs_region().all()
    assert d12[-1] > 1.0 and v12[-1] > 2.0 * v12[0]                       # pumped up by > 1 kg/m^3 (1.6 kPa at c0 = 40), motion grows
