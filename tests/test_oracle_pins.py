"""Pins of the fp64 oracle against things other than itself (-m "not gpu").

P-numbers follow SURVEY.md section 8(c) / DESIGN.md section 5.  Each test is chosen so that a
plausible slip in oracle/sph_oracle.c (a dropped term, a sign, a factor 2, a transposed operand)
fails it: closed forms, limits, conservation laws, brute force, the paper's Table 3 benchmark.
"""
import math

import numpy as np
import pytest
from scipy import integrate, special

from oracle import oracle as orc
from paper_2512_09904_b200 import workloads as wl


# ------------------------------------------------------------------------------------------------
# helpers (input construction only)
# ------------------------------------------------------------------------------------------------
def lattice_cloud(n, dx, h_over_dx=1.3, **over):
    """n^3 unjittered lattice, no walls, no gravity."""
    w = wl.still_tank(n=n, dx=dx, jitter=0.0, g=[0.0, 0.0, 0.0], h=h_over_dx * dx, **over)
    params = dict(w.params)
    return params, w.pos_f.copy()


def make_oracle(params, pos, vel=None, rho=None, T=None, walls=None, bodies=None, backend=0):
    o = orc.Oracle(params, bodies, backend)
    n = len(pos)
    vel = np.zeros((n, 3), np.float32) if vel is None else vel
    T = np.zeros(n, np.float32) if T is None else T
    if walls is None:
        o.load_particles(pos, vel, rho, T)
    else:
        o.load_particles(pos, vel, rho, T, *walls)
    return o


def centre_index(pos):
    c = 0.5 * (pos.min(axis=0) + pos.max(axis=0))
    return int(np.argmin(((pos - c) ** 2).sum(axis=1)))


# ------------------------------------------------------------------------------------------------
# P2  kernel: normalisation, derivative, lattice partition of unity
# ------------------------------------------------------------------------------------------------
def test_P2_kernel_integrates_to_one():
    for h in (0.7, 1.0, 2.6e-3):
        val, _ = integrate.quad(lambda r: 4.0 * math.pi * r * r * orc.W(r, h), 0.0, 2.0 * h, epsabs=0, epsrel=1e-12)
        assert abs(val - 1.0) < 1e-10
        assert orc.W(2.0 * h, h) == 0.0 and orc.W(2.5 * h, h) == 0.0


def test_P2_dWdr_is_derivative_of_W():
    h = 1.3
    for r in np.linspace(0.05, 2.55, 26):
        e = 1e-6
        fd = (orc.W(r + e, h) - orc.W(r - e, h)) / (2 * e)
        assert abs(fd - orc.dWdr(r, h)) < 1e-8
    # first moment: int r W' dV = -3 int W dV = -3 (integration by parts)
    val, _ = integrate.quad(lambda r: 4.0 * math.pi * r ** 3 * orc.dWdr(r, h), 0.0, 2.0 * h, epsrel=1e-12)
    assert abs(val + 3.0) < 1e-9


def test_P2_lattice_partition_of_unity(golden):
    g = golden("kernel_lattice_sums.txt")
    assert abs(orc.sigma0(1.0, 1.3) - g["partition_h1.3"]) < 5e-10
    assert abs(orc.sigma0(1.0, 1.0) - g["partition_h1.0"]) < 5e-10
    assert abs(orc.sigma0(1.0, 4.0) - 1.0) < 2e-5             # -> 1 as h/dx grows
    # scaling: sum W * dx^3 is independent of dx
    assert abs(orc.sigma0(2e-3, 2.6e-3) * 8e-9 - g["partition_h1.3"]) < 1e-9


def test_P2_density_reinit_on_full_lattice_returns_rho0():
    params, pos = lattice_cloud(9, 2e-3, flags=wl.FLAGS_ALL_PHYSICS | wl.FLAG_DENSITY_REINIT)
    o = make_oracle(params, pos, rho=np.full(len(pos), 800.0, np.float32))
    o.rebuild()
    rho = o.get("RHO")
    i = centre_index(pos)
    assert abs(rho[i] - 870.0) < 1e-3                          # Eq. 15: rho0 * sigma/sigma0 (fp32 input positions)
    assert rho.min() < 0.6 * 870.0                             # corners see a truncated support


def test_P2_density_reinit_free_surface_keeps_larger(golden):
    params, pos = lattice_cloud(7, 2e-3, flags=wl.FLAGS_ALL_PHYSICS | wl.FLAG_DENSITY_REINIT | wl.FLAG_FREE_SURFACE)
    o = make_oracle(params, pos, rho=np.full(len(pos), 871.0, np.float32))
    o.rebuild()
    np.testing.assert_allclose(o.get("RHO"), 871.0, rtol=0, atol=1e-9)   # Eq. 14: max(rho*, ...) keeps 871 everywhere


# ------------------------------------------------------------------------------------------------
# P1 / P13  neighbour sets: cell list == brute force == the mathematical definition
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("extent,seed", [((5, 4, 3), 7), ((1, 1, 1), 8), ((9, 1, 2), 9)])
def test_P1_cell_list_equals_brute_force(extent, seed):
    w = wl.random_cloud(1500, 400, extent=extent, seed=seed)
    a = orc.Oracle.from_workload(w, neigh_backend=0)
    b = orc.Oracle.from_workload(w, neigh_backend=1)
    a.rebuild(); b.rebuild()
    for which in (0, 1):
        sa, ia = a.csr(which)
        sb, ib = b.csr(which)
        np.testing.assert_array_equal(sa, sb)
        np.testing.assert_array_equal(ia, ib)
    np.testing.assert_array_equal(a.neigh()[2], b.neigh()[2])


def test_P1_sets_match_exact_distance_definition():
    w = wl.random_cloud(1200, 300, extent=(4, 4, 4), seed=21)
    o = orc.Oracle.from_workload(w, neigh_backend=0)
    o.rebuild()
    rc2 = float(np.float32(np.float32(2.0 * w.params["h"]) ** 2))
    pf = w.pos_f.astype(np.float64)
    for which, other in ((0, pf), (1, w.pos_w.astype(np.float64))):
        start, idx = o.csr(which)
        d2 = ((pf[:, None, :] - other[None, :, :]) ** 2).sum(-1)       # exact products of fp32 differences
        member = np.zeros_like(d2, bool)
        rows = np.repeat(np.arange(len(pf)), np.diff(start))
        member[rows, idx] = True
        clear = np.abs(d2 - rc2) > 1e-6 * rc2                           # outside the fp32 rounding band
        if which == 0:
            clear &= ~np.eye(len(pf), dtype=bool)
            assert not member[np.eye(len(pf), dtype=bool)].any()         # j != i
            np.testing.assert_array_equal(member, member.T)              # symmetric
        np.testing.assert_array_equal(member[clear], (d2 < rc2)[clear])
        for i in range(0, len(pf), 97):                                   # P13: lists ascending, no duplicates
            li = idx[start[i]:start[i + 1]]
            assert np.all(np.diff(li) > 0)


def test_P1_cells_are_floor_of_scaled_coordinate():
    w = wl.random_cloud(2000, 0, extent=(6, 5, 4), seed=3, snap_fraction=0.0)
    o = orc.Oracle.from_workload(w)
    o.rebuild()
    cf, _ = o.cells()
    ell = 2.0 * w.params["h"] * (1.0 + 2.0 ** -10)
    exact = w.pos_f.astype(np.float64) / ell
    safe = np.abs(exact - np.round(exact)) > 1e-4
    np.testing.assert_array_equal(cf[safe], np.floor(exact).astype(np.int32)[safe])
    assert o.grid_dims() == (6, 5, 4)


def test_P2_lattice_has_80_neighbours(golden):
    g = golden("kernel_lattice_sums.txt")
    for hod, key in ((1.3, "neighbours_h1.3"), (1.0, "neighbours_h1.0")):
        params, pos = lattice_cloud(9, 2e-3, h_over_dx=hod)
        o = make_oracle(params, pos)
        o.rebuild()
        got = int(o.neigh()[0][centre_index(pos)])
        if hod == 1.3:
            assert got == int(g[key])
        else:       # |n| = 2 sites sit exactly on the cut-off; fp32 positions put some just inside (W = 0 there)
            assert int(g[key]) <= got <= int(g[key]) + 6


# ------------------------------------------------------------------------------------------------
# P3 / P4  conservation: pairwise antisymmetry of the momentum and heat sums
# ------------------------------------------------------------------------------------------------
def _cloud_no_walls(seed=5, n=1500):
    w = wl.random_cloud(n, 0, extent=(4, 4, 4), seed=seed, snap_fraction=0.0, g=[0.0, 0.0, 0.0],
                        flags=wl.FLAGS_ALL_PHYSICS)
    # keep particles apart (no coincident points): thin the cloud onto distinct lattice sites + jitter
    dx = w.params["dx"]
    sites = np.unique(np.round(w.pos_f / dx).astype(np.int64), axis=0)
    rng = np.random.Generator(np.random.Philox(seed))
    pos = (sites + rng.uniform(-0.2, 0.2, size=sites.shape)) * dx
    n = len(pos)
    vel = rng.normal(scale=0.5, size=(n, 3))
    rho = 870.0 * (1.0 + 1e-3 * rng.normal(size=n))
    T = 313.0 + 5.0 * rng.normal(size=n)
    w.params["domain_min"] = [float(x) for x in pos.min(0) - 0.01]
    w.params["domain_max"] = [float(x) for x in pos.max(0) + 0.01]
    return w.params, pos.astype(np.float32), vel.astype(np.float32), rho.astype(np.float32), T.astype(np.float32)


def test_P3_momentum_conserved_without_walls():
    params, pos, vel, rho, T = _cloud_no_walls()
    o = make_oracle(params, pos, vel, rho, T)
    o.eval_rates()
    m = params["rho0"] * params["dx"] ** 3
    for name in ("ACC_P", "ACC_V", "ACC"):
        a = o.get(name)
        tot = np.abs((m * a).sum(axis=0)).max()
        ref = np.abs(m * a).sum()
        assert ref > 0 and tot < 1e-12 * ref, (name, tot, ref)
    # angular momentum of the central pressure force (along e_ij) is conserved too
    L = np.cross(o.get("POS"), m * o.get("ACC_P")).sum(axis=0)
    assert np.abs(L).max() < 1e-11 * np.abs(np.cross(o.get("POS"), m * o.get("ACC_P"))).sum()


def test_P4_thermal_energy_conserved_adiabatic():
    params, pos, vel, rho, T = _cloud_no_walls(seed=6)
    o = make_oracle(params, pos, vel, rho, T)
    o.eval_rates()
    m = params["rho0"] * params["dx"] ** 3
    q = m * params["cp_f"] * o.get("DT_DT")
    assert np.abs(q).sum() > 0 and abs(q.sum()) < 1e-12 * np.abs(q).sum()


def test_P4_energy_drift_1000_steps_closed_adiabatic_box():
    w = wl.still_tank(n=8, flags=wl.FLAG_THERMAL, dt_fixed=5.0, rebuild_every=1000)    # hydro off: heat only; dt < dt_T = 45 s (Eq. 26)
    for b in w.bodies:
        b.k_s = 0.0                                                                      # every wall adiabatic
    w = wl.perturb_state(w, T_scale=10.0)
    o = orc.Oracle.from_workload(w)
    E0 = o.get("T").sum()
    spread0 = o.get("T").std()
    o.step(1000)
    T = o.get("T")
    assert abs(T.sum() - E0) / E0 < 1e-12                   # uniform m, cp: sum T is the energy
    assert T.std() < 0.9 * spread0                          # and it does diffuse


# ------------------------------------------------------------------------------------------------
# P7 / P9  signs and factors: linear / quadratic fields on a lattice, limit h/dx -> large
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("hod,n,key,tol", [(1.3, 9, "c1_h1.3", 2e-6), (1.0, 7, "c1_h1.0", 2e-6), (3.0, 15, None, 2e-3)])
def test_P7_continuity_heat_viscous_on_polynomial_fields(hod, n, key, tol, golden):
    dx = 2e-3
    params, pos = lattice_cloud(n, dx, h_over_dx=hod, flags=wl.FLAGS_ALL_PHYSICS)
    c = 0.5 * (pos.min(0) + pos.max(0)).astype(np.float64)
    x = pos.astype(np.float64) - c
    c1 = golden("kernel_lattice_sums.txt")[key] if key else 1.0
    i = centre_index(pos)
    rho0, nu, k, cp = params["rho0"], params["nu"], params["k_f"], params["cp_f"]
    scale = 1.0 / dx      # keep fp32 inputs well conditioned

    # (a) v = A r with a full matrix A: drho/dt = -rho tr(A) c1   (Eq. 10 l.1; Riemann terms vanish for uniform p)
    A = np.array([[0.7, 0.2, -0.4], [0.1, -1.1, 0.3], [0.5, -0.6, 2.0]]) * scale * 1e-3
    o = make_oracle(params, pos, vel=(x @ A.T).astype(np.float32))
    o.eval_rates()
    got = o.get("DRHO_DT")[i]
    want = -rho0 * np.trace(A) * c1
    assert abs(got - want) < max(tol, 3e-6) * abs(rho0 * np.abs(A).sum()), (got, want)

    # (b) T = x^2: dT/dt = 2 alpha c1   (Eq. 22 with K_ii = 2k)
    T = (x[:, 0] * scale) ** 2
    o = make_oracle(params, pos, T=T.astype(np.float32))
    o.eval_rates()
    got = o.get("DT_DT")[i]
    want = 2.0 * k / (rho0 * cp) * scale ** 2 * c1
    assert abs(got - want) < max(tol, 3e-6) * abs(want), (got, want)

    # (c) v_x = y^2: viscous acceleration a_x = 2 nu c1, a_y = a_z = 0   (Eq. 10 l.2, second sum)
    v = np.zeros_like(x)
    v[:, 0] = (x[:, 1] * scale) ** 2 * 1e-3
    o = make_oracle(params, pos, vel=v.astype(np.float32))
    o.eval_rates()
    got = o.get("ACC_V")[i]
    want = 2.0 * nu * scale ** 2 * 1e-3 * c1
    assert abs(got[0] - want) < max(tol, 3e-6) * abs(want), (got, want)
    assert abs(got[1]) + abs(got[2]) < 1e-9 * abs(want)


def test_P9_linear_shear_has_no_viscous_force_inside():
    dx = 2e-3
    params, pos = lattice_cloud(9, dx, flags=wl.FLAGS_ALL_PHYSICS)
    x = pos.astype(np.float64)
    v = np.zeros_like(x)
    v[:, 0] = 3.0 * x[:, 1] / dx * 1e-2
    o = make_oracle(params, pos, vel=v.astype(np.float32))
    o.eval_rates()
    a = o.get("ACC_V")
    i = centre_index(pos)
    assert np.abs(a[i]).max() < 5e-6 * np.abs(a).max()       # inputs are fp32: cancellation to input rounding
    assert np.abs(a).max() > 0          # the truncated surface particles do feel a force


def test_P7_uniform_pressure_gives_no_force_inside():
    params, pos = lattice_cloud(9, 2e-3, flags=wl.FLAGS_ALL_PHYSICS)
    o = make_oracle(params, pos, rho=np.full(len(pos), 871.0, np.float32))
    o.eval_rates()
    a = o.get("ACC_P")
    assert np.abs(a[centre_index(pos)]).max() < 5e-6 * np.abs(a).max()      # fp32 input positions
    # surface particles are pushed OUTWARD by a positive pressure (sign of -grad p)
    c = 0.5 * (pos.min(0) + pos.max(0))
    j = int(np.argmax(pos[:, 0]))
    assert a[j, 0] > 0 and (pos[j, 0] - c[0]) > 0


def test_P7_linear_pressure_field_gives_minus_grad_p_over_rho(golden):
    dx = 2e-3
    c1 = golden("kernel_lattice_sums.txt")["c1_h1.3"]
    params, pos = lattice_cloud(9, dx, flags=wl.FLAGS_ALL_PHYSICS)
    c0, rho0 = params["c0"], params["rho0"]
    x = pos.astype(np.float64)
    gp = 500.0                                           # dp/dz in Pa/m
    rho = rho0 + gp * (x[:, 2] - x[:, 2].mean()) / c0 ** 2
    o = make_oracle(params, pos, rho=rho.astype(np.float32))
    o.eval_rates()
    a = o.get("ACC_P")[centre_index(pos)]
    # -(2/rho) sum V p* gradW  ->  -(1/rho) grad p  (times the lattice constant c1); rho ~ rho0 to 1e-6
    assert abs(a[2] + gp / rho0 * c1) < 2e-3 * gp / rho0, a
    assert abs(a[0]) + abs(a[1]) < 1e-6 * gp / rho0


# ------------------------------------------------------------------------------------------------
# P8  Riemann solver: dissipation only in compression, signs of Eq. 13 (reading R3)
# ------------------------------------------------------------------------------------------------
def test_P8_riemann_limiter_and_means():
    c0 = 20.0
    # receding pair: U_L < U_R -> beta = 0, p* = density-weighted mean
    us, ps, ub = orc.riemann(870.0, -1.0, 100.0, 880.0, 1.0, 300.0, c0)
    assert ps == pytest.approx((870.0 * 300.0 + 880.0 * 100.0) / 1750.0, rel=1e-14)
    assert ub == pytest.approx((870.0 * -1.0 + 880.0 * 1.0) / 1750.0, rel=1e-14)
    assert us == pytest.approx(ub + (100.0 - 300.0) / (c0 * 1750.0), rel=1e-14)
    # approaching pair, small closing speed: beta = 3 dU
    us, ps, _ = orc.riemann(870.0, 0.5, 0.0, 870.0, -0.5, 0.0, c0)
    assert ps == pytest.approx(870.0 * 870.0 * 3.0 * 1.0 * 1.0 / 1740.0, rel=1e-14)
    # approaching pair, large closing speed: beta capped at c0
    us, ps, _ = orc.riemann(870.0, 10.0, 0.0, 870.0, -10.0, 0.0, c0)
    assert ps == pytest.approx(870.0 * 870.0 * c0 * 20.0 / 1740.0, rel=1e-14)


def _two_particles(rho_i, rho_j, v_i, v_j, sep=1.0):
    dx = 2e-3
    params = wl.default_params(dx, g=[0.0, 0.0, 0.0], flags=wl.FLAGS_ALL_PHYSICS)
    params["domain_min"] = [-0.02] * 3
    params["domain_max"] = [0.02] * 3
    pos = np.array([[0.0, 0.0, 0.0], [sep * dx, 0.0, 0.0]], np.float32)
    vel = np.array([v_i, v_j], np.float32)
    rho = np.array([rho_i, rho_j], np.float32)
    o = make_oracle(params, pos, vel, rho)
    o.eval_rates()
    return params, o


def test_P8_pressure_difference_at_rest_lowers_density_of_high_side():
    _, o = _two_particles(871.0, 870.0, [0, 0, 0], [0, 0, 0])
    d = o.get("DRHO_DT")
    assert d[0] < 0 < d[1]                                  # reading R3: relaxation, not anti-diffusion
    a = o.get("ACC_P")
    assert a[0, 0] < 0 < a[1, 0]                            # positive p* pushes the pair apart (i sits at x=0)


def test_P8_approach_raises_density_and_repels():
    _, o = _two_particles(870.0, 870.0, [0.3, 0, 0], [-0.3, 0, 0])
    d = o.get("DRHO_DT")
    assert d[0] > 0 and d[1] > 0 and d[0] == pytest.approx(d[1], rel=1e-12)
    a = o.get("ACC_P")
    assert a[0, 0] < 0 < a[1, 0]                            # dissipative p* opposes the approach
    _, o2 = _two_particles(870.0, 870.0, [-0.3, 0, 0], [0.3, 0, 0])
    assert np.abs(o2.get("ACC_P")).max() == 0.0             # receding: beta = 0 and p = 0 -> no force
    assert (o2.get("DRHO_DT") < 0).all()


def test_P8_single_pair_hand_value():
    # one pair, separation s = 1.5 dx along x, at rest, rho_i = 871, rho_j = 870 (c0 = 20, h = 1.3 dx)
    params, o = _two_particles(871.0, 870.0, [0, 0, 0], [0, 0, 0], sep=1.5)
    dx, h, c0, rho0 = params["dx"], params["h"], params["c0"], params["rho0"]
    s = float(np.float32(1.5 * dx))
    q = s / h
    dW = -(5.0 * 21.0 / (16.0 * math.pi * h ** 4)) * q * (1 - q / 2) ** 3
    m = rho0 * dx ** 3
    p_i, p_j = c0 * c0 * 1.0, 0.0
    pstar = (871.0 * p_j + 870.0 * p_i) / 1741.0
    # e_ij = (r_i - r_j)/|..| = -x_hat for particle i at the origin
    ax_i = -(2.0 / m) * (m / 871.0) * (m / 870.0) * pstar * (-1.0) * dW
    assert o.get("ACC_P")[0, 0] == pytest.approx(ax_i, rel=1e-12)
    # continuity: (v_i - v*) . e W' = (U* - Ubar) W' = (p_i - p_j)/(c0 (rho_i+rho_j)) W'
    drho_i = 2.0 * 871.0 * (m / 870.0) * (p_i - p_j) / (c0 * 1741.0) * dW
    assert o.get("DRHO_DT")[0] == pytest.approx(drho_i, rel=1e-12)


# ------------------------------------------------------------------------------------------------
# P5  wall model + gravity: hydrostatic tank stays at rest with p = rho0 g depth
# ------------------------------------------------------------------------------------------------
@pytest.mark.timeout(300)
def test_P5_hydrostatic_tank_stays_still():
    w = wl.still_tank(n=10, fill=0.8, jitter=0.0,
                      flags=wl.FLAGS_ALL_PHYSICS | wl.FLAG_FREE_SURFACE)      # re-init off (R12)
    p = w.params
    g, rho0, c0, dx = 9.81, p["rho0"], p["c0"], p["dx"]
    z_surface = 8 * dx
    depth = z_surface - w.pos_f[:, 2].astype(np.float64)
    w.rho_f = (rho0 + rho0 * g * depth / c0 ** 2).astype(np.float32)
    o = orc.Oracle.from_workload(w, rebuild_every=1)
    o.step(600)
    v = np.linalg.norm(o.get("VEL"), axis=1)
    H = 8 * dx
    assert v.max() < 0.02 * math.sqrt(g * H)                # SURVEY probe: 2e-3 m/s vs sqrt(gH) = 0.4
    pos = o.get("POS")
    depth = z_surface - pos[:, 2]
    bulk = depth > 2.5 * dx
    err = np.abs(o.get("P")[bulk] - rho0 * g * depth[bulk])
    assert err.max() < 0.05 * rho0 * g * H, err.max() / (rho0 * g * H)
    assert np.abs(pos - w.pos_f).max() < 0.05 * dx


# ------------------------------------------------------------------------------------------------
# P6  conduction across a material discontinuity: PAPER.md section 3.2 / Table 3 vs the erfc solution
# ------------------------------------------------------------------------------------------------
@pytest.mark.timeout(300)
def test_P6_two_slab_conduction_matches_analytic(golden):
    g = golden("two_slab_conduction.txt")
    dx = g["dx"]
    nx, ny = 80, 13
    sites = np.stack(np.meshgrid(np.arange(nx), np.arange(ny), np.arange(ny), indexing="ij"), -1).reshape(-1, 3)
    pos = ((sites + 0.5) * dx).astype(np.float32)
    left = pos[:, 0] < g["x_iface"]
    params = wl.default_params(dx, h=g["h_over_dx"] * dx, flags=wl.FLAG_THERMAL, rho0=1000.0, g=[0, 0, 0],
                               dt_fixed=0.01, rebuild_every=10 ** 6, k_f=1.0, cp_f=1.0)
    params["domain_min"] = [-0.05] * 3
    params["domain_max"] = [1.05, 0.25, 0.25]
    rho = np.where(left, g["rho_l"], g["rho_r"])
    o = make_oracle(params, pos, rho=rho.astype(np.float32), T=np.where(left, g["T_left0"], g["T_right0"]).astype(np.float32))
    o.set_materials(mass=rho * dx ** 3, k=np.where(left, g["k_l"], g["k_r"]), cp=np.where(left, g["cp_l"], g["cp_r"]))
    E0 = (rho * o.get("T")).sum()
    o.step(int(round(g["t_end"] / 0.01)))
    T = o.get("T")
    assert abs((rho * T).sum() - E0) < 1e-12 * E0

    # closed form for two semi-infinite bodies in contact (textbook), penetration << 0.5
    el, er = math.sqrt(g["k_l"] * g["rho_l"] * g["cp_l"]), math.sqrt(g["k_r"] * g["rho_r"] * g["cp_r"])
    Tc = er / (el + er)
    assert Tc == pytest.approx(g["T_contact"], abs=1e-9)
    assert g["alpha_l"] == pytest.approx(g["k_l"] / (g["rho_l"] * g["cp_l"])) and g["alpha_r"] == pytest.approx(g["k_r"] / (g["rho_r"] * g["cp_r"]))
    x = pos[:, 0].astype(np.float64)
    t = g["t_end"]
    ana = np.where(left,
                   Tc * special.erfc(np.abs(x - 0.5) / (2 * math.sqrt(g["alpha_l"] * t))),
                   1.0 - (1.0 - Tc) * special.erfc(np.abs(x - 0.5) / (2 * math.sqrt(g["alpha_r"] * t))))
    line = (sites[:, 1] == ny // 2) & (sites[:, 2] == ny // 2)
    err = np.abs(T[line] - ana[line])
    assert err.max() < 1.0e-2, err.max()
    # the discontinuity in the gradient is captured: flux continuity k_l dT/dx|- = k_r dT/dx|+ (within 15 %)
    xs, Ts = x[line], T[line]
    order = np.argsort(xs); xs, Ts = xs[order], Ts[order]
    il = np.searchsorted(xs, 0.5) - 1
    gl = (Ts[il - 1] - Ts[il - 3]) / (xs[il - 1] - xs[il - 3])
    gr = (Ts[il + 4] - Ts[il + 2]) / (xs[il + 4] - xs[il + 2])
    assert g["k_l"] * gl == pytest.approx(g["k_r"] * gr, rel=0.15)


# ------------------------------------------------------------------------------------------------
# P10  wall kinematics: rigid rotation, closed form
# ------------------------------------------------------------------------------------------------
def test_P10_rigid_rotation_matches_closed_form():
    w = wl.still_tank(n=6, flags=wl.FLAGS_ALL_PHYSICS, dt_fixed=1e-4, rebuild_every=1)
    origin = np.array([0.006, 0.005, 0.004])
    w.bodies[1] = wl.Body(k_s=0.13, origin=tuple(origin), axis=(0.0, 0.0, 2.0), omega=300.0)   # axis gets normalised
    o = orc.Oracle.from_workload(w)
    o.step(11)                                   # walls were placed at t = 10 dt (last rebuild)
    th = 300.0 * 10 * 1e-4
    sel = w.body_w == 1
    ref = w.pos_w[sel].astype(np.float64) - origin
    c, s = math.cos(th), math.sin(th)
    want = np.stack([c * ref[:, 0] - s * ref[:, 1], s * ref[:, 0] + c * ref[:, 1], ref[:, 2]], 1) + origin
    got = o.get("WALL_POS")
    # R21: the closed-form rotation, rounded once to fp32 (wall particle state is fp32)
    np.testing.assert_allclose(got[sel], want, rtol=0, atol=1e-9)
    assert np.mean(got[sel] == want.astype(np.float32).astype(np.float64)) > 0.999
    assert np.array_equal(got[sel], got[sel].astype(np.float32).astype(np.float64))
    np.testing.assert_allclose(got[~sel], w.pos_w[~sel].astype(np.float64), rtol=0, atol=0)
    nref = w.normal_w[sel].astype(np.float64)
    nwant = np.stack([c * nref[:, 0] - s * nref[:, 1], s * nref[:, 0] + c * nref[:, 1], nref[:, 2]], 1)
    np.testing.assert_allclose(o.get("WALL_NORMAL")[sel], nwant, rtol=0, atol=1e-7)
    np.testing.assert_allclose(np.linalg.norm(got[sel] - origin, axis=1), np.linalg.norm(ref, axis=1), rtol=2e-6)


def test_P10_clock_moved_to_t_places_bodies_at_omega_t():
    """shared-state steps (tests/test_gpu_full_size.py): set_time(t) then a rebuild = closed-form rotation by omega t."""
    w = wl.still_tank(n=6, flags=wl.FLAGS_ALL_PHYSICS, dt_fixed=1e-4, rebuild_every=1)
    origin = np.array([0.006, 0.005, 0.004])
    w.bodies[1] = wl.Body(k_s=0.13, origin=tuple(origin), axis=(0.0, 0.0, 1.0), omega=300.0)
    o = orc.Oracle.from_workload(w)
    t = 3.7e-3
    o.set_time(t)
    o.rebuild()
    sel = w.body_w == 1
    ref = w.pos_w[sel].astype(np.float64) - origin
    c, s = math.cos(300.0 * t), math.sin(300.0 * t)
    want = np.stack([c * ref[:, 0] - s * ref[:, 1], s * ref[:, 0] + c * ref[:, 1], ref[:, 2]], 1) + origin
    np.testing.assert_allclose(o.get("WALL_POS")[sel], want, rtol=0, atol=1e-9)
    assert np.mean(o.get("WALL_POS")[sel] == want.astype(np.float32).astype(np.float64)) > 0.999
    assert abs(o.stats()["t"] - t) == 0.0


def test_P10_general_axis_preserves_distances_and_axis_component():
    w = wl.still_tank(n=6, flags=wl.FLAGS_ALL_PHYSICS, dt_fixed=1e-4, rebuild_every=1)
    axis = np.array([1.0, 2.0, -0.5]); axis /= np.linalg.norm(axis)
    origin = np.array([0.001, 0.002, 0.003])
    w.bodies[0] = wl.Body(k_s=0.0, origin=tuple(origin), axis=tuple(axis), omega=-450.0)
    o = orc.Oracle.from_workload(w)
    o.step(8)
    sel = w.body_w == 0
    ref = w.pos_w[sel].astype(np.float64) - origin
    got = o.get("WALL_POS")[sel] - origin
    np.testing.assert_allclose(np.linalg.norm(got, axis=1), np.linalg.norm(ref, axis=1), rtol=2e-6)
    np.testing.assert_allclose(got @ axis, ref @ axis, rtol=0, atol=2e-9)
    th = -450.0 * 7 * 1e-4
    perp_r = ref - np.outer(ref @ axis, axis)
    perp_g = got - np.outer(got @ axis, axis)
    cosang = (perp_r * perp_g).sum(1) / (np.linalg.norm(perp_r, axis=1) * np.linalg.norm(perp_g, axis=1))
    np.testing.assert_allclose(cosang, math.cos(th), atol=1e-6)
    sinang = np.cross(perp_r, perp_g) @ axis / (np.linalg.norm(perp_r, axis=1) * np.linalg.norm(perp_g, axis=1))
    np.testing.assert_allclose(sinang, math.sin(th), atol=1e-6)


# ------------------------------------------------------------------------------------------------
# P11  torque: action-reaction, single-pair hand value
# ------------------------------------------------------------------------------------------------
def test_P11_wall_forces_balance_fluid_accelerations_and_torque_is_their_moment():
    w = wl.perturb_state(wl.still_tank(n=8, flags=wl.FLAGS_ALL_PHYSICS))
    origin = np.array([0.004, 0.003, 0.011])
    w.bodies[1] = wl.Body(k_s=0.13, origin=tuple(origin), axis=(0.0, 1.0, 0.0), omega=120.0)
    o = orc.Oracle.from_workload(w)
    o.eval_rates()
    m = w.params["rho0"] * w.params["dx"] ** 3
    F = o.get("WALL_FORCE")
    a_wall = o.get("ACC_WP") + o.get("ACC_WV")
    np.testing.assert_allclose(F.sum(axis=0), -(m * a_wall).sum(axis=0), rtol=1e-10, atol=1e-14 * np.abs(F).sum())
    for b in (0, 1):
        sel = w.body_w == b
        ob = np.array(w.bodies[b].origin)
        tau = np.cross(o.get("WALL_POS")[sel] - ob, F[sel]).sum(axis=0)
        got, axial = o.torque(b)
        np.testing.assert_allclose(got, tau, rtol=1e-10, atol=1e-18)
        assert axial == pytest.approx(float(tau @ np.array(w.bodies[b].axis)), rel=1e-10, abs=1e-18)
    assert np.abs(o.torque(1)[0]).max() > 0


def test_P11_single_fluid_wall_pair_hand_value():
    dx = 2e-3
    params = wl.default_params(dx, g=[0.0, 0.0, 0.0], flags=wl.FLAGS_ALL_PHYSICS)
    params["domain_min"] = [-0.02] * 3
    params["domain_max"] = [0.02] * 3
    h, c0, rho0, nu = params["h"], params["c0"], params["rho0"], params["nu"]
    pos = np.array([[0.0, 0.0, float(np.float32(1.2 * dx))]], np.float32)    # fluid above the wall particle
    vel = np.array([[0.4, 0.0, 0.0]], np.float32)
    rho = np.array([871.0], np.float32)
    walls = (np.zeros((1, 3), np.float32), np.array([[0, 0, 1]], np.float32), np.array([1], np.int32), np.array([353.0], np.float32))
    bodies = [wl.Body(), wl.Body(k_s=0.13, origin=(0.0, -0.01, 0.0), axis=(0, 1, 0), omega=0.0)]
    o = make_oracle(params, pos, vel, rho, np.array([313.0], np.float32), walls=walls, bodies=bodies)
    o.eval_rates()
    s = float(pos[0, 2]); q = s / h
    dW = -(5.0 * 21.0 / (16.0 * math.pi * h ** 4)) * q * (1 - q / 2) ** 3
    m, Vw = rho0 * dx ** 3, dx ** 3
    p_i = c0 * c0 * 1.0
    # g = 0: P_R = P_L, rho_R = rho_L -> p* = p_i (Eq. 17, 19); e_iw = +z
    a_p = -(2.0 / m) * (m / 871.0) * Vw * p_i * dW                    # along +z: wall pushes fluid away
    a_v = (2.0 / m) * (m / 871.0) * Vw * (rho0 * nu) * float(np.float32(0.4)) / s * dW   # along x: opposes the slip
    assert a_p > 0 > a_v
    np.testing.assert_allclose(o.get("ACC_WP")[0], [0, 0, a_p], rtol=1e-12, atol=0)
    np.testing.assert_allclose(o.get("ACC_WV")[0], [a_v, 0, 0], rtol=1e-12, atol=0)
    F = -m * np.array([a_v, 0.0, a_p])
    lever = np.array([0.0, 0.01, 0.0])                                # r_w - o_b
    tau, axial = o.torque(1)
    np.testing.assert_allclose(tau, np.cross(lever, F), rtol=1e-12)
    assert axial == pytest.approx(0.0, abs=1e-30)
    # wall continuity term (R6): still wall, fluid sliding tangentially -> U_L = 0 -> no density change
    assert o.get("DRHO_DT")[0] == pytest.approx(0.0, abs=1e-9)
    # heat: dT/dt = V_w K (T_i - T_w)/r W' / (rho cp), K = 4 k k /(2k) = 2k  -> warms up (T_w > T_i)
    want = Vw * 2.0 * 0.13 * (313.0 - 353.0) / s * dW / (871.0 * params["cp_f"])
    assert want > 0 and o.get("DT_DT")[0] == pytest.approx(want, rel=1e-12)


def test_P11_wall_normal_approach_compresses_fluid():
    dx = 2e-3
    params = wl.default_params(dx, g=[0.0, 0.0, 0.0], flags=wl.FLAGS_ALL_PHYSICS)
    params["domain_min"] = [-0.02] * 3
    params["domain_max"] = [0.02] * 3
    pos = np.array([[0.0, 0.0, 1.2 * dx]], np.float32)
    walls = (np.zeros((1, 3), np.float32), np.array([[0, 0, 1]], np.float32), np.array([0], np.int32), np.array([313.0], np.float32))
    for vz, sign in ((-0.5, +1), (+0.5, -1)):
        o = make_oracle(params, pos, np.array([[0, 0, vz]], np.float32), None, walls=walls, bodies=[wl.Body()])
        o.eval_rates()
        assert np.sign(o.get("DRHO_DT")[0]) == sign
    # a wall moving with the fluid (same normal velocity) leaves the density alone: U_R = -U_L + 2 u_w = U_L
    bodies = [wl.Body(origin=(0.0, 1.0, 0.0), axis=(1, 0, 0), omega=0.5)]     # v_w = omega x (r_w - o) = (0,0,-0.5)... sign below
    o = make_oracle(params, pos, np.array([[0, 0, 0.5]], np.float32), None, walls=walls, bodies=bodies)
    o.eval_rates()
    # omega e_x x (0,-1,0) = (0,0,-omega): choose fluid velocity equal to it
    o2 = make_oracle(params, pos, np.array([[0, 0, -0.5]], np.float32), None, walls=walls, bodies=bodies)
    o2.eval_rates()
    assert abs(o2.get("DRHO_DT")[0]) < 1e-9 < abs(o.get("DRHO_DT")[0])


# ------------------------------------------------------------------------------------------------
# P12  time-step criteria, Eq. 25-26
# ------------------------------------------------------------------------------------------------
def test_P12_dt_criteria(golden):
    g = golden("dt_criteria.txt")
    h = 2.6e-3
    assert orc.dt_ac(h, 20.0, 0.0) == pytest.approx(g["dt_ac_rest"], rel=1e-6)
    assert orc.dt_ac(h, 20.0, 2.0) == pytest.approx(g["dt_ac_v2"], rel=1e-6)
    assert orc.dt_ad(h, 2.0, 1e-4) == pytest.approx(g["dt_ad_v2"], rel=1e-6)
    assert orc.dt_ad(h, 1e-9, 1e-4) == pytest.approx(g["dt_ad_visc"], rel=1e-6)
    assert orc.dt_thermal(870.0, 2000.0, h, 0.13) == pytest.approx(g["dt_T_oil"], rel=1e-3)
    assert orc.dt_thermal(7850.0, 460.0, h, 45.0) == pytest.approx(g["dt_T_steel"], rel=1e-3)


def test_P12_dual_criteria_clock():
    w = wl.still_tank(n=6, flags=wl.FLAGS_ALL_PHYSICS | wl.FLAG_DUAL_CRITERIA)     # adaptive dt, dt_ad rule
    o = orc.Oracle.from_workload(w)
    o.step(12)
    s = o.stats()
    # at rest with u_ref = c0/10: dt_ad/dt_ac = 0.25 (c0+u)/(0.6 u) = 4.58 -> 5 acoustic steps per rebuild,
    # the last one truncated so that the advection step is hit exactly (R14)
    assert s["rebuilds"] == 3 and s["steps"] == 12
    assert s["dt_ad"] == pytest.approx(3.25e-4, rel=1e-3)
    assert s["t"] == pytest.approx(2 * s["dt_ad"] + 2 * 7.0909e-5, rel=1e-3)


# ------------------------------------------------------------------------------------------------
# Contact factor, Eq. 24, reading R22
# ------------------------------------------------------------------------------------------------
def _wall_layer_and_interior(w, n, dx):
    """innermost wall layer (half a spacing outside the cavity) away from the cavity's edges, by axis-aligned geometry"""
    p = w.pos_w.astype(np.float64) / dx                      # cavity spans [0, n] in lattice units
    out = np.maximum(np.maximum(-p, p - n), 0.0)             # distance outside the cavity per axis
    depth = out.max(axis=1)
    n_out = (out > 0).sum(axis=1)
    inner = (np.abs(depth - 0.5) < 1e-3) & (n_out == 1)
    inside = ((p > 3.0) & (p < n - 3.0)).sum(axis=1) == 2     # the two in-plane coordinates far from the edges
    return inner & inside


def test_contact_factor_fully_immersed_lattice_is_one():
    n, dx = 10, 2.0e-3
    w = wl.still_tank(n=n, dx=dx, jitter=0.0)
    o = orc.Oracle.from_workload(w)
    o.rebuild()
    z = o.contact_factor()
    sel = _wall_layer_and_interior(w, n, dx)
    assert sel.sum() > 50
    np.testing.assert_allclose(z[sel], 1.0, rtol=0, atol=5e-6)      # the fp32 lattice coordinates are rounded
    assert (z >= 0).all() and z.max() <= 1.0 + 5e-5       # particles with a small open part amplify the rounding
    # second and third layer: part of their support lies outside the 3-layer wall, where no lubricant is
    p = w.pos_w.astype(np.float64) / dx
    depth = np.maximum(np.maximum(-p, p - n), 0.0).max(axis=1)
    assert z[np.abs(depth - 1.5) < 1e-3].max() < 1.0 and z[np.abs(depth - 2.5) < 1e-3].max() < z[np.abs(depth - 1.5) < 1e-3].max()


def test_contact_factor_dry_wall_is_zero_and_grows_with_fill():
    n, dx = 10, 2.0e-3
    means = []
    for fill in (0.3, 0.6, 1.0):
        w = wl.still_tank(n=n, dx=dx, jitter=0.0, fill=fill)
        o = orc.Oracle.from_workload(w)
        o.rebuild()
        z = o.contact_factor()
        p = w.pos_w.astype(np.float64) / dx
        top = p[:, 2] > n * fill + 2.6 + 1e-6                # wall particles more than a support radius above the surface
        if fill < 1.0:
            assert top.any() and np.all(z[top] == 0.0)
        # innermost layer of the x_min face over the cavity's whole height, away from the y edges
        side = (np.abs(p[:, 0] + 0.5) < 1e-3) & (p[:, 1] > 3) & (p[:, 1] < n - 3) & (p[:, 2] > 0) & (p[:, 2] < n)
        means.append(z[side].mean())
    assert means[0] < means[1] < means[2] and abs(means[2] - 1.0) < 5e-6
    assert abs(means[0] - 0.3) < 0.08 and abs(means[1] - 0.6) < 0.08    # wetted fraction of the face


def test_contact_factor_equals_brute_force_definition():
    """tiny jittered tank with a free surface and non-uniform densities: Eq. 24 / R22 evaluated pair by pair in numpy"""
    n, dx = 6, 2.0e-3
    w = wl.perturb_state(wl.still_tank(n=n, dx=dx, fill=0.5), rho_rel=2e-2)
    o = orc.Oracle.from_workload(w, flags=int(w.params["flags"]) & ~wl.FLAG_DENSITY_REINIT)
    o.rebuild()
    z = o.contact_factor()
    h = float(w.params["h"])
    rf, rw = w.pos_f.astype(np.float64), w.pos_w.astype(np.float64)
    Vf = float(w.params["rho0"]) * dx ** 3 / w.rho_f.astype(np.float64)

    def Wk(r):
        q = r / h
        return np.where(q < 2.0, 21.0 / (16.0 * np.pi * h ** 3) * (1 - 0.5 * q) ** 4 * (1 + 2 * q), 0.0)
    d_wf = np.linalg.norm(rw[:, None, :] - rf[None, :, :], axis=2)
    d_ww = np.linalg.norm(rw[:, None, :] - rw[None, :, :], axis=2)
    num = (Wk(d_wf) * Vf[None, :]).sum(axis=1)
    full = dx ** 3 * orc.sigma0(dx, h) - dx ** 3 * Wk(d_ww).sum(axis=1)
    want = np.where(full > 1e-3 * dx ** 3 * orc.sigma0(dx, h), num / np.where(full > 0, full, 1.0), 0.0)
    np.testing.assert_allclose(z, want, rtol=1e-11, atol=1e-13)
    assert 0.2 < z.max() <= 1.1


# ------------------------------------------------------------------------------------------------
# Evolving solid temperature, Eq. 20, reading R23
# ------------------------------------------------------------------------------------------------
def _evolving_tank(n=8, modes=(1, 1)):
    w = wl.perturb_state(wl.still_tank(n=n, flags=wl.FLAGS_ALL_PHYSICS & ~wl.FLAG_DENSITY_REINIT), T_scale=8.0)
    w.bodies[0] = wl.Body(k_s=45.0, rho_s=7850.0, cp_s=460.0, thermal_mode=modes[0])
    w.bodies[1] = wl.Body(k_s=0.5, rho_s=2700.0, cp_s=900.0, thermal_mode=modes[1])
    rng = np.random.default_rng(5)
    return dataclasses_replace(w, T_w=(330.0 + 10.0 * rng.normal(size=w.n_w)).astype(np.float32))


def dataclasses_replace(w, **kw):
    import dataclasses
    return dataclasses.replace(w, **kw)


def _total_energy(o, w):
    dx = float(w.params["dx"])
    m = float(w.params["rho0"]) * dx ** 3
    cs = np.array([w.bodies[b].rho_s * w.bodies[b].cp_s for b in w.body_w]) * dx ** 3
    return m * float(w.params["cp_f"]) * o.get("T").sum() + (cs * o.get("WALL_T")).sum(), cs


def test_R23_fluid_solid_energy_is_conserved():
    w = _evolving_tank()
    o = orc.Oracle.from_workload(w, dt_fixed=2e-5, rebuild_every=5)
    o.eval_rates()
    dx = float(w.params["dx"])
    m = float(w.params["rho0"]) * dx ** 3
    _, cs = _total_energy(o, w)
    f, s = m * float(w.params["cp_f"]) * o.get("DT_DT"), cs * o.get("WALL_DT_DT")
    assert np.abs(s).max() > 0 and np.abs(f).max() > 0
    assert abs(f.sum() + s.sum()) <= 1e-12 * (np.abs(f).sum() + np.abs(s).sum())     # antisymmetric pair exchange
    E0, _ = _total_energy(o, w)
    o.step(200)
    E1, _ = _total_energy(o, w)
    assert abs(E1 - E0) <= 1e-12 * abs(E0)
    assert np.abs(o.get("WALL_T") - w.T_w).max() > 1e-4                              # the solid did change


def test_R23_uniform_temperature_is_stationary_and_held_bodies_stay():
    w = _evolving_tank(modes=(1, 0))
    wu = dataclasses_replace(w, T_f=np.full(w.n_f, 320.0, np.float32), T_w=np.full(w.n_w, 320.0, np.float32))
    o = orc.Oracle.from_workload(wu, dt_fixed=2e-5, rebuild_every=5)
    o.eval_rates()
    assert np.all(o.get("WALL_DT_DT") == 0.0) and np.all(o.get("DT_DT") == 0.0)
    o2 = orc.Oracle.from_workload(w, dt_fixed=2e-5, rebuild_every=5)
    o2.step(20)
    held = w.body_w == 1
    assert np.array_equal(o2.get("WALL_T")[held], w.T_w[held].astype(np.float64))    # mode 0: R10
    assert np.all(o2.get("WALL_DT_DT")[held] == 0.0)
    assert np.abs(o2.get("WALL_T")[~held] - w.T_w[~held]).max() > 0


@pytest.mark.timeout(300)
def test_R23_fluid_solid_slab_conduction_matches_analytic(golden):
    """Table 3's two-slab benchmark with the right slab made of SOLID particles whose temperature
    evolves: the same erfc solution of two semi-infinite bodies in contact"""
    g = golden("two_slab_conduction.txt")
    dx = g["dx"]
    nx, ny = 80, 13
    sites = np.stack(np.meshgrid(np.arange(nx), np.arange(ny), np.arange(ny), indexing="ij"), -1).reshape(-1, 3)
    pos = ((sites + 0.5) * dx).astype(np.float32)
    left = pos[:, 0] < g["x_iface"]
    params = wl.default_params(dx, h=g["h_over_dx"] * dx, flags=wl.FLAG_THERMAL, rho0=g["rho_l"], g=[0, 0, 0],
                               dt_fixed=0.01, rebuild_every=10 ** 6, k_f=g["k_l"], cp_f=g["cp_l"])
    params["domain_min"] = [-0.05] * 3
    params["domain_max"] = [1.05, 0.25, 0.25]
    bodies = [wl.Body(k_s=g["k_r"], rho_s=g["rho_r"], cp_s=g["cp_r"], thermal_mode=1)]
    nl, nr = int(left.sum()), int((~left).sum())
    nrm = np.tile(np.array([[-1.0, 0.0, 0.0]], np.float32), (nr, 1))
    o = make_oracle(params, pos[left], rho=np.full(nl, g["rho_l"], np.float32), T=np.full(nl, g["T_left0"], np.float32),
                    walls=(pos[~left], nrm, np.zeros(nr, np.int32), np.full(nr, g["T_right0"], np.float32)), bodies=bodies)
    E0 = g["rho_l"] * g["cp_l"] * o.get("T").sum() + g["rho_r"] * g["cp_r"] * nr * g["T_right0"]
    o.step(int(round(g["t_end"] / 0.01)))
    Tf, Ts = o.get("T"), o.get("WALL_T")
    assert abs(g["rho_l"] * g["cp_l"] * Tf.sum() + g["rho_r"] * g["cp_r"] * Ts.sum() - E0) < 1e-12 * E0
    el, er = math.sqrt(g["k_l"] * g["rho_l"] * g["cp_l"]), math.sqrt(g["k_r"] * g["rho_r"] * g["cp_r"])
    Tc = er / (el + er)
    assert Tc == pytest.approx(g["T_contact"], abs=1e-9)
    t = g["t_end"]
    xl, xr = pos[left][:, 0].astype(np.float64), pos[~left][:, 0].astype(np.float64)
    ana_l = Tc * special.erfc(np.abs(xl - 0.5) / (2 * math.sqrt(g["alpha_l"] * t)))
    ana_r = 1.0 - (1.0 - Tc) * special.erfc(np.abs(xr - 0.5) / (2 * math.sqrt(g["alpha_r"] * t)))
    line_l = (sites[left][:, 1] == ny // 2) & (sites[left][:, 2] == ny // 2)
    line_r = (sites[~left][:, 1] == ny // 2) & (sites[~left][:, 2] == ny // 2)
    assert np.abs(Tf[line_l] - ana_l[line_l]).max() < 1.0e-2
    assert np.abs(Ts[line_r] - ana_r[line_r]).max() < 1.0e-2
    assert Ts[line_r].min() < 0.9                              # the solid slab did cool near the interface


# ------------------------------------------------------------------------------------------------
# Particle relaxation, Eq. 6-9, reading R24
# ------------------------------------------------------------------------------------------------
def test_relaxation_two_particles_hand_value():
    """Eq. 7-9 by hand: F = -(2/m) V^2 p0 W'(r) e_ij (repulsive), dt = 0.25 sqrt(h/|F|), so each particle moves
    F dt^2 / 2 = h / 32 away from the other, whatever p0"""
    dx = 2.0e-3
    params = wl.default_params(dx, flags=wl.FLAGS_ALL_PHYSICS)
    params["domain_min"] = [0.0] * 3
    params["domain_max"] = [0.05] * 3
    h = float(params["h"])
    pos = np.array([[0.02, 0.02, 0.02], [0.02 + 1.2 * dx, 0.02, 0.02]], np.float32)
    for p0 in (1.0, 250.0):
        o = make_oracle(params, pos, rho=np.full(2, 870.0, np.float32))
        r = float(pos[1, 0]) - float(pos[0, 0])
        fmax = o.relax(1, p0)
        assert fmax == pytest.approx(2.0 / (870.0 * dx ** 3) * dx ** 6 * p0 * abs(orc.dWdr(r, h)), rel=1e-12)
        d = o.get("POS") - pos.astype(np.float64)
        np.testing.assert_allclose(d[0], [-h / 32.0, 0.0, 0.0], rtol=1e-12, atol=1e-18)
        np.testing.assert_allclose(d[1], [+h / 32.0, 0.0, 0.0], rtol=1e-12, atol=1e-18)


def test_relaxation_lattice_is_a_fixed_point_and_jitter_relaxes():
    n, dx = 8, 2.0e-3
    w0 = wl.still_tank(n=n, dx=dx, jitter=0.0)
    o = orc.Oracle.from_workload(w0)
    fmax = o.relax(1, 100.0)
    p = w0.pos_f.astype(np.float64) / dx
    inner = ((p > 2.7) & (p < n - 2.7)).all(axis=1)          # support inside the filled, walled cavity
    # on the full lattice (fluid + 3 wall layers) the pair forces cancel by symmetry: what is left is the fp32
    # rounding of the coordinates, ~1e-6 of one pair's force (Eq. 8-9 then scale the largest move to h/32 anyway)
    F1 = 2.0 / (870.0 * dx ** 3) * dx ** 6 * 100.0 * abs(orc.dWdr(dx, 1.3 * dx))
    assert fmax < 1e-5 * F1
    d = np.linalg.norm(o.get("POS") - w0.pos_f, axis=1)
    assert d.max() == pytest.approx(1.3 * dx / 32.0, rel=1e-9)
    # a jittered lattice becomes more regular: the spread of the kernel sums shrinks
    wj = wl.still_tank(n=n, dx=dx, jitter=0.12)
    oj = orc.Oracle.from_workload(wj)

    def sigma_spread(pos):
        h = 1.3 * dx
        allp = np.concatenate([pos, wj.pos_w.astype(np.float64)])
        dd = np.linalg.norm(pos[inner][:, None, :] - allp[None, :, :], axis=2)
        q = dd / h
        W = np.where(q < 2, (1 - 0.5 * q) ** 4 * (1 + 2 * q), 0.0).sum(axis=1)
        return W.std() / W.mean()
    s0 = sigma_spread(wj.pos_f.astype(np.float64))
    oj.relax(40, 100.0)
    s1 = sigma_spread(oj.get("POS"))
    assert s1 < 0.5 * s0, (s0, s1)


# ------------------------------------------------------------------------------------------------
# Planar mode (reading R25) and the paper's own section 3.2 benchmark in two dimensions
# ------------------------------------------------------------------------------------------------
def test_R25_planar_kernel_integrates_to_one_and_lattice_sum():
    for h in (0.7, 0.0125):
        val, _ = integrate.quad(lambda r: 2.0 * math.pi * r * orc.W2d(r, h), 0.0, 2.0 * h, epsabs=0, epsrel=1e-12)
        assert val == pytest.approx(1.0, rel=1e-10)
        r, e = 0.83 * h, 1e-6 * h
        assert orc.dWdr2d(r, h) == pytest.approx((orc.W2d(r + e, h) - orc.W2d(r - e, h)) / (2 * e), rel=1e-6)
        assert orc.W2d(2.0 * h, h) == 0.0 and orc.W2d(0.0, h) == pytest.approx(7.0 / (4.0 * math.pi * h * h), rel=1e-14)
    # square-lattice partition of unity at h = dx, summed here site by site (8 + 4 + ... neighbours inside 2h)
    dx = 0.0125
    s = sum(orc.W2d(dx * math.hypot(a, b), dx) for a in range(-3, 4) for b in range(-3, 4))
    assert orc.sigma0_2d(dx, dx) == pytest.approx(s, rel=1e-14)
    assert dx * dx * s == pytest.approx(1.0, abs=0.05)


@pytest.mark.timeout(300)
def test_R25_two_slab_benchmark_as_in_the_paper(golden):
    """PAPER.md:231-268 as printed: a 1 x 0.5 slab in two dimensions, dx = 0.0125, h = dx, Table 3 materials,
    profile on the line y = 0.25 at t = 2.0 against the analytic solution (Fig. 2b)"""
    g = golden("two_slab_conduction.txt")
    dx = g["dx"]
    nx, ny = 80, 40
    sites = np.stack(np.meshgrid(np.arange(nx), np.arange(ny), indexing="ij"), -1).reshape(-1, 2)
    pos = np.concatenate([(sites + 0.5) * dx, np.full((len(sites), 1), 0.5 * dx)], axis=1).astype(np.float32)
    left = pos[:, 0] < g["x_iface"]
    params = wl.default_params(dx, h=g["h_over_dx"] * dx, flags=wl.FLAG_THERMAL, rho0=1000.0, g=[0, 0, 0],
                               dt_fixed=0.01, rebuild_every=10 ** 6, k_f=1.0, cp_f=1.0, dim=2)
    params["domain_min"] = [-0.05, -0.05, 0.0]
    params["domain_max"] = [1.05, 0.55, dx]
    rho = np.where(left, g["rho_l"], g["rho_r"])
    o = make_oracle(params, pos, rho=rho.astype(np.float32), T=np.where(left, g["T_left0"], g["T_right0"]).astype(np.float32))
    o.set_materials(mass=rho * dx ** 2, k=np.where(left, g["k_l"], g["k_r"]), cp=np.where(left, g["cp_l"], g["cp_r"]))
    E0 = (rho * o.get("T")).sum()
    o.step(int(round(g["t_end"] / 0.01)))
    T = o.get("T")
    assert abs((rho * T).sum() - E0) < 1e-12 * E0
    el, er = math.sqrt(g["k_l"] * g["rho_l"] * g["cp_l"]), math.sqrt(g["k_r"] * g["rho_r"] * g["cp_r"])
    Tc = er / (el + er)
    x = pos[:, 0].astype(np.float64)
    t = g["t_end"]
    ana = np.where(left, Tc * special.erfc(np.abs(x - 0.5) / (2 * math.sqrt(g["alpha_l"] * t))),
                   1.0 - (1.0 - Tc) * special.erfc(np.abs(x - 0.5) / (2 * math.sqrt(g["alpha_r"] * t))))
    line = sites[:, 1] == ny // 2                               # y = 0.25 (Fig. 2b)
    assert np.abs(T[line] - ana[line]).max() < 1.0e-2
    # the middle rows show the same profile (nothing leaks through the sides; next to a side the truncated kernel
    # support slows the conduction a little, which is felt a few spacings inwards by t = 2)
    rows = T.reshape(nx, ny)
    assert np.abs(rows[:, 12:-12] - rows[:, [ny // 2]]).max() < 1e-3
    assert np.abs(rows - rows[:, [ny // 2]]).max() < 1e-2


# ------------------------------------------------------------------------------------------------
# R26  viscous sums evaluated once per advection step and held (the scheme of ref [45])
# ------------------------------------------------------------------------------------------------
def _shear_pair(flags, K, dt, v0=0.4, sep=1.2):
    """two particles on the x axis sliding past each other along y: v_ij . r_ij = 0, so the pressure and
    continuity sums vanish (U_L = U_R, p_i = p_j) and only the viscous sum acts, along y."""
    dx = 2e-3
    params = wl.default_params(dx, g=[0.0, 0.0, 0.0], flags=flags, dt_fixed=dt, rebuild_every=K)
    params["domain_min"] = [-0.02] * 3
    params["domain_max"] = [0.02] * 3
    pos = np.array([[0.0, 0.0, 0.0], [sep * dx, 0.0, 0.0]], np.float32)
    vel = np.array([[0.0, v0, 0.0], [0.0, -v0, 0.0]], np.float32)
    o = make_oracle(params, pos, vel)
    s = float(pos[1, 0]); h = params["h"]; q = s / h
    F = -(5.0 * 21.0 / (16.0 * math.pi * h ** 4)) * q * (1 - q / 2) ** 3 / s          # W'(s) / s
    m, rho0 = params["rho0"] * dx ** 3, params["rho0"]
    c = 2.0 * (m / rho0 ** 2) * (rho0 * params["nu"]) * F          # a^nu_i = c v_ij (Eq. 10 l.2), c < 0
    return o, c, float(np.float32(v0))


def test_R26_held_viscous_force_is_constant_within_an_advection_step_hand_value():
    K, dt = 4, 2.0e-5
    o, c, v0 = _shear_pair(wl.FLAGS_ALL_PHYSICS | wl.FLAG_VISCOUS_HELD, K, dt)
    a_held = c * 2.0 * v0                    # v_ij = 2 v_y at the rebuild; closed form: v_y linear in the step number
    for k in range(1, K + 1):
        o.step(1)
        v = o.get("VEL")
        np.testing.assert_allclose(v[:, 1], [v0 + k * dt * a_held, -(v0 + k * dt * a_held)], rtol=1e-13)
        np.testing.assert_allclose(o.get("ACC")[:, 1], [a_held, -a_held], rtol=1e-12)
        assert np.abs(v[:, [0, 2]]).max() == 0.0
    np.testing.assert_allclose(o.get("RHO"), 870.0, rtol=1e-15)
    # step K + 1 rebuilds (the pair has sheared: r_ij has a y component now): new value, again constant for K steps
    o.step(1)
    a1 = o.get("ACC_V").copy()
    assert abs(a1[0, 1] - a_held) > 1e-9 * abs(a_held)
    o.step(K - 1)
    assert np.array_equal(o.get("ACC_V"), a1)
    # the per-acoustic-step evaluation (R8) decays geometrically instead: v_y (1 + 2 c dt)^k
    o2, c2, _ = _shear_pair(wl.FLAGS_ALL_PHYSICS, K, dt)
    o2.step(K)
    assert o2.get("VEL")[0, 1] == pytest.approx(v0 * (1.0 + 2.0 * c2 * dt) ** K, rel=1e-13)
    assert abs(o2.get("VEL")[0, 1] - (v0 + K * dt * a_held)) > 1e-7 * v0          # the two variants are distinguishable here


def test_R26_rebuild_every_step_equals_the_per_step_evaluation():
    w = wl.perturb_state(wl.still_tank(n=6, flags=wl.FLAGS_ALL_PHYSICS, dt_fixed=2.0e-5, rebuild_every=1))
    w.bodies[1] = wl.Body(k_s=0.13, origin=(0.004, 0.003, 0.011), axis=(0.0, 1.0, 0.0), omega=120.0)
    a = orc.Oracle.from_workload(w)
    b = orc.Oracle.from_workload(w, flags=w.params["flags"] | wl.FLAG_VISCOUS_HELD)
    a.step(3); b.step(3)
    for f in ("POS", "VEL", "RHO", "T", "ACC"):
        assert np.array_equal(a.get(f), b.get(f)), f
    assert np.array_equal(a.torque(1)[0], b.torque(1)[0])


def test_R26_held_wall_forces_balance_held_fluid_accelerations():
    """action-reaction (P11) with held viscous sums: after k > 1 steps of one advection step the viscous part of the wall
    forces is still minus the sum of the (held) fluid-side viscous accelerations, and equals the first step's; a
    fluid-wall pair's hand value: constant viscous deceleration of a particle sliding along a wall."""
    w = wl.perturb_state(wl.still_tank(n=6, flags=wl.FLAGS_ALL_PHYSICS | wl.FLAG_VISCOUS_HELD, dt_fixed=2.0e-5, rebuild_every=4))
    w.bodies[1] = wl.Body(k_s=0.13, origin=(0.004, 0.003, 0.011), axis=(0.0, 1.0, 0.0), omega=120.0)
    o = orc.Oracle.from_workload(w)
    m = w.params["rho0"] * w.params["dx"] ** 3
    o.step(1)
    awv0, aw0, F0 = o.get("ACC_WV").copy(), o.get("ACC_V").copy(), o.get("WALL_FORCE").copy()
    Fp0 = F0.sum(axis=0) + (m * awv0).sum(axis=0)                          # pressure part of the total wall force, step 1
    o.step(2)
    assert np.array_equal(o.get("ACC_WV"), awv0) and np.array_equal(o.get("ACC_V"), aw0)
    F = o.get("WALL_FORCE")
    a_wall = o.get("ACC_WP") + o.get("ACC_WV")
    np.testing.assert_allclose(F.sum(axis=0), -(m * a_wall).sum(axis=0), rtol=1e-10, atol=1e-14 * np.abs(F).sum())
    assert np.abs(F.sum(axis=0) + (m * awv0).sum(axis=0) - Fp0).max() > 0  # the pressure part did move on
    tau = np.cross(o.get("WALL_POS")[w.body_w == 1] - np.array(w.bodies[1].origin), F[w.body_w == 1]).sum(axis=0)
    np.testing.assert_allclose(o.torque(1)[0], tau, rtol=1e-10, atol=1e-18)
    o.step(2)                                                              # step 5 rebuilt: new viscous sums
    assert not np.array_equal(o.get("ACC_WV"), awv0)

    # hand value: one fluid particle sliding at 0.4 m/s over one still wall particle, 3 steps without a rebuild
    dx = 2e-3
    params = wl.default_params(dx, g=[0.0, 0.0, 0.0], flags=wl.FLAG_VISCOUS | wl.FLAG_HYDRO | wl.FLAG_VISCOUS_HELD, dt_fixed=2.0e-5, rebuild_every=8)
    params["domain_min"] = [-0.02] * 3
    params["domain_max"] = [0.02] * 3
    pos = np.array([[0.0, 0.0, float(np.float32(1.2 * dx))]], np.float32)
    vel = np.array([[0.4, 0.0, 0.0]], np.float32)
    walls = (np.zeros((1, 3), np.float32), np.array([[0, 0, 1]], np.float32), np.array([1], np.int32), np.array([353.0], np.float32))
    bodies = [wl.Body(), wl.Body(k_s=0.0, origin=(0.0, -0.01, 0.0), axis=(0, 1, 0), omega=0.0)]
    o = make_oracle(params, pos, vel, None, np.array([313.0], np.float32), walls=walls, bodies=bodies)
    o.step(3)
    s = float(pos[0, 2]); h = params["h"]; q = s / h
    dW = -(5.0 * 21.0 / (16.0 * math.pi * h ** 4)) * q * (1 - q / 2) ** 3
    rho0 = params["rho0"]; mm = rho0 * dx ** 3
    a_v = (2.0 / mm) * (mm / rho0) * dx ** 3 * (rho0 * params["nu"]) * float(np.float32(0.4)) / s * dW
    assert o.get("VEL")[0, 0] == pytest.approx(float(np.float32(0.4)) + 3 * 2.0e-5 * a_v, rel=1e-13)
    np.testing.assert_allclose(o.torque(1)[0], np.cross([0.0, 0.01, 0.0], [-mm * a_v, 0.0, 0.0]), rtol=1e-12)
