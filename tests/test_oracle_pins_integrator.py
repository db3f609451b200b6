"""Pins of the oracle's time integrator, of the wall part of the density re-initialisation and of the wall
continuity term against closed forms (-m "not gpu").

These are the parts of oracle/sph_oracle.c that round 1 left checked by nothing but the kernel written to match them
("What's missing" 2).  Every test names, in its docstring, the one-token mutation of sph_oracle.c that
makes it fail; the mutations were applied one by one and each test was seen to fail on its own (round-2 notes in DESIGN.md section 5).

  I1  free-streaming particle: the kick-drift-kick halves of the position-Verlet step (ref [45]; R7) are
      exact for a constant acceleration;
  I2  homogeneous expansion v = A r on a lattice: rho after step 1 and step 2 in closed form with the lattice constant
      c1: pins the dt/2 factors of a7 / a11 and the hand-over of the saved rate;
  I3  full tank WITH its three wall layers: Eq. 15 returns rho0 next to the wall (R12 "sum includes
      walls");
  I4  one fluid-wall pair moving along the wall normal: DRHO_DT from Eq. 12 / 16 / 17 in closed form (R6), with and
      without gravity in P_R;
  I5  plane acoustic pulse in a block of fluid: splits into two halves travelling at c0, amplitude never grows
      (SURVEY.md P8 third item; Eq. 2, Eq. 10-13).
"""
import math

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2512_09904_b200 import workloads as wl

HYDRO_ONLY = wl.FLAG_HYDRO | wl.FLAG_PRESSURE | wl.FLAG_VISCOUS


def _one_particle(params, r0, v0, rho=None):
    o = orc.Oracle(params, None, 1)
    o.load_particles(np.asarray([r0], np.float32), np.asarray([v0], np.float32),
                     None if rho is None else np.asarray([rho], np.float32), np.zeros(1, np.float32))
    return o


# ------------------------------------------------------------------------------------------------
# I1  free streaming: r = r0 + n dt v0 + (n dt)^2 g / 2, v = v0 + n dt g  (exact for the kick-drift scheme)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("g", [[0.0, 0.0, 0.0], [0.3, -0.2, -9.81]])
def test_I1_free_particle_follows_the_parabola_exactly(g):
    """position-Verlet halves a7 / a9 (R7).  Fails when `o->r[3 * i + d] += 0.5 * dt * o->v[3 * i + d]`
    loses its 0.5 in a7 or in a9 of orc_step_once (r is off by n dt v0 / 2), or when the kick `o->v += dt * o->acc`
    is moved after the second drift."""
    dx, dt, n = 2e-3, 2.5e-5, 40
    params = wl.default_params(dx, g=g, flags=HYDRO_ONLY, dt_fixed=dt, rebuild_every=7)
    params["domain_min"], params["domain_max"] = [-0.5] * 3, [0.5] * 3
    r0 = np.array([0.01, -0.02, 0.03], np.float32).astype(np.float64)
    v0 = np.array([0.7, 0.4, -0.9], np.float32).astype(np.float64)
    o = _one_particle(params, r0, v0)
    for k in range(1, n + 1):
        o.step(1)
        t = k * dt
        np.testing.assert_allclose(o.get("VEL")[0], v0 + t * np.asarray(g), rtol=0, atol=1e-14)
        np.testing.assert_allclose(o.get("POS")[0], r0 + t * v0 + 0.5 * t * t * np.asarray(g), rtol=0, atol=1e-15)
    assert o.get("RHO")[0] == 870.0 and o.get("DRHO_DT")[0] == 0.0          # no neighbours: the density stays
    assert o.stats()["t"] == pytest.approx(n * dt, rel=1e-12)


# ------------------------------------------------------------------------------------------------
# I2  homogeneous expansion on a lattice: density after one and two acoustic steps
# ------------------------------------------------------------------------------------------------
def test_I2_density_after_one_and_two_steps_of_a_homogeneous_expansion(golden):
    """a7 / a10 / a11 (R7): with v = A r, A positive definite (every pair recedes: beta = 0, p* = Pbar), uniform
    rho0 and g = 0 the interior of a lattice feels no force, so v stays and, the geometry being frozen (no rebuild,
    PAPER.md:191), sweep B returns D = -c1 rho0 tr A at every step (rho cancels from 2 rho_i V_j (v_i - v*) when rho is
    uniform).  Hence  rho^1 = rho0 + dt/2 D  (first half adds the saved rate, 0 at t = 0; second half adds dt/2 D) and
    rho^2 = rho^1 + dt/2 D (saved by step 1) + dt/2 D = rho0 + 3/2 dt D.
    Fails when either `0.5 * dt` of the density halves in orc_step_once becomes `dt` (rho^1 = rho0 + dt D or
    rho^2 = rho0 + 2 dt D), when `o->drho_saved[i] = o->drho_dt[i]` is dropped (rho^2 = rho0 + dt D), or when the
    factor 2 of `2.0 * rho_i * sr` in orc_sweep_B is lost."""
    c1 = golden("kernel_lattice_sums.txt")["c1_h1.3"]
    dx, dt, n = 2e-3, 2e-5, 17            # centre particle is 8.5 dx from the surface: three supports (7.8 dx) of clean interior
    w = wl.still_tank(n=n, dx=dx, jitter=0.0, g=[0.0, 0.0, 0.0], flags=HYDRO_ONLY, dt_fixed=dt, rebuild_every=1000)
    pos = w.pos_f
    c = 0.5 * (pos.min(0) + pos.max(0)).astype(np.float64)
    x = pos.astype(np.float64) - c
    A = np.diag([9.0, 14.0, 5.0])
    o = orc.Oracle(dict(w.params), None, 0)
    o.load_particles(pos, (x @ A.T).astype(np.float32), None, np.zeros(len(pos), np.float32))
    i = int(np.argmin((x ** 2).sum(axis=1)))
    rho0 = 870.0
    D = -c1 * rho0 * np.trace(A)
    o.step(1)
    assert o.get("DRHO_DT")[i] == pytest.approx(D, rel=3e-6)
    assert o.get("RHO")[i] - rho0 == pytest.approx(0.5 * dt * D, rel=3e-6)
    assert np.abs(o.get("ACC")[i]).max() < 1e-6 * abs(D) / rho0 * 20.0       # no force in the interior (scale: c0 |D| / rho0)
    o.step(1)
    assert o.get("DRHO_DT")[i] == pytest.approx(D, rel=3e-6)
    assert o.get("RHO")[i] - rho0 == pytest.approx(1.5 * dt * D, rel=3e-6)
    assert o.get("DRHO_SAVED")[i] == pytest.approx(D, rel=3e-6)
    assert o.stats()["rebuilds"] == 1


# ------------------------------------------------------------------------------------------------
# I3  density re-initialisation next to a wall (Eq. 14-15 with wall neighbours)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("free_surface", [False, True])
def test_I3_reinit_next_to_a_three_layer_wall_returns_rho0(free_surface):
    """a5 (R12: the sum runs over fluid AND wall neighbours, sigma0 is the full-lattice sum).  In the
    unjittered full tank the three wall layers (3 dx > 2h = 2.6 dx) complete every fluid particle's support, so
    sigma_i = sigma0 and Eq. 15 returns rho0 for EVERY particle, those touching the wall included; Eq. 14 returns
    max(rho*, rho0).  Fails when the wall loop of orc_density_reinit is dropped or reads `o->r_frz` instead of `o->rw`
    (the corner particle then sees 1/8 of its support), and when W(0) is left out of `s`."""
    flags = wl.FLAGS_ALL_PHYSICS | wl.FLAG_DENSITY_REINIT | (wl.FLAG_FREE_SURFACE if free_surface else 0)
    w = wl.still_tank(n=8, jitter=0.0, flags=flags)
    n = w.n_f
    rho_in = np.where(np.arange(n) % 2 == 0, 860.0, 873.0).astype(np.float32)
    o = orc.Oracle.from_workload(wl.dataclasses.replace(w, rho_f=rho_in))
    o.rebuild()
    rho = o.get("RHO")
    want = np.maximum(rho_in.astype(np.float64), 870.0) if free_surface else np.full(n, 870.0)
    np.testing.assert_allclose(rho, want, rtol=1e-6, atol=0)
    corner = int(np.argmin(w.pos_f.sum(axis=1)))
    cff, cfw, _ = o.neigh()
    assert cff[corner] + cfw[corner] == 80 and cfw[corner] > cff[corner]     # the pin does go through the wall sum


# ------------------------------------------------------------------------------------------------
# I4  wall continuity term (R6): closed forms for one fluid-wall pair
# ------------------------------------------------------------------------------------------------
def _wall_pair(vz, g, rho_i=871.5, s_over_dx=1.2, omega=0.0):
    dx = 2e-3
    params = wl.default_params(dx, g=g, flags=wl.FLAGS_ALL_PHYSICS)
    params["domain_min"], params["domain_max"] = [-0.02] * 3, [0.02] * 3
    s = float(np.float32(s_over_dx * dx))
    pos = np.array([[0.0, 0.0, s]], np.float32)
    walls = (np.zeros((1, 3), np.float32), np.array([[0, 0, 1]], np.float32), np.array([0], np.int32), np.array([313.0], np.float32))
    # body 0 turning about the x axis through (0, 1, 0): v_w = omega e_x x (0, -1, 0) = (0, 0, -omega)
    bodies = [wl.Body(origin=(0.0, 1.0, 0.0), axis=(1, 0, 0), omega=omega)]
    o = orc.Oracle(params, bodies, 0)
    o.load_particles(pos, np.array([[0.0, 0.0, vz]], np.float32), np.array([rho_i], np.float32), np.array([313.0], np.float32), *walls)
    o.eval_rates()
    h = params["h"]
    q = s / h
    dW = -(5.0 * 21.0 / (16.0 * math.pi * h ** 4)) * q * (1.0 - 0.5 * q) ** 3
    return o, params, s, dW


@pytest.mark.parametrize("vz", [-0.5, 0.25])
def test_I4_wall_continuity_hand_value_without_gravity(vz):
    """Eq. 16-17 + Eq. 12, R6.  Still wall, g = 0: U_L = -v_z, U_R = -U_L, P_R = P_L, rho_R = rho_L,
    so Ubar = 0, U* = 0, U* - U_L = v_z and  drho/dt = 2 rho_i V_w v_z W'(s)  (n_w . e_iw = 1): positive on approach.
    Fails when the factor 2 of `UR = -UL + 2.0 * uw` or of `2.0 * rho_i * sr` is lost, when `Vw` is replaced by V_i, or
    when `(Us - UL)` becomes `(Us - Ub)` (which is 0 here)."""
    rho_i = float(np.float32(871.5))
    o, params, s, dW = _wall_pair(vz, [0.0, 0.0, 0.0], rho_i)
    want = 2.0 * rho_i * params["dx"] ** 3 * float(np.float32(vz)) * dW
    assert o.get("DRHO_DT")[0] == pytest.approx(want, rel=1e-12)
    assert (want > 0) == (vz < 0)


def test_I4_wall_continuity_hand_value_with_gravity_and_moving_wall():
    """the same pair with g = (0, 0, -9.81) and the wall moving along its normal at u_z = -0.3 (Eq. 17: U_R = -U_L + 2 u_w,
    P_R = P_L + rho_f g . r_fw, r_fw = r_w - r_f; rho_R from Eq. 2).  Eq. 12 written out for these states:
        U_L = -v_z, u_w = -u_z, U_R = v_z - 2 u_z,  P_R - P_L = rho_i 9.81 s  (the wall particle lies BELOW the fluid one),
        U* = (rho_L U_L + rho_R U_R)/(rho_L + rho_R) - (P_R - P_L)/(c0 (rho_L + rho_R)).
    Fails when the sign of `riw` in `pR = p_i - rho_i * (g . riw)` flips (r_fw taken as r_f - r_w), when `c0 * rs` in
    orc_riemann loses c0, or when u_w is projected with the wrong sign (`uw = +(nw . vw)`)."""
    vz, uz, gz = 0.2, -0.3, -9.81
    rho_i = float(np.float32(871.5))
    o, params, s, dW = _wall_pair(vz, [0.0, 0.0, gz], rho_i, omega=-uz)      # v_w = (0, 0, -omega) = (0, 0, uz)
    c0, rho0, Vw = params["c0"], params["rho0"], params["dx"] ** 3
    vzf = float(np.float32(vz))
    UL, UR = -vzf, vzf - 2.0 * uz
    dP = rho_i * 9.81 * s                                                    # P_R - P_L > 0: hydrostatic increase downwards
    rhoL = rho_i
    rhoR = rho0 + (c0 * c0 * (rho_i - rho0) + dP) / (c0 * c0)
    Ustar = (rhoL * UL + rhoR * UR) / (rhoL + rhoR) - dP / (c0 * (rhoL + rhoR))
    want = 2.0 * rho_i * Vw * (Ustar - UL) * dW
    assert o.get("DRHO_DT")[0] == pytest.approx(want, rel=1e-11)
    # the gravity part on its own is visible at this tolerance: dropping it moves the value by > 1e-3 relative
    no_g = 2.0 * rho_i * Vw * ((rhoL * UL + rhoL * UR) / (2.0 * rhoL) - UL) * dW
    assert abs(no_g - want) > 1e-3 * abs(want)


# ------------------------------------------------------------------------------------------------
# I5  plane acoustic pulse in a block of fluid
# ------------------------------------------------------------------------------------------------
@pytest.mark.timeout(300)
def test_I5_acoustic_pulse_splits_travels_at_c0_and_never_grows():
    """Eq. 2 + Eq. 10-13 together: a small plane Gaussian density pulse at rest splits into two
    halves moving at +-c0 (linear acoustics); the Riemann terms only ever remove amplitude (the
    (p_L - p_R)/(c (rho_L + rho_R)) part of U*, Eq. 12, diffuses density, so each half arrives with less than A/2).  A block
    of fluid without walls: at rho0 the pressure is zero, so its free faces stay at rest, and the release waves from the
    side faces (20 dx away) reach the centre line only after the measurement (14 dx of travel; with faces 16 dx
    away the peak is already 3 % early at 12 dx).  [A duct with
    dummy-particle walls is no 1-D test bed: Eq. 19 gives p* = p_i for wall neighbours, which removes their part of
    the axial pressure gradient and slows the wave next to the wall -- 0.85 c0 in a 6 dx duct.]
    The speed pins the PRODUCT of the continuity and momentum prefactors, c^2 = (2 x 1/2)(2 x 1/2) c0^2: losing the 2 of
    `-(2.0 / m_i)` in orc_sweep_A or of `2.0 * rho_i * sr` in orc_sweep_B gives c0 / sqrt(2) (peak 4 dx short after 14 dx);
    the '+' sign of Eq. 13 as printed (R3: `vbar + (Us - Ub) * e[d]`) makes the amplitude grow; `ps` without its Pbar
    term leaves the pulse where it is."""
    dx, c0 = 2e-3, 20.0
    L, Wd = 64, 40
    w = wl.dam_break(dx=dx, box=(L * dx, Wd * dx, Wd * dx), column=(L * dx, Wd * dx, Wd * dx), jitter=0.0, c0=c0,
                     g=[0.0, 0.0, 0.0], flags=wl.FLAG_HYDRO | wl.FLAG_PRESSURE, rebuild_every=1000)
    none3, none1 = np.zeros((0, 3), np.float32), np.zeros(0, np.float32)
    w = wl.dataclasses.replace(w, pos_w=none3, normal_w=none3, body_w=np.zeros(0, np.int32), T_w=none1)      # no walls
    h = w.params["h"]
    dt = 0.25 * h / c0
    x = w.pos_f[:, 0].astype(np.float64)
    x0, sig, A = 0.5 * L * dx, 4.0 * dx, 0.5
    rho_in = (870.0 + A * np.exp(-0.5 * ((x - x0) / sig) ** 2)).astype(np.float32)
    o = orc.Oracle.from_workload(wl.dataclasses.replace(w, rho_f=rho_in), dt_fixed=dt)
    mid = (Wd / 2 - 0.5) * dx
    centre_line = (np.abs(w.pos_f[:, 1] - mid) < 0.1 * dx) & (np.abs(w.pos_f[:, 2] - mid) < 0.1 * dx)
    xs = x[centre_line]
    order = np.argsort(xs)
    xs = xs[order]
    amp_prev = float((rho_in.astype(np.float64) - 870.0)[centre_line].max())
    n_steps = int(round(14.0 * dx / (c0 * dt)))
    for k in range(n_steps):
        o.step(1)
        amp = float((o.get("RHO") - 870.0)[centre_line].max())
        assert amp <= amp_prev * (1.0 + 1e-9), (k, amp, amp_prev)               # never grows
        amp_prev = amp
    d = (o.get("RHO") - 870.0)[centre_line][order]
    t = n_steps * dt

    def peak(side):                                                            # three-point parabola through the maximum
        i = int(np.argmax(np.where(side, d, -np.inf)))
        off = 0.5 * (d[i - 1] - d[i + 1]) / (d[i - 1] - 2.0 * d[i] + d[i + 1])
        return xs[i] + off * dx, d[i]
    (xr, ar), (xl, al) = peak(xs > x0), peak(xs < x0)
    assert abs((xr - x0) - c0 * t) <= 0.5 * dx, ((xr - x0) / dx, c0 * t / dx)
    assert abs((x0 - xl) - c0 * t) <= 0.5 * dx, ((x0 - xl) / dx, c0 * t / dx)
    assert 0.30 * A <= ar <= 0.5 * A and 0.30 * A <= al <= 0.5 * A
    assert abs(ar - al) < 1e-6 * A                                             # mirror symmetry
    assert abs(d[np.argmin(np.abs(xs - x0))]) < 0.10 * A                       # nothing is left behind at the centre
    v = o.get("VEL")[centre_line][order]
    u_wave = c0 * 0.5 * A / 870.0                                               # particle velocity of a half pulse, c0 drho / rho0
    ip = int(np.argmax(np.where(xs > x0, d, -np.inf)))
    assert np.abs(v[:, 1:]).max() < 0.05 * u_wave                              # still a plane wave on the centre line
    assert v[ip, 0] == pytest.approx(c0 * d[ip] / 870.0, rel=0.05)             # moving outwards with u = c0 drho / rho0


# ------------------------------------------------------------------------------------------------
# I6  Eq. 26: bound of the explicit thermal step
# ------------------------------------------------------------------------------------------------
def test_I6_thermal_step_bound_of_eq26(golden):
    """Eq. 26: dt_T = 0.5 rho C_p h^2 / k.  Heat only (hydrodynamics off, adaptive dt): the step is dt_T itself,
    45.24 s for config 0's oil (tests/golden/dt_criteria.txt); with the hydrodynamics on the acoustic step of Eq. 25 applies
    unless a very conductive fluid pushes dt_T below it; an evolving steel body (R23) brings its own, smaller bound.
    Fails when the bound is left out of orc_step_once (`dt = dtT` dropped: the heat-only run takes 7.8e-5 s steps, the
    conductive fluid steps past its stability limit) or when 0.5 in orc_dt_thermal becomes 1."""
    g = golden("dt_criteria.txt")
    heat_only = wl.FLAG_THERMAL
    w = wl.still_tank(n=6, flags=heat_only)
    o = orc.Oracle.from_workload(w)
    o.step(3)
    assert o.stats()["dt"] == pytest.approx(g["dt_T_oil"], rel=1e-3) and o.stats()["t"] == pytest.approx(3 * g["dt_T_oil"], rel=1e-3)
    # an evolving steel wall: its bound (0.27 s) is the smaller one
    w.bodies[1] = wl.Body(k_s=45.0, rho_s=7850.0, cp_s=460.0, thermal_mode=1)
    o = orc.Oracle.from_workload(w)
    o.step(1)
    assert o.stats()["dt"] == pytest.approx(g["dt_T_steel"], rel=1e-3)
    # hydrodynamics on: the acoustic step rules ...
    w = wl.still_tank(n=6)
    o = orc.Oracle.from_workload(w)
    o.step(1)
    assert o.stats()["dt"] == pytest.approx(0.6 * 2.6e-3 / (20.0 + 2.0), rel=1e-6)          # u_ref = c0 / 10 (R13)
    # ... until the fluid conducts so well that dt_T = 0.5 rho cp h^2 / k falls below it
    k_big = 0.5 * 870.0 * 2000.0 * 2.6e-3 ** 2 / 2.0e-5                                      # dt_T = 2e-5 s
    o = orc.Oracle.from_workload(w, k_f=k_big)
    o.step(1)
    assert o.stats()["dt"] == pytest.approx(2.0e-5, rel=1e-9)
