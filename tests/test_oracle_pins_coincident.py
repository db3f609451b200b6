"""Pins of reading R28: two particles at the same place.  -m "not gpu".

The pair terms of the paper carry e_ij = r_ij / r_ij and W'(r_ij) / r_ij (Eq. 10-13, 16-22); at r_ij = 0 both are
0/0 and the paper is silent.  Reading: e_ij -> the zero vector, W'/r -> its limit F(0) = -5 alpha / h^2 (Wendland C2).  In a
long dam break two particles of the collapsing column DO reach the same fp32 position (measured: step 5,840 of config 1), and
without a reading every field of their neighbourhood turns into NaN.

  C1  an isolated coincident pair: hand values -- no pressure force and no mass flux (both act along e_ij), viscous force
      2 eta V_j F(0) (v_i - v_j) / rho_i, heat flux V_j K F(0) (T_i - T_j) / (rho_i c_p); everything finite;
  C2  continuity of the reading: the fields of a pair at separation s -> 0 converge to those of the coincident pair;
  C3  for r > 0 nothing changes: the single-pair hand value of P8 holds to rounding (tests/test_oracle_pins.py) and a random
      cloud with one duplicated particle stays finite, its other pairs untouched.
"""
import math

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2512_09904_b200 import workloads as wl


def _pair(sep, rho=(873.0, 868.0), v=((0.3, -0.2, 0.1), (-0.1, 0.4, 0.25)), T=(320.0, 300.0)):
    dx = 2e-3
    params = wl.default_params(dx, g=[0.0, 0.0, 0.0], flags=wl.FLAGS_ALL_PHYSICS)
    params["domain_min"] = [-0.02] * 3
    params["domain_max"] = [0.02] * 3
    pos = np.array([[1e-3, 2e-3, -1e-3], [1e-3 + sep, 2e-3, -1e-3]], np.float32)
    o = orc.Oracle(params, None, 0)
    o.load_particles(pos, np.array(v, np.float32), np.array(rho, np.float32), np.array(T, np.float32))
    o.eval_rates()
    return params, o


def test_C1_isolated_coincident_pair_hand_values():
    """Fails when e_ij is left as 0/0 (NaN), when W'/r is set to 0 at r = 0 (no viscous force, no heat) and when the limit is
    taken with the wrong constant (e.g. W'(0) = 0 divided by a floor distance)."""
    params, o = _pair(0.0)
    dx, h, rho0, nu, kf, cp = (params[k] for k in ("dx", "h", "rho0", "nu", "k_f", "cp_f"))
    alpha = 21.0 / (16.0 * math.pi * h ** 3)
    F0 = -5.0 * alpha / (h * h)
    m = rho0 * dx ** 3
    rho_i, rho_j = 873.0, 868.0
    v_i, v_j = np.array([0.3, -0.2, 0.1], np.float32).astype(np.float64), np.array([-0.1, 0.4, 0.25], np.float32).astype(np.float64)
    for name in ("ACC", "ACC_P", "ACC_V", "DRHO_DT", "DT_DT"):
        assert np.isfinite(o.get(name)).all(), name
    assert np.abs(o.get("ACC_P")).max() == 0.0                              # the pressure force acts along e_ij = 0
    assert np.abs(o.get("DRHO_DT")).max() == 0.0                            # and so does the mass flux (v_i - v*) . e_ij
    eta = rho0 * nu
    a_i = (2.0 / m) * (m / rho_i) * (m / rho_j) * eta * (v_i - v_j) * F0    # Eq. 10 l.2, viscous term with W'/r -> F(0)
    np.testing.assert_allclose(o.get("ACC_V")[0], a_i, rtol=1e-12)
    np.testing.assert_allclose(o.get("ACC_V")[1], -a_i, rtol=1e-12)                     # action = reaction (equal masses)
    dT_i = (m / rho_j) * (2.0 * kf) * (320.0 - 300.0) * F0 / (rho_i * cp)  # Eq. 22, K = 4 k k / (2 k)
    assert o.get("DT_DT")[0] == pytest.approx(dT_i, rel=1e-12)
    assert dT_i < 0.0                                                       # the hot particle cools


def test_C2_the_reading_is_the_limit_of_small_separations():
    """Fails when the coincident pair is given a value that the formulas do not approach (a jump at r = 0)."""
    _, o0 = _pair(0.0)
    ref = {k: o0.get(k).copy() for k in ("ACC_V", "DT_DT")}
    for sep, tol in ((1e-5, 2e-2), (1e-6, 2e-3)):
        _, o = _pair(sep)
        for k in ref:
            scale = np.abs(ref[k]).max()
            assert np.abs(o.get(k) - ref[k]).max() <= tol * scale, (k, sep)
        # the terms along e_ij stay bounded as the separation goes to zero and carry the factor W' ~ r: they vanish
        assert np.abs(o.get("ACC_P")).max() <= 50.0 * sep / 1e-5 * np.abs(ref["ACC_V"]).max()


def test_C3_duplicated_particle_in_a_cloud_leaves_the_other_pairs_alone():
    """Fails when the guard touches pairs at r > 0."""
    w = wl.random_cloud(3000, 600, extent=(8, 8, 8), seed=21)
    o_ref = orc.Oracle.from_workload(w, neigh_backend=1)
    o_ref.eval_rates()
    k, j = 17, 1400
    w2 = wl.dataclasses.replace(w, pos_f=w.pos_f.copy())
    far = np.linalg.norm(w.pos_f - w.pos_f[k], axis=1) > 2.2 * 2.0 * w.params["h"]   # beyond two cut-offs (re-initialised densities) of the old and the new place
    far &= np.linalg.norm(w.pos_f - w.pos_f[j], axis=1) > 2.2 * 2.0 * w.params["h"]
    assert far.sum() > 500
    w2.pos_f[j] = w.pos_f[k]                                                 # particle j now sits on particle k
    o = orc.Oracle.from_workload(w2, neigh_backend=1)
    o.eval_rates()
    for name in ("ACC", "DRHO_DT", "DT_DT"):
        got, ref = o.get(name), o_ref.get(name)
        assert np.isfinite(got).all(), name
        np.testing.assert_array_equal(got[far], ref[far])
    cff, _, _ = o.neigh()
    assert cff[j] == cff[k] and cff[k] == o_ref.neigh()[0][k] + 1            # each of the two counts the other one
