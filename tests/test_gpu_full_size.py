"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (Eq. 25 adaptive dt, the
rebuild decision taken on the device, default list capacities).

The oracle cannot follow millions of particles for hundreds of steps, so parity is "single step from a shared
state": the CUDA path runs k acoustic steps on its own, is advanced to the eve of a
neighbour rebuild, its fp32 state is handed to the fp64 oracle, and both advance one step.  Compared:
  * cell coordinates, neighbour counts and 64-bit neighbour digests of every particle: bit-exact;
  * ACC - g, DRHO_DT, DT_DT over all fluid particles: relative L2 <= 1e-5;
  * every particle still present exactly once (finite positions, permutation intact) after the run;
  * contact factor (Eq. 24) of all wall particles: relative L2 <= 1e-5;
  * per-body torque: |tau_gpu - tau_oracle| <= 1e-5 sum_w |(r_w - o_b) x F_w|.
"""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2512_09904_b200 import workloads as wl

pytestmark = pytest.mark.gpu

REL_L2 = 1.0e-5


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2512_09904_b200 import api as _api
    _api.lib()
    return _api


def rel_l2(a, b):
    a = np.asarray(a, np.float64); b = np.asarray(b, np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def advance_to_rebuild_eve(sim, max_steps=64):
    """step until the next acoustic step will rebuild the neighbour configuration (R14: elapsed >= dt_ad)."""
    for _ in range(max_steps):
        st = sim.stats()
        if st["elapsed"] >= st["dt_ad"]:
            return st
        sim.step(1)
        sim.sync()
    raise AssertionError("no rebuild became due within %d steps" % max_steps)


def shared_state_step(api, w, k):
    sim = api.Simulation(w)                       # bench.py's configuration: rebuild_every = 0, adaptive dt
    sim.step(k)
    sim.sync()
    st = advance_to_rebuild_eve(sim)
    rho0, T_ref = float(w.params["rho0"]), float(w.params.get("T_ref", 313.0))
    pos = sim.get("POS")
    assert pos.shape == (w.n_f, 3) and np.isfinite(pos).all()
    o = orc.Oracle.from_workload(w)
    # bring the oracle's bodies to the GPU's time, then take over the fluid state
    o.set_state(r=pos, v=sim.get("VEL"), rho=rho0 + sim.get("DRHO").astype(np.float64),
                T=T_ref + sim.get("THETA").astype(np.float64), drho_saved=sim.get("DRHO_SAVED"))
    o.set_time(st["t"])
    rebuilds = st["rebuilds"]
    sim.step(1)
    sim.sync()
    o.step(1)
    assert sim.stats()["rebuilds"] == rebuilds + 1, "the shared-state step must be a rebuild step on the GPU"
    return sim, o


def compare(sim, o, w):
    cf, _ = o.cells()
    assert np.array_equal(sim.get("CELL"), cf)
    cff, cfw, dg = o.neigh()
    cnt = sim.get("NEIGH_COUNT")
    assert np.array_equal(cnt[:, 0], cff)
    assert np.array_equal(cnt[:, 1], cfw)
    assert np.array_equal(sim.get("NEIGH_DIGEST"), dg)
    g = np.asarray(w.params["g"], np.float64)
    err = {"ACC-g": rel_l2(sim.get("ACC").astype(np.float64) - g, o.get("ACC") - g),
           "DRHO_DT": rel_l2(sim.get("DRHO_DT"), o.get("DRHO_DT"))}
    if int(w.params["flags"]) & wl.FLAG_THERMAL:
        err["DT_DT"] = rel_l2(sim.get("DT_DT"), o.get("DT_DT"))
    print(w.name, w.n_f, w.n_w, err, {k: sim.stats()[k] for k in ("tiles", "split_tiles", "direct_tiles")})
    for k, v in err.items():
        assert v <= REL_L2, (k, v)
    zg, zo = sim.get("CONTACT_FACTOR"), o.contact_factor()          # Eq. 24, all wall particles
    assert rel_l2(zg, zo) <= REL_L2 and np.max(np.abs(zg - zo)) <= 2e-5
    Fw, rw = o.get("WALL_FORCE"), o.get("WALL_POS")
    for b, body in enumerate(w.bodies):
        sel = w.body_w == b
        if not sel.any():
            continue
        tg, ag = sim.torque(b)
        to, ao = o.torque(b)
        gross = np.linalg.norm(np.cross(rw[sel] - np.asarray(body.origin), Fw[sel]), axis=1).sum()
        assert np.linalg.norm(tg - to) <= 1e-5 * gross + 1e-30, (b, tg, to, gross)
        assert abs(ag - ao) <= 1e-5 * gross + 1e-30


@pytest.mark.parametrize("name,k", [("cfg1", 40), ("cfg2", 25), ("cfg3", 25), ("cfg4", 12)])
def test_full_size_shared_state_step(api, name, k):
    w = wl.by_name(name)
    sim, o = shared_state_step(api, w, k)
    try:
        compare(sim, o, w)
    finally:
        sim.close()
        o.close()


def test_cfg1_runs_its_2000_steps(api):
    """BASELINE.json configs[1]: "Run 2,000 steps".  The full-size dam break in bench.py's launch configuration (step
    graphs, device-decided rebuilds): no device error, every particle finite and inside the box, weakly compressible
    (|rho - rho0| / rho0 below 1 %, the premise of Eq. 2), the heated floor warms the oil next to it."""
    w = wl.by_name("cfg1")
    sim = api.Simulation(w)
    for _ in range(8):
        sim.step(250)
        sim.sync()                                  # raises on a domain / NaN / capacity error
    st = sim.stats()
    assert st["steps"] == 2000 and 300 <= st["rebuilds"] <= 600
    pos, rho, T = sim.get("POS"), sim.get("RHO"), sim.get("T")
    assert np.isfinite(pos).all() and np.isfinite(sim.get("VEL")).all()
    lo, hi = np.asarray(w.params["domain_min"]), np.asarray(w.params["domain_max"])
    assert ((pos > lo) & (pos < hi)).all()
    assert np.abs(rho / 870.0 - 1.0).max() < 0.01
    assert T.min() >= 313.0 - 1e-3 and 313.0 + 1e-3 < T.max() < 353.0
    assert st["vmax"] < 0.25 * float(w.params["c0"])
    sim.close()
