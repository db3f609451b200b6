#!/usr/bin/env python
"""bench.py -- throughput of the whole WCSPH hot path on synthetic workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg1] [--impl ours|reference]

One "step" = one acoustic step of `sph_step` (control + dt reduction, neighbour rebuild when the
advection criterion of Eq. 25 says so, sweep A, kick/drift, sweep B, finish, torque).  The metric is
BASELINE.json's: particle-steps/s = N_fluid * K / time, whole job, inputs resident in HBM.
`e2e` is the same metric through the C ABI with HOST buffers, as a continuing host-coupled run: every
step uploads the fluid state from pinned host memory (sph_set_state: the clock, the gears and the saved
rates are kept; a moved particle would force a neighbour rebuild), advances one step, and reads
POS/VEL/RHO/T and the torque back.  The line also carries full sub-records (value, e2e, roofline, clocks) for the two 8 M+
workloads the north_star names (`at_8m`: dam8m and cfg4).

N > 1 (under torchrun): the path does not shard (north_star: one GPU), so every rank runs an
independent replica ("replicas only"); value = sum of all ranks' units / max time.

`--impl reference` times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "particle-steps/s"
WORKLOADS = {
    # name: (generator name, kwargs, description)
    "cfg0": ("still_tank", {}, "still oil tank 24^3, dx=2mm (BASELINE.json configs[0])"),
    "cfg1": ("dam_break", {}, "3-D dam break with heated floor, dx=3mm (BASELINE.json configs[1])"),
    "cfg2": ("cfg2", {}, "spur gear 150 rad/s isothermal, dx=1.5mm (configs[2])"),
    "cfg3": ("cfg3", {}, "spur gear 600 rad/s thermal, dx=1.2mm (configs[3])"),
    "cfg4": ("cfg4", {}, "bevel-helical reducer 300 rad/s, dx=1mm (configs[4])"),
    "dam8m": ("dam_break", {"dx": 1.89e-3}, "configs[1] geometry at dx=1.89mm (~8M fluid)"),
}

# algorithmic bytes per launch of the pair sweeps: every sorted record is
# fetched from HBM once and every result written once.
#   sweep A: read {r_frozen,drho} 16 + {v,T} 16 + {r_current,drho_saved} 16, write {v,T} 16 + r_current 16 + a 16
#   sweep B: read 16 + 16, write {drho/dt, dT/dt} 8;  walls: WA 16 (A), WA + WB 32 (B) per wall particle
BYTES_SWEEP_A = (96, 16)
BYTES_SWEEP_B = (40, 32)
# algorithmic fp32 operations per neighbour pair (FMA = 2), counted from the formulas of Eq. 10-13, 18-19, 22
# (DESIGN.md section 4): (fluid-fluid pair, fluid-wall pair)
FLOPS_SWEEP_A = (54, 62)
FLOPS_SWEEP_B = (38, 58)
# plain fp32 peak: 148 SMs x 128 lanes x 2 (FMA) x 1.965 GHz (B200_PROFILING.md: 148 SMs, clocks.max.sm 1965 MHz)
ALU_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--workload", default="cfg1", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--rebuild-every", type=int, default=0, help="0 = Eq. 25 advection criterion on the device")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--cpu-sample-scale", type=float, default=0.0,
                    help="linear scale of the workload geometry used for the bounded oracle sample (0 = sized for ~10-30 s)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--viscous-held", action="store_true",
                    help="SPH_FLAG_VISCOUS_HELD: viscous sums once per advection step (ref [45], DESIGN.md R26) instead of every acoustic step")
    ap.add_argument("--no-8m", action="store_true", help="skip the 8 M+ sub-records (north_star: 8M+ on one GPU)")
    ap.add_argument("--spinup", type=int, default=-1,
                    help="acoustic steps run before the warm-up so that the timed region sees a developed flow (-1: per workload)")
    ap.add_argument("--steps-8m", type=int, default=200, help="timed steps of each 8 M+ sub-record")
    return ap.parse_args()


def make_workload(name, **extra):
    from paper_2512_09904_b200 import workloads as wl
    gen, kw, _ = WORKLOADS[name]
    kw = dict(kw); kw.update(extra)
    return wl.by_name(gen, **kw)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            pass
        self.t.join(timeout=2)
        if not self.rows:                       # a timed region shorter than the sampling interval: one query right after it
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=10).stdout
                self.rows = [[x.strip() for x in line.split(",")] for line in out.splitlines() if line.strip()]
            except Exception:
                pass
        sm, smax, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); smax.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for k, nm in enumerate(names):
                if len(r) > 3 + k and r[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------------------------------------
# CPU oracle legs
# ------------------------------------------------------------------------------------------------
def sample_scale(steps, warmup, budget=4.0e7, full=2.0e6):
    """linear scale of the dam-break geometry whose fluid count times (steps + warmup) is about `budget`
    particle-steps (roughly 10-30 s of oracle time on 8-16 host cores)."""
    n = min(max(budget / max(steps + warmup, 1), 4.0e4), 1.0e6)
    return round((n / full) ** (1.0 / 3.0), 3)


def oracle_rate(workload, scale, steps, warmup, rebuild_every):
    """particle-steps/s of the fp64 oracle, as it stands, on a geometrically scaled-down sample."""
    from oracle import oracle as orc
    from paper_2512_09904_b200 import workloads as wl
    gen, kw, _ = WORKLOADS[workload]
    kw = dict(kw)
    if scale <= 0:
        scale = sample_scale(steps, warmup, full=0.054 / float(kw.get("dx", 3.0e-3)) ** 3)
    if gen == "dam_break":
        w = wl.dam_break(scale=scale, **kw)
        sample = f"{workload} geometry scaled x{scale:g} in every length at the same dx"
    elif gen == "still_tank":
        w = wl.still_tank(**kw)
        sample = "cfg0 in full"
    else:
        w = wl.spur_gear(dx=4.0e-3, omega=150.0, thermal=True, box=(0.16, 0.06, 0.16), z=16, module=6e-3, width=24e-3)
        sample = "small spur-gear box (dx=4mm) standing in for the gear configs"
    o = orc.Oracle.from_workload(w, rebuild_every=rebuild_every)
    o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    return w.n_f * steps / dt, dt, {"cores": orc.num_threads(), "kind": "oracle",
                                     "sample": f"{sample}: {w.n_f} fluid + {w.n_w} wall particles, {steps} acoustic steps "
                                               f"(+{warmup} warm-up), rebuild_every={rebuild_every}", "seconds": dt}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    re = args.rebuild_every if args.rebuild_every > 0 else 4
    steps = max(1, args.steps)
    warm = max(0, args.warmup)
    v, dt, info = oracle_rate(args.workload, args.cpu_sample_scale, steps, warm, re)
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": "particle-steps/s", "n_gpus": args.gpus,
            "steps": steps, "warmup": warm, "ms_per_step": 1e3 * dt / steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload + ": " + WORKLOADS[args.workload][2]},
            "cpu_baseline": dict(info, value=v, unit="particle-steps/s"),
            "e2e": {"value": v, "unit": "particle-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
# N > 1: replicas only -- no data-path collective; the only exchange is this one
# ------------------------------------------------------------------------------------------------
def aggregate_over_ranks(ms, units, dist=None, device="cpu"):
    """whole-job figures of N independent replicas: time = MAX over ranks, units = SUM over ranks."""
    import torch
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ------------------------------------------------------------------------------------------------
# CUDA arm
# ------------------------------------------------------------------------------------------------
# acoustic steps run before the warm-up (not timed, not counted as warm-up): the timed region then sees a flow that has
# started to move (dam break: the column has begun to collapse and splash tiles exist; gears: the oil has been picked up)
SPINUP = {"cfg0": 0, "cfg1": 1000, "dam8m": 300, "cfg2": 300, "cfg3": 300, "cfg4": 200}


def load_traffic(workload, kernel):
    """dram bytes per launch of `kernel` from the committed ncu --set full capture (profiles/traffic.csv), or None"""
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(tpath):
        with open(tpath) as f:
            for line in f.read().splitlines()[1:]:
                cols = line.split(",")
                if len(cols) >= 3 and cols[0] == workload and cols[1] == kernel:
                    return int(cols[2])
    return None


def measure(args, api, torch, name, w, K, W, spinup, e2e_steps, dist, local, with_e2e=True):
    """one workload: spin-up, W warm-up steps, K timed steps (CUDA events on the library's stream, barrier + synchronize on
    both sides), a profiled region for the per-kernel figures, and the end-to-end loop through the C ABI with host buffers."""
    stream = torch.cuda.current_stream()
    from paper_2512_09904_b200.workloads import FLAG_VISCOUS_HELD
    over = {"flags": int(w.params["flags"]) | FLAG_VISCOUS_HELD} if args.viscous_held else {}
    sim = api.Simulation(w, device=local, cuda_stream=stream.cuda_stream, rebuild_every=args.rebuild_every, **over)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def checked_sync():
        try:
            sim.sync()
            return None
        except api.SphError as e:                 # a particle left the grid (gear workloads late in a run): reported, the run goes on
            return str(e)

    # ---- device-resident timing: no per-kernel events, the library runs each acoustic step as one CUDA graph launch
    sampler = ClockSampler(local)
    sampler.start()                           # runs through spin-up, warm-up and timed region: continuous load
    reports = []
    for done in range(0, spinup, 250):
        sim.step(min(250, spinup - done))
        r = checked_sync()
        if r:
            reports.append(r)
    sim.step(W)
    r = checked_sync()
    if r:
        reports.append(r)
    st0 = sim.stats()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    sim.step(K)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    clocks["window"] = "spin-up + warm-up + timed region (continuous load)"
    r = checked_sync()
    if r:
        reports.append(r)
    st1 = sim.stats()
    launches = int(st1["launches"] - st0["launches"])
    rebuilds = int(st1["rebuilds"] - st0["rebuilds"])
    # per-kernel durations: a second region of the same steps with the library's CUDA events around every launch
    # (predicated launches instead of the graph; the kernels and their launch configurations are the same)
    Kp = max(1, min(K, 60))
    api.sph_profile(sim.ctx, True)
    e0.record(stream)
    sim.step(Kp)
    e1.record(stream)
    checked_sync()
    ms_prof = e0.elapsed_time(e1)
    prof_rebuilds = int(sim.stats()["rebuilds"] - st1["rebuilds"])
    prof = api.sph_get_profile(sim.ctx)
    api.sph_profile(sim.ctx, False)

    ms_max, total_units = aggregate_over_ranks(ms, float(w.n_f) * K, dist, "cuda")
    value = total_units / (ms_max * 1e-3)

    # ---- roofline of the dominant kernel: the pair sweeps are bound by plain fp32 issue + shared-memory gathers, not by HBM
    # (ncu: profiles/), so the roofline object is the ALU one; the HBM fraction the north_star asks for is reported beside it
    peak, peak_src = measured_peaks()
    top = max(("sweep_A", "sweep_B"), key=lambda k: prof[k][0])
    ms_top, n_top = prof[top]
    n_top = min(n_top, Kp)                    # one working launch of each sweep per step (under --viscous-held the class also
                                              # counts the instantiation that returns at once, R26)
    avg_s = ms_top / max(n_top, 1) * 1e-3
    cnt = sim.get("NEIGH_COUNT").astype(np.int64)
    pairs_f, pairs_w = int(cnt[:, 0].sum()), int(cnt[:, 1].sum())
    per = {"sweep_A": BYTES_SWEEP_A, "sweep_B": BYTES_SWEEP_B}[top]
    fl = {"sweep_A": FLOPS_SWEEP_A, "sweep_B": FLOPS_SWEEP_B}[top]
    alg_bytes = per[0] * w.n_f + per[1] * w.n_w
    alg_flops = fl[0] * pairs_f + fl[1] * pairs_w
    traffic = load_traffic(name, "k_" + top)
    hbm_gbs = alg_bytes / avg_s / 1e9 if avg_s > 0 else 0.0
    tflops = alg_flops / avg_s / 1e12 if avg_s > 0 else 0.0
    # the derived ALU peak, checked against a measured one (independent FFMA chains on every SM, the library's own micro-benchmark,
    # run right here under the same clocks; outside the timed region)
    try:
        peak_meas = api.sph_measure_fma_peak(local, stream.cuda_stream)
    except Exception:                                          # a measurement beside the derived peak, never a reason to lose the line
        peak_meas = None
    roofline = {"bound": "alu", "kernel": "k_" + top, "achieved": tflops, "peak": ALU_PEAK_TFLOPS, "unit": "TFLOP/s",
                "frac": tflops / ALU_PEAK_TFLOPS, "traffic": traffic,
                "peak_measured": peak_meas, "frac_of_measured": (tflops / peak_meas) if peak_meas else None,
                "peak_measured_source": "sph_measure_fma_peak: 8 independent fp32 FFMA chains per thread, 8 x 256 threads per SM, CUDA events",
                "traffic_source": "profiles/traffic.csv (ncu --set full capture of this workload)" if traffic else None,
                "peak_source": "derived: 148 SMs x 128 fp32 lanes x 2 x 1.965 GHz (DESIGN.md section 4)",
                "algorithmic_flops_per_launch": alg_flops, "pairs_per_launch": {"fluid": pairs_f, "wall": pairs_w},
                "avg_launch_ms": avg_s * 1e3, "share_of_step": ms_top / ms_prof if ms_prof > 0 else None,
                "profiled_steps": Kp, "profiled_rebuilds": prof_rebuilds, "profiled_ms_per_step": ms_prof / Kp,
                "class_ms": {k: round(v[0], 3) for k, v in prof.items() if v[1]}}
    roofline_hbm = {"bound": "hbm", "kernel": "k_" + top, "achieved": hbm_gbs, "peak": peak, "unit": "GB/s",
                    "frac": hbm_gbs / peak, "traffic": traffic, "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": alg_bytes}
    # whole step against HBM: algorithmic bytes of every kernel class per acoustic step
    step_bytes = (48 + 56 + BYTES_SWEEP_A[0] + BYTES_SWEEP_B[0]) * w.n_f + (BYTES_SWEEP_A[1] + BYTES_SWEEP_B[1]) * w.n_w
    roofline_hbm["whole_step"] = {"algorithmic_bytes_per_step": step_bytes, "achieved": step_bytes / (ms / K * 1e-3) / 1e9,
                                  "frac": step_bytes / (ms / K * 1e-3) / 1e9 / peak}

    # ---- end to end through the C ABI with HOST buffers: a continuing host-coupled run -------------------------------
    e2e = None
    if with_e2e:
        def pinned(shape, dtype):
            return torch.empty(shape, dtype=dtype).pin_memory().numpy()
        # the fluid state lives in four pinned host arrays that every step uploads from and reads back into
        state = {"POS": pinned((w.n_f, 3), torch.float32), "VEL": pinned((w.n_f, 3), torch.float32),
                 "RHO": pinned((w.n_f,), torch.float32), "T": pinned((w.n_f,), torch.float32)}
        for f, buf in state.items():
            api.sph_get_fields(sim.ctx, f, buf.reshape(-1))
        h2d = sum(int(a.nbytes) for a in state.values())
        d2h = sum(int(a.nbytes) for a in state.values()) + 32

        def e2e_step():
            api.sph_set_state(sim.ctx, state["POS"], state["VEL"], state["RHO"], state["T"], api.SPH_MEM_HOST)
            api.sph_step(sim.ctx, 1)
            for f, buf in state.items():
                api.sph_get_fields(sim.ctx, f, buf.reshape(-1))
            api.sph_get_torque(sim.ctx, 0)

        try:
            for _ in range(2):
                e2e_step()
            barrier()
            t0 = time.perf_counter()
            e0.record(stream)
            for _ in range(e2e_steps):
                e2e_step()
            e1.record(stream)
            barrier()
            wall = time.perf_counter() - t0
            e2e_ms, e2e_units = aggregate_over_ranks(max(wall * 1e3, e0.elapsed_time(e1)), float(w.n_f) * e2e_steps, dist, "cuda")
            e2e = {"value": e2e_units / (e2e_ms * 1e-3), "unit": "particle-steps/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                   "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps,
                   "what": "per step: sph_set_state (POS, VEL, RHO, T from pinned host arrays; clock, gears and saved rates kept; the host loop "
                           "here changes nothing, so the positions come back bit for bit and the neighbour configuration stands) + "
                           "sph_step(1) + sph_get_fields POS / VEL / RHO / T to pinned host arrays + sph_get_torque"}
        except api.SphError as ex:
            reports.append(str(ex))
    st2 = sim.stats()
    sim.close()
    rec = {"value": value, "unit": "particle-steps/s", "steps": K, "warmup": W, "spinup_steps": spinup, "ms_per_step": ms_max / K,
           "config": {"workload": name + ": " + WORKLOADS[name][2], "n_fluid": w.n_f, "n_wall": w.n_w,
                      "rebuild_every": args.rebuild_every, "rebuilds_in_timed_region": rebuilds,
                      "vmax_over_c0_at_end": float(st1["vmax"]) / float(w.params["c0"]),
                      "density_reinit": "Eq. 14 in the identified free-surface region, Eq. 15 elsewhere (DESIGN.md R27)",
                      "viscous": "held per advection step (R26)" if args.viscous_held else "every acoustic step (R8)",
                      "tiles": int(st1["tiles"]), "direct_tiles": int(st1["direct_tiles"]), "split_tiles": int(st1["split_tiles"]),
                      "dt": "Eq. 25 adaptive, dual criteria" if args.rebuild_every == 0 else "Eq. 25 adaptive",
                      "l2": "state (>1 GB) larger than the 126 MB L2; no flush needed",
                      "launch": "one CUDA graph launch per acoustic step (rebuild chain = conditional node)" if args.rebuild_every == 0 else "stream launches",
                      "device_reports": reports},
           "clocks": clocks, "gpu_launches": launches, "roofline": roofline, "roofline_hbm": roofline_hbm}
    if e2e is not None:
        rec["e2e"] = e2e
    del st2
    return rec


def run_ours(args):
    import torch
    from paper_2512_09904_b200 import api

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    api.lib()
    w = make_workload(args.workload, seed=1 + rank) if WORKLOADS[args.workload][0] == "dam_break" else make_workload(args.workload)
    K, W = args.steps, args.warmup
    spin = args.spinup if args.spinup >= 0 else SPINUP.get(args.workload, 0)
    head = measure(args, api, torch, args.workload, w, K, W, spin, args.e2e_steps, dist, local)
    del w

    # ---- the 8 M+ points the north_star names: full sub-records (own timed region of >= 200 steps, e2e, roofline, clocks) ------
    at_8m = None
    if rank == 0 and world == 1 and not args.no_8m and args.workload == "cfg1":
        at_8m = []
        for name in ("dam8m", "cfg4"):
            w8 = make_workload(name, seed=1) if name == "dam8m" else make_workload(name)
            rec = measure(args, api, torch, name, w8, max(args.steps_8m, 1), max(W, 5), SPINUP[name], 3, None, local)
            rec["n_fluid"], rec["n_wall"] = w8.n_f, w8.n_w
            at_8m.append(rec)
            del w8

    # ---- CPU baseline: the oracle as it stands, bounded sample, rank 0, N = 1 only ----------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        re = args.rebuild_every if args.rebuild_every > 0 else 4
        v, _, info = oracle_rate(args.workload, args.cpu_sample_scale, 32, 1, re)
        cpu = dict(info, value=v, unit="particle-steps/s")

    if rank == 0:
        line = {"metric": METRIC, "value": head["value"], "unit": "particle-steps/s", "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": dict(head["config"], spinup_steps=head["spinup_steps"], parallelism="replicas only" if world > 1 else "single GPU"),
                "clocks": head["clocks"], "gpu_launches": head["gpu_launches"], "e2e": head.get("e2e"),
                "roofline": head["roofline"], "roofline_hbm": head["roofline_hbm"]}
        if cpu is not None:
            line["cpu_baseline"] = cpu
        if at_8m is not None:
            line["at_8m"] = at_8m
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
