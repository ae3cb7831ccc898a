#!/usr/bin/env python
"""bench.py -- zone-updates/s of the fp64 MHD step (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A "step" is one full RK2 step of the whole hot path (ghost fill, cons->prim, PLM+HLLD sweeps,
flux update, CT, RK2 combine, dt reduction) over the whole grid of the workload.  The workload at
N = 1 is BASELINE.json configs[3] (3D MHD blast 256^3, minmod, CFL 0.3): the configuration the
north_star's target is quoted on.  Inputs are seeded and synthetic (paper_2511_20337_b200.workloads).

Prints ONE JSON line (rank 0).  Timing: CUDA events on the library's stream, barrier +
synchronize on both sides, max over ranks.  The state (>= 1 GB) is larger than L2 (126 MB), so no
explicit flush is needed between steps.

Multi-GPU (torchrun): the path has no exchange step on one GPU and the north_star names none, so
ranks run independent replicas of the workload ("replicas only") and value is the sum.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "zone-updates/sec (fp64 3D MHD step, 1 B200); achieved HBM GB/s vs peak"
UNIT = "zone-updates/s"

# Algorithmic traffic of the sweep kernels, doubles per zone and launch; a
# state is 5 hydro arrays + 3 face arrays (cell-centred B is never stored):
#   sweep_xy  : read S 8, write S' 5, write CT data 9 (4 induction fluxes, 2 weights, 3 cell EMFs) = 22;
#               the combine stage also reads S^n 5 = 27; the two launches of a step average 24.5
#   sweep_x   : read S 8, write S' 5, CT data 6 (2 fluxes, 1 weight, 3 cell EMFs)                  = 19
#   sweep_y/z : read S 8, read + write S' 5 + 5, CT data 3                                           = 21
#   ct        : read CT data 12 + faces 3, write faces 3 = 18; the combine stage also reads S^n faces 3 = 21;
#               the two launches of a step average 19.5
#   dt_max    : read S 8
ALGO_DOUBLES = {"sweep_xy": 24.5, "sweep_x": 19, "sweep_y": 21, "sweep_z": 21, "ct": 19.5, "dt_max": 8}

# From the committed ncu capture of the same workload (profiles/, `ncu --set full`, per launch, mean of the
# stage-1 and stage-2 launches of a step): DRAM bytes moved and fp64-pipe instructions executed per zone.
NCU = {
    "sweep_xy": {"dram_bytes_per_launch": 3.54e9, "fp64_instr_per_zone": 576, "profile": "profiles/r1c_step_kernels.md"},
    "sweep_z": {"dram_bytes_per_launch": 2.88e9, "fp64_instr_per_zone": 285, "profile": "profiles/r1c_step_kernels.md"},
    "ct": {"dram_bytes_per_launch": 2.89e9, "fp64_instr_per_zone": 117, "profile": "profiles/r1c_step_kernels.md"},
}


def max_over_ranks(value, dist, device="cpu"):
    """a time measured on every rank -> the maximum over ranks (a job is as slow as its slowest replica)"""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(zones_per_rank, steps, ms_max, world):
    """whole-job zone-updates/s of `world` independent replicas (replicas only)"""
    return world * zones_per_rank * steps / (ms_max * 1e-3)


WORKLOAD_NAMES = {0: "configs[0] C0_orszag_tang_2d_128", 1: "configs[1] C1_cp_alfven_3d_64x32x32",
                  2: "configs[2] C2_orszag_tang_2d_2048", 3: "configs[3] C3_blast_3d_256", 4: "configs[4] C4_blast_3d_512",
                  5: "paper section 4.1 workload (not a BASELINE config) P1_orszag_tang_3d_256"}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region"""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [l.split(", ") for t, l in self.lines if t0 <= t <= t1 + 0.2] or [l.split(", ") for _, l in self.lines[-3:]]
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[1]))
                smax.append(float(r[2]))
                power.append(float(r[3]))
                for nm, val in zip(names, r[5:9]):
                    if val.strip().lower() == "active":
                        reasons.add(nm)
            except (ValueError, IndexError):
                pass
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w": statistics.median(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_throughput(workload_small, budget_s=12.0, threads=None, rk=2, max_steps=400):
    """the oracle as it stands, timed on the host cores (zone-updates/s): whole steps until ~budget_s
    seconds of CPU work are done"""
    from oracle import Oracle
    o = Oracle()
    if threads:
        o.set_threads(threads)
    o.load(workload_small)
    o.set_integrator(rk)
    o.step(1)                                   # touch memory
    t0 = time.perf_counter()
    steps = 0
    while steps < max_steps:
        assert o.step(1) == 0
        steps += 1
        dt = time.perf_counter() - t0
        if dt >= budget_s:
            break
    cores = o.get_threads()
    o.finalize()
    return workload_small.zones * steps / dt, cores, dt, steps


def sample_workload(cfg):
    """bounded sample of configs[cfg] for the CPU legs: the same generator at a size the oracle steps in seconds"""
    from paper_2511_20337_b200 import workloads as wl
    if cfg == 5:
        return wl.orszag_tang_3d(128, noise=1e-3), "orszag_tang_3d 128^3 (1/8 of the zones of the 256^3 run)"
    if cfg in (3, 4):
        return wl.blast_3d(128, name="blast_3d_128 (1/8 of the zones of configs[3])"), "blast_3d 128^3, same recipe and seed as configs[3]"
    if cfg == 2:
        return wl.orszag_tang_2d(1024), "orszag_tang_2d 1024^2 (1/4 of the zones of configs[2])"
    return wl.config(cfg), f"configs[{cfg}] at full size"


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/config keys (rank 0 only)"""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    w, what = sample_workload(args.config)
    if args.wenoz:
        w.limiter = 2
    from oracle import Oracle
    o = Oracle()
    o.load(w)
    o.set_integrator(args.rk)
    for _ in range(args.warmup):
        o.step(1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        assert o.step(1) == 0
    dt = time.perf_counter() - t0
    val = w.zones * args.steps / dt
    cores = o.get_threads()
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD_NAMES.get(args.config, f"configs[{args.config}]"), "sample": what,
                   "scheme": "recon(%s)+HLLD+RK%d+CT, CFL %.2g" % (("minmod", "MC", "WENOZ")[w.limiter], args.rk, w.cfl)},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": f"{what}, {args.steps} steps"},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--wenoz", action="store_true", help="WENO-Z reconstruction instead of the config's PLM limiter")
    ap.add_argument("--rk", type=int, default=2, help="2: SSP-RK2 (the north_star's step, default); 3: SSP-RK3 of Eq. 5")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=3)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_2511_20337_b200 import workloads as wl
    from paper_2511_20337_b200.binding import Pluto

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA path has no CPU fallback")
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()

    w = wl.config(args.config)
    if args.wenoz:
        w.limiter = 2
    sim = Pluto(device=local)
    sim.set_integrator(args.rk)
    sim.load(w)
    K, W = args.steps, max(args.warmup, 3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    # ---------------- device-resident timing: K steps, state already in HBM
    sim.step(W)
    launches0 = sim.launch_count()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    barrier()
    torch.cuda.synchronize()
    t0 = time.time()
    e0.record(sim.stream)
    sim.step_async(K)
    e1.record(sim.stream)
    sim.sync()
    torch.cuda.synchronize()
    barrier()
    t1 = time.time()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop(t0, t1)
    launches = sim.launch_count() - launches0
    ms = max_over_ranks(ms, dist, "cuda")
    value = aggregate_throughput(w.zones, K, ms, world)

    # ---------------- per-kernel timing of the same K steps (events around every launch)
    sim.profile(True)
    torch.cuda.synchronize()
    e0.record(sim.stream)
    sim.step_async(K)
    e1.record(sim.stream)
    sim.sync()
    ms_prof = e0.elapsed_time(e1)
    sim.profile(False)
    rep = sim.profile_report()
    total_kernel_ms = sum(v[0] for v in rep.values())
    dom = max(rep, key=lambda k: rep[k][0])
    dom_ms, dom_cnt = rep[dom]
    hbm_peak, peak_src = peaks()
    # units one launch of the dominant kernel processes
    units = w.zones
    algo_bytes = ALGO_DOUBLES.get(dom, 0) * 8 * units
    dur = dom_ms * 1e-3 / max(dom_cnt, 1)
    achieved = algo_bytes / dur * 1e-9 if dur > 0 else 0.0
    roofline = {"kernel": dom, "bound": "hbm", "achieved": achieved, "peak": hbm_peak, "unit": "GB/s",
                "frac": achieved / hbm_peak, "traffic": None, "peak_source": peak_src,
                "avg_launch_ms": dur * 1e3, "launches": dom_cnt, "share_of_step": dom_ms / total_kernel_ms,
                "algorithmic_bytes_per_launch": algo_bytes,
                "kernels_ms_per_step": {k: v[0] / K for k, v in rep.items() if v[1]},
                "profiled_ms_per_step": ms_prof / K}
    # the same HBM view for every kernel of the step (algorithmic bytes / live launch time / HBM peak)
    roofline["all_kernels_hbm_frac"] = {
        k: round(ALGO_DOUBLES[k] * 8 * units / (v[0] * 1e-3 / v[1]) * 1e-9 / hbm_peak, 4)
        for k, v in rep.items() if v[1] and k in ALGO_DOUBLES}
    if dom in NCU:
        roofline["traffic"] = NCU[dom]["dram_bytes_per_launch"] * (units / 256 ** 3)   # scaled from the 256^3 capture
        roofline["traffic_source"] = NCU[dom]["profile"]
        # the same kernel against the fp64 pipe: instructions executed per second vs the probed DFMA rate
        fp64_peak = sim.probe_fp64_gflops() * 0.5e9            # DFMA/s (2 flops each)
        rate = NCU[dom]["fp64_instr_per_zone"] * units / dur if dur > 0 else 0.0
        roofline["alu"] = {"bound": "alu", "achieved": rate * 1e-12, "peak": fp64_peak * 1e-12, "unit": "T fp64-instr/s",
                           "frac": rate / fp64_peak, "peak_source": "pluto_probe_fp64_gflops (register-resident DFMA loop, this run)",
                           "fp64_instr_per_zone": NCU[dom]["fp64_instr_per_zone"]}
    # whole-step view: minimum traffic 320 B per zone-update
    roofline["step_hbm_frac_at_320B"] = value / world * 320.0 / (hbm_peak * 1e9)

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": (f"configs[{args.config}] {w.name}" if args.config < 5 else f"paper section 4.1 workload (not a BASELINE config) {w.name}"), "grid": [w.nx, w.ny, w.nz], "zones": w.zones,
                   "scheme": "recon(%s)+HLLD+RK%d+CT, CFL %.2g" % (("minmod", "MC", "WENOZ")[w.limiter], args.rk, w.cfl),
                   "l2": "inputs larger than L2 (state %.2f GB)" % (11 * w.zones * 8 / 1e9),
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "clocks": clocks, "gpu_launches": int(launches), "roofline": roofline,
    }

    # ---------------- end to end through the C ABI with HOST buffers
    if rank == 0 or world > 1:
        Uh = torch.from_numpy(w.U).pin_memory()
        Bh = torch.from_numpy(w.Bface).pin_memory()
        Uo = torch.empty_like(Uh).pin_memory()
        Bo = torch.empty_like(Bh).pin_memory()
        Un, Bn, Uon, Bon = Uh.numpy(), Bh.numpy(), Uo.numpy(), Bo.numpy()
        sim.set_state(Un, Bn)
        sim.step(1)
        sim.get_state(Uon, Bon)
        barrier()
        torch.cuda.synchronize()
        tw0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            sim.set_state(Un, Bn)               # host -> device inside the timed region
            sim.step(1)
            sim.get_state(Uon, Bon)             # device -> host read of the step's result
        torch.cuda.synchronize()
        te = (time.perf_counter() - tw0) / args.e2e_steps
        te = max_over_ranks(te, dist, "cuda")
        nbytes = (Uh.numel() + Bh.numel()) * 8
        # pluto_set_state does not copy U[4..6] of the active dimensions (the cell-centred B is the face mean)
        h2d = (Uh.numel() // 8 * (5 if w.nz > 1 else 6) + Bh.numel()) * 8
        line["e2e"] = {"value": world * w.zones / te, "unit": UNIT, "h2d_bytes_per_step": h2d,
                       "d2h_bytes_per_step": nbytes, "ms_per_step": te * 1e3, "steps": args.e2e_steps}

    # ---------------- the oracle timed beside it (rank 0, N = 1 only)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        ws, what = sample_workload(args.config)
        if args.wenoz:
            ws.limiter = 2
        v, cores, secs, steps = oracle_throughput(ws, rk=args.rk)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"{what}, {steps} steps, {secs:.1f} s"}
    else:
        line["cpu_baseline"] = None

    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
