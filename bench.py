#!/usr/bin/env python
"""bench.py -- zone-updates/s of the fp64 MHD step (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A "step" is one full RK2 step of the whole hot path (ghost fill, cons->prim, PLM+HLLD sweeps,
flux update, CT, RK2 combine, dt reduction) over the whole grid of the workload.  The workload at
N = 1 is BASELINE.json configs[3] (3D MHD blast 256^3, minmod, CFL 0.3): the configuration the
north_star's target is quoted on.  Inputs are seeded and synthetic (paper_2511_20337_b200.workloads).

`python bench.py --gpus N` with N > 1 re-executes itself under torch.distributed.run (one rank per GPU) when no
launcher set WORLD_SIZE, and refuses when the box has fewer than N devices.  `--gpus 1 --slab-path` times the
same decomposed code path as a one-rank NCCL group.

Prints ONE JSON line (rank 0).  Timing: CUDA events on the library's stream, barrier +
synchronize on both sides, max over ranks.  The state (>= 1 GB) is larger than L2 (126 MB), so no
explicit flush is needed between steps.

Multi-GPU (torchrun, N > 1): the domain-decomposed step of the paper's section 3.4 in
its weak-scaling shape (a fixed mesh per GPU): the box grows along z with N, every rank
holds one 256^3 slab (configs[3]'s zones per GPU, one blast per slab-sized section), the ghost planes
are pulled from the neighbour GPUs' memory inside the ghost-fill kernel and dt is one MAX all-reduce.
value = all zones of the box x steps / max-over-ranks time; "scaling": "weak".
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

# Bytes per zone and launch, two accountings (a state is 5 hydro + 3 face arrays):
#   METHOD  -- what the method itself must move through this kernel if every stage reads each state
#              array once and writes it once (320 B per zone-update for the whole step);
#              this is the `achieved` / `frac` of the roofline object;
#   DESIGN  -- what this implementation's kernel is written to move (METHOD + the CT work arrays it
#              exchanges with the other kernels through HBM + re-reads across kernels); reported as
#              `design_*` next to it, so that wasted traffic is visible.
# Keyed by kernel class; values = doubles per zone for (first stage, combine stage).
def kernel_doubles(ndim, rk, glm=False):
    """(method, design) doubles per zone per launch, averaged over the stages of one step"""
    if glm:
        # GLM variant (first version, one kernel per direction; a state is 9 arrays): the x sweep reads S and
        # writes S', the y and z sweeps read S and read-modify-write S'
        m = {"sweep_x": 18.0, "sweep_y": 27.0, "sweep_z": 27.0, "dt_max": 8.0}
        return m, dict(m)
    nface = 3 if ndim == 3 else 2
    nct_xy = 9 if ndim == 3 else 5            # x/y induction fluxes + weights + cell EMFs kept for CT
    combine_stages = rk - 1                   # stages that also read S^n
    def avg(first, comb):
        return (first + combine_stages * comb) / rk
    method = {
        # the x+y sweep reads S (8 arrays) [+ S^n hydro 5 in a combine stage] and writes S' hydro (5)
        "sweep_xy": avg(8 + 5, 8 + 5 + 5),
        "sweep_x": avg(8 + 5, 8 + 5 + 5), "sweep_y": avg(8 + 5, 8 + 5), "sweep_z": avg(8 + 5, 8 + 5),
        # CT reads the faces (nface) [+ S^n faces] and writes them
        "ct": avg(2 * nface, 3 * nface),
        "dt_max": 8.0,
    }
    design = {
        "sweep_xy": avg(8 + 5 + nct_xy, 8 + 5 + 5 + nct_xy),
        "sweep_x": avg(8 + 5 + 6, 8 + 5 + 5 + 6), "sweep_y": 8 + 5 + 5 + 3, "sweep_z": 8 + 5 + 5 + 3,
        "ct": avg((12 if ndim == 3 else 5) + 2 * nface, (12 if ndim == 3 else 5) + 3 * nface),
        "dt_max": 8.0,
    }
    return method, design


def ncu_table(ndim, rk, limiter, zones):
    """per-kernel DRAM bytes per launch and fp64-pipe instructions per zone from the newest committed
    `profiles/r*_step_kernels.md` (an `ncu --set full` capture of configs[3], RK2, minmod); None for any
    other scheme: those numbers do not transfer"""
    import glob
    import re
    if not (ndim == 3 and rk == 2 and limiter == 0):
        return None, None
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_step_kernels.md")))
    if not files:
        return None, None
    path = files[-1]
    cls = {"k_sweep_xy": "sweep_xy", "k_sweep_march<2": "sweep_z", "k_sweep_march<1": "sweep_y", "k_sweep_x<": "sweep_x",
           "k_ct_tma": "ct", "k_ct<": "ct", "k_dtmax": "dt_max"}
    acc = {}
    for line in open(path):
        m = re.match(r"\|\s*(k_[^|]+?)\s*\|(.+)\|\s*$", line)
        if not m:
            continue
        cells = [c.strip() for c in m.group(2).split("|")]
        if len(cells) < 10:
            continue
        name = m.group(1)
        key = next((v for k, v in cls.items() if name.startswith(k)), None)
        if key is None:
            continue
        try:
            rd, wr, dp = float(cells[1]), float(cells[2]), float(cells[9])
        except ValueError:
            continue
        acc.setdefault(key, []).append(((rd + wr) * 1e9, dp))
    out = {k: {"dram_bytes_per_launch": sum(x[0] for x in v) / len(v) * (zones / 256 ** 3),
               "fp64_instr_per_zone": sum(x[1] for x in v) / len(v)} for k, v in acc.items()}
    return out, os.path.relpath(path, ROOT)


def max_over_ranks(value, dist, device="cpu"):
    """a time measured on every rank -> the maximum over ranks (a job is as slow as its slowest replica)"""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(zones_per_rank, steps, ms_max, world):
    """whole-job zone-updates/s: every rank advances its slab of zones_per_rank zones, the job takes as
    long as its slowest rank"""
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


def oracle_run(w, steps, threads=None, rk=2, warmup=1, glm=False, uct=False):
    """the oracle as it stands on the host cores: `steps` whole steps of workload w; returns
    (zone-updates/s, threads used, seconds, per-step seconds)"""
    from oracle import Oracle
    o = Oracle()
    if threads:
        o.set_threads(threads)
    if glm:
        o.load_glm(w)
    else:
        o.load(w)
        if uct:
            assert o.set_emf(1) == 0
    o.set_integrator(rk)
    for _ in range(warmup):
        assert o.step(1) == 0                   # touch memory
    per = []
    for _ in range(steps):
        t0 = time.perf_counter()
        assert o.step(1) == 0
        per.append(time.perf_counter() - t0)
    cores = o.get_threads()
    o.finalize()
    return w.zones * steps / sum(per), cores, sum(per), per


def small_sample(cfg):
    """a smaller instance of configs[cfg] from the same generator, for the single-thread figure"""
    from paper_2511_20337_b200 import workloads as wl
    if cfg == 5:
        return wl.orszag_tang_3d(96, noise=1e-3), "orszag_tang_3d 96^3"
    if cfg in (3, 4):
        return wl.blast_3d(96, name="blast_3d_96"), "blast_3d 96^3, same recipe and seed as configs[3]"
    if cfg == 2:
        return wl.orszag_tang_2d(768), "orszag_tang_2d 768^2"
    return wl.config(cfg), f"configs[{cfg}] at full size"


def cpu_workload(cfg):
    """what the CPU legs step: the bench workload itself, except configs[4] (512^3: the oracle needs
    ~70 GB and 25 s per step), which is represented by configs[3] -- same recipe, 1/8 of the zones"""
    from paper_2511_20337_b200 import workloads as wl
    if cfg == 4:
        return wl.config(3), "configs[3] (256^3) standing in for configs[4]: same recipe and seed"
    return wl.config(cfg), "the bench workload itself, full size"


def scheme_of(w, rk, glm=False, uct=False):
    return "recon(%s)+HLLD+RK%d+%s, CFL %.2g" % (("minmod", "MC", "WENOZ")[w.limiter], rk,
                                                 "GLM" if glm else ("CT(UCT-HLLD)" if uct else "CT"), w.cfl)


def config_of(args, w, world):
    name = (f"configs[{args.config}] {w.name}" if args.config < 5 and not getattr(args, "grid", None)
            else f"paper section 4.1 workload (not a BASELINE config) {w.name}" if args.config == 5
            else f"recipe of configs[{args.config}] on another mesh (not a BASELINE config) {w.name}")
    return {"workload": name, "grid": [w.nx, w.ny, w.nz], "zones": w.zones, "scheme": scheme_of(w, args.rk, args.glm, args.uct),
            "l2": "inputs larger than L2 (state %.2f GB)" % (11 * w.zones * 8 / 1e9) if w.zones * 88 > 126e6
                  else "L2 flushed between timed repeats (a 256 MB buffer is rewritten); the state fits in L2",
            "parallelism": "single GPU" if world == 1 else "z-slab domain decomposition, one slab per GPU"}


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric / config keys (rank 0 only).  Each step
    is one whole oracle step of the bench workload (configs[3]: 256^3, ~3 s per step on 16 threads)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    w, what = cpu_workload(args.config)
    if args.wenoz:
        w.limiter = 2
    val, cores, secs, per = oracle_run(w, args.steps, rk=args.rk, warmup=max(1, min(args.warmup, 2)), glm=args.glm, uct=args.uct)
    from paper_2511_20337_b200 import workloads as wl
    wcfg = wl.config(args.config) if args.config != 4 else w
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_of(args, wcfg, 1),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{what}, {args.steps} steps, {secs:.1f} s; warm-up capped at 2 steps",
                         "best_step_s": min(per), "median_step_s": statistics.median(per)},
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
    ap.add_argument("--glm", action="store_true", help="GLM divergence cleaning (cell-centred B) instead of constrained transport")
    ap.add_argument("--uct", action="store_true", help="UCT-HLLD EMF average (reading R19) instead of the contact-mode rule (R6)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--repeats", type=int, default=3, help="timed repeats of the K steps (median and best reported)")
    ap.add_argument("--no-sustained", action="store_true", help="skip the one-second sustained-stepping figure")
    ap.add_argument("--grid", default=None, help="NXxNYxNZ: the recipe of --config 3/4/5 on another mesh (N = 1; not a BASELINE config)")
    ap.add_argument("--slab-path", action="store_true",
                    help="with --gpus 1: time the z-slab decomposed step (the N > 1 code path: SlabPluto, NCCL collectives on "
                         "the library's stream) with the whole box as the single slab of a one-rank group")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_2511_20337_b200 import workloads as wl
    from paper_2511_20337_b200.binding import Pluto

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA path has no CPU fallback")
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        return respawn_under_torchrun(args)          # plain `python bench.py --gpus N`: start the N ranks ourselves
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch one rank per GPU")
    if world > torch.cuda.device_count():
        raise SystemExit(f"bench.py: --gpus {world} needs {world} CUDA devices, this box has {torch.cuda.device_count()}")
    if world > 1 or args.slab_path:
        if "WORLD_SIZE" not in os.environ:           # --gpus 1 --slab-path: a one-rank NCCL group in this process
            os.environ.update({"MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(free_port()), "RANK": "0", "WORLD_SIZE": "1"})
        return main_slabs(args, rank, world, local)

    w = wl.config(args.config)
    if args.grid:
        # another mesh of the same recipe (context runs, e.g. the paper's per-GPU mesh 704x704x88 of Tab. 2,
        # PAPER.md:262-269): not a BASELINE.json config, and named as such in config.workload
        shape = tuple(int(t) for t in args.grid.lower().split("x"))
        if len(shape) != 3 or args.config not in (3, 4, 5):
            raise SystemExit("--grid NXxNYxNZ applies to the 3D recipes: --config 3, 4 (blast) or 5 (3D Orszag-Tang)")
        w = (wl.orszag_tang_3d(shape=shape, noise=1e-3, name="orszag_tang_3d_%dx%dx%d" % shape) if args.config == 5
             else wl.blast_3d(shape=shape, nsteps=20, name="blast_3d_%dx%dx%d" % shape))
    if args.wenoz:
        w.limiter = 2
    sim = Pluto(device=local)
    sim.set_integrator(args.rk)
    if args.uct:
        sim.set_emf(1)
    if args.glm:
        sim.load_glm(w)
    else:
        sim.load(w)
    K, W = args.steps, max(args.warmup, 3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    small = w.zones * 88 <= 126e6                 # the state fits in L2: flush it between repeats
    flush = torch.empty(256 * 2 ** 20, dtype=torch.uint8, device=sim.device) if small else None

    # ---------------- the fp64 peak, probed on the cold board before any stepping (and again at the very end)
    fp64_peak_first = sim.probe_fp64_gflops() * 0.5e9        # DFMA/s (2 flops each), register-resident loop

    # ---------------- burst figure: the first K-step window after the warm-up, before the board reaches its power limit
    sim.step(W)
    if flush is not None:
        flush.fill_(255)
    torch.cuda.synchronize()
    e0.record(sim.stream)
    sim.step_async(K)
    e1.record(sim.stream)
    sim.sync()
    torch.cuda.synchronize()
    burst_ms = e0.elapsed_time(e1)

    # ---------------- sustained figure: at least one second of continuous stepping (the board settles at its power
    # limit: DESIGN.md section 5), with its own clock / power samples.  It runs BEFORE the timed windows, so that
    # `value` is measured at the clock a long run has (the paper's runs last minutes).
    sustained = None
    if not args.no_sustained:
        n_s = max(K, min(5000, int(1.0 / (burst_ms / K * 1e-3)) + 1))
        s2 = ClockSampler(local)
        s2.start()
        ts0 = time.time()
        e0.record(sim.stream)
        sim.step_async(n_s)
        e1.record(sim.stream)
        sim.sync()
        torch.cuda.synchronize()
        c2 = s2.stop(ts0 + 0.3, time.time())
        sustained = {"steps": n_s, "ms_per_step": e0.elapsed_time(e1) / n_s, "clocks": c2}

    # ---------------- device-resident timing: K steps, state already in HBM; >= 3 repeats, back to back behind the
    # sustained run
    sampler = ClockSampler(local)
    sampler.start()
    times, launches = [], 0
    t0 = time.time()
    for rep_i in range(max(args.repeats, 1)):
        if flush is not None:
            flush.fill_(rep_i)
        torch.cuda.synchronize()
        l0 = sim.launch_count()
        e0.record(sim.stream)
        sim.step_async(K)
        e1.record(sim.stream)
        sim.sync()
        torch.cuda.synchronize()
        times.append(e0.elapsed_time(e1))
        launches = sim.launch_count() - l0
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    ms = statistics.median(times)
    value = w.zones * K / (ms * 1e-3)

    # ---------------- per-kernel timing (events around every launch) over about half a second of the same steps, with
    # the SM clock sampled meanwhile: the denominator of alu.frac_at_clock
    per_step_launches = max(1, launches // K)
    Kp = max(K, min(int(0.5 / (ms / K * 1e-3)) + 1, 8000 // per_step_launches))
    sim.profile(True)
    torch.cuda.synchronize()
    s3 = ClockSampler(local)
    s3.start()
    tp0 = time.time()
    e0.record(sim.stream)
    sim.step_async(Kp)
    e1.record(sim.stream)
    sim.sync()
    ms_prof = e0.elapsed_time(e1)
    clocks_prof = s3.stop(tp0, time.time())
    sim.profile(False)
    rep = sim.profile_report()
    total_kernel_ms = sum(v[0] for v in rep.values())
    dom = max(rep, key=lambda k: rep[k][0])
    dom_ms, dom_cnt = rep[dom]
    hbm_peak, peak_src = peaks()
    units = w.zones                              # zones one launch of the dominant kernel processes
    method, design = kernel_doubles(w.ndim, args.rk, args.glm)
    ncu, ncu_src = ncu_table(w.ndim, args.rk, w.limiter, units) if not (args.glm or args.uct) else (None, None)
    dur = dom_ms * 1e-3 / max(dom_cnt, 1)
    method_bytes = method.get(dom, 0) * 8 * units
    design_bytes = design.get(dom, 0) * 8 * units
    hbm_achieved = method_bytes / dur * 1e-9 if dur > 0 else 0.0
    hbm = {"bound": "hbm", "achieved": hbm_achieved, "peak": hbm_peak, "unit": "GB/s", "frac": hbm_achieved / hbm_peak,
           "algorithmic_bytes_per_launch": method_bytes, "algorithmic_doubles_per_zone": method.get(dom),
           "design_bytes_per_launch": design_bytes, "design_doubles_per_zone": design.get(dom),
           "design_frac": design_bytes / dur * 1e-9 / hbm_peak if dur > 0 else 0.0,
           "peak_source": peak_src}
    # the probe again, on the hot board; the roofline's peak is the LARGER of the two readings (a frac that cannot be
    # flattered by a denominator read under the power cap), both are printed
    fp64_peak_last = sim.probe_fp64_gflops() * 0.5e9
    fp64_peak = max(fp64_peak_first, fp64_peak_last)
    sms = torch.cuda.get_device_properties(sim.device).multi_processor_count
    alu = None
    if ncu and dom in ncu:
        rate = ncu[dom]["fp64_instr_per_zone"] * units / dur if dur > 0 else 0.0
        mhz = clocks_prof.get("sm_mhz")
        at_clock = sms * 64 * mhz * 1e6 if mhz else None
        alu = {"bound": "alu", "achieved": rate * 1e-12, "peak": fp64_peak * 1e-12, "unit": "T fp64-instr/s",
               "frac": rate / fp64_peak, "fp64_instr_per_zone": ncu[dom]["fp64_instr_per_zone"],
               "peak_probe_first": fp64_peak_first * 1e-12, "peak_probe_last": fp64_peak_last * 1e-12,
               "frac_at_clock": rate / at_clock if at_clock else None,
               "peak_at_clock": at_clock * 1e-12 if at_clock else None, "sm_mhz_profiled_pass": mhz,
               "peak_source": "max of two runs of pluto_probe_fp64_gflops (register-resident DFMA loop): before any stepping "
                              "and after the last pass; frac_at_clock = achieved / (%d SM x 64 lanes x the SM clock sampled "
                              "during the profiled pass); nominal %d x 64 x 1.965 GHz = %.1f T/s" % (sms, sms, sms * 64 * 1.965e-3)}
    # the roofline that binds the dominant kernel is the one it is closer to
    primary = alu if (alu and alu["frac"] > hbm["frac"]) else hbm
    roofline = dict(primary)
    roofline.update({"kernel": dom, "traffic": ncu[dom]["dram_bytes_per_launch"] if ncu and dom in ncu else None,
                     "traffic_source": ncu_src if ncu and dom in ncu else "no ncu capture of this scheme is committed",
                     "avg_launch_ms": dur * 1e3, "launches": dom_cnt, "share_of_step": dom_ms / total_kernel_ms,
                     "hbm": hbm, "alu": alu,
                     "kernels_ms_per_step": {k: v[0] / Kp for k, v in rep.items() if v[1]},
                     "profiled_ms_per_step": ms_prof / Kp, "profiled_steps": Kp, "profiled_clocks": clocks_prof})
    # the same two views for every kernel of the step
    roofline["all_kernels"] = {
        k: {"hbm_frac": round(method[k] * 8 * units / (v[0] * 1e-3 / v[1]) * 1e-9 / hbm_peak, 4),
            "design_hbm_frac": round(design[k] * 8 * units / (v[0] * 1e-3 / v[1]) * 1e-9 / hbm_peak, 4),
            "alu_frac": round(ncu[k]["fp64_instr_per_zone"] * units / (v[0] * 1e-3 / v[1]) / fp64_peak, 4) if ncu and k in ncu else None}
        for k, v in rep.items() if v[1] and k in method}
    # whole-step view: 320 B per zone-update against the HBM peak, and the step's fp64-pipe
    # instructions against the probed fp64 peak
    roofline["step_hbm_frac_at_320B"] = value * 320.0 / (hbm_peak * 1e9)
    if ncu:
        per_zu = sum(ncu[k]["fp64_instr_per_zone"] * (rep[k][1] / Kp) for k in ncu if k in rep and rep[k][1])
        roofline["step_fp64_instr_per_zone_update"] = per_zu
        roofline["step_alu_frac"] = value * per_zu / fp64_peak
        roofline["step_dram_bytes_per_zone_update"] = sum(ncu[k]["dram_bytes_per_launch"] * (rep[k][1] / Kp)
                                                          for k in ncu if k in rep and rep[k][1]) / units

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": config_of(args, w, world),
        "timing": {"repeats": len(times), "median_ms_per_step": ms / K, "best_ms_per_step": min(times) / K,
                   "all_ms_per_step": [t / K for t in times], "burst_ms_per_step": burst_ms / K,
                   "order": "warm-up, burst window, sustained run (>= 1 s), then the timed repeats back to back",
                   "sustained": sustained},
        "clocks": clocks, "gpu_launches": int(launches), "roofline": roofline,
    }

    # ---------------- end to end through the C ABI with HOST buffers
    Uh = torch.from_numpy(w.U).pin_memory()
    Bh = torch.from_numpy(w.Bface).pin_memory()
    Uo = torch.empty_like(Uh).pin_memory()
    Bo = torch.empty_like(Bh).pin_memory()
    Un, Bn, Uon, Bon = Uh.numpy(), Bh.numpy(), Uo.numpy(), Bo.numpy()
    sim.set_state(Un, Bn)
    sim.step(1)
    sim.get_state(Uon, Bon)
    torch.cuda.synchronize()
    tw0 = time.perf_counter()
    for _ in range(args.e2e_steps):
        sim.set_state(Un, Bn)               # host -> device inside the timed region
        sim.step(1)
        sim.get_state(Uon, Bon)             # device -> host read of the step's result
    torch.cuda.synchronize()
    te = (time.perf_counter() - tw0) / args.e2e_steps
    nbytes = (Uh.numel() + Bh.numel()) * 8
    # pluto_set_state does not copy U[4..6] of the active dimensions (the cell-centred B is the face mean)
    h2d = (Uh.numel() // 8 * (5 if w.nz > 1 else 6) + Bh.numel()) * 8
    line["e2e"] = {"value": w.zones / te, "unit": UNIT, "h2d_bytes_per_step": h2d,
                   "d2h_bytes_per_step": nbytes, "ms_per_step": te * 1e3, "steps": args.e2e_steps}
    sim.finalize()

    # ---------------- the oracle timed beside it (N = 1 only): the bench workload itself on every host
    # thread (3 steps), and a single-thread figure on a smaller instance of the same generator
    if not args.no_cpu_baseline:
        wc, what = cpu_workload(args.config)
        if args.wenoz:
            wc.limiter = 2
        v, cores, secs, per = oracle_run(wc, 3, rk=args.rk, glm=args.glm, uct=args.uct)
        ws, what1 = small_sample(args.config)
        if args.wenoz:
            ws.limiter = 2
        v1, _, secs1, _ = oracle_run(ws, 1, threads=1, rk=args.rk, warmup=0, glm=args.glm, uct=args.uct)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"{what}, 3 steps, {secs:.1f} s",
                                "best_step_s": min(per), "median_step_s": statistics.median(per),
                                "single_thread": {"value": v1, "cores": 1, "sample": f"{what1}, 1 step, {secs1:.1f} s"}}
    else:
        line["cpu_baseline"] = None
    print(json.dumps(line))


def free_port():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` with N > 1 and no launcher: re-execute under torch.distributed.run, one rank per
    GPU of this node; refuse loudly when the box has fewer devices (never time one GPU and call it N)"""
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} needs {args.gpus} CUDA devices, this box has {have}")
    os.environ.setdefault("NCCL_DEBUG", "INFO")      # the log names the ranks and the transport (NVLS / P2P)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__), *sys.argv[1:]]
    sys.stdout.flush()
    os.execv(sys.executable, cmd)


def main_slabs(args, rank, world, local):
    """N > 1: one z slab per rank (paper_2511_20337_b200.distributed.SlabPluto), weak scaling"""
    import torch
    import torch.distributed as dist
    from paper_2511_20337_b200 import workloads as wl
    from paper_2511_20337_b200.distributed import SlabPluto

    torch.cuda.set_device(local)
    dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if args.config not in (3, 4):
        raise SystemExit("--gpus N > 1 times the weak-scaling blast: per-GPU mesh and scheme of configs[3] (default) or configs[4]")
    base = wl.config(args.config)                    # scheme parameters and the per-GPU mesh
    nx, ny, nzl = base.nx, base.ny, base.nz
    nz = nzl * world
    sim = SlabPluto(dist, device=local)
    sim.set_integrator(args.rk)
    limiter = 2 if args.wenoz else base.limiter
    ghost = 3 if args.wenoz else 2
    U, Bl, box = wl.blast_3d_planes(nx, ny, nz, rank * nzl, nzl, nblast=world, gamma=base.gamma)
    sim.init(nx, ny, nz, ghost, base.gamma, base.cfl, limiter, box=box)
    assert (sim.k0, sim.nzl) == (rank * nzl, nzl)
    Uh, Bh = torch.from_numpy(U).pin_memory(), torch.from_numpy(Bl).pin_memory()
    sim.set_state(Uh.numpy(), Bh.numpy())
    K, W = args.steps, max(args.warmup, 3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sim.step(W)
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    times = []
    t0 = time.time()
    for _ in range(max(args.repeats, 1)):
        dist.barrier()
        torch.cuda.synchronize()
        l0 = sim.launch_count()
        e0.record(sim.stream)
        sim.step_async(K)
        e1.record(sim.stream)
        sim.sync()
        torch.cuda.synchronize()
        dist.barrier()
        times.append(max_over_ranks(e0.elapsed_time(e1), dist, "cuda"))
        launches = sim.launch_count() - l0
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    ms = statistics.median(times)
    zones = nx * ny * nzl
    value = aggregate_throughput(zones, K, ms, world)
    hbm_peak, peak_src = peaks()
    # end to end: every rank's planes from pinned host memory and back, every step
    tw0 = time.perf_counter()
    for _ in range(args.e2e_steps):
        sim.set_state(Uh.numpy(), Bh.numpy())
        sim.step(1)
        sim.get_state()
    torch.cuda.synchronize()
    te = max_over_ranks((time.perf_counter() - tw0) / args.e2e_steps, dist, "cuda")
    h2d = (U.size // 8 * 5 + Bl.size) * 8
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[%d] %s per GPU, box %dx%dx%d cut into %d z slabs (one blast per slab-sized section)"
                               % (args.config, base.name, nx, ny, nz, world),
                   "grid": [nx, ny, nz], "zones": zones * world, "zones_per_gpu": zones,
                   "scheme": scheme_of(base, args.rk) if not args.wenoz else scheme_of(base, args.rk).replace("minmod", "WENOZ").replace("MC", "WENOZ"),
                   "l2": "inputs larger than L2 (state %.2f GB per GPU)" % (11 * zones * 8 / 1e9),
                   "parallelism": "z-slab domain decomposition, one slab per GPU; ghost planes pulled from peer memory "
                                  "(CUDA IPC over NVLink) inside the ghost-fill kernel; 1 MAX all-reduce + %d barriers per step" % (args.rk - 1)},
        "timing": {"repeats": len(times), "median_ms_per_step": ms / K, "best_ms_per_step": min(times) / K},
        "clocks": clocks, "gpu_launches": int(launches),
        "roofline": {"bound": "hbm", "achieved": value / world * 320.0 * 1e-9, "peak": hbm_peak, "unit": "GB/s",
                     "frac": value / world * 320.0 / (hbm_peak * 1e9), "traffic": None, "peak_source": peak_src,
                     "note": "per-GPU whole-step view at the method's 320 B per zone-update; the per-kernel rooflines are those of the N = 1 line"},
        "e2e": {"value": world * zones / te, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": (U.size + Bl.size) * 8,
                "ms_per_step": te * 1e3, "steps": args.e2e_steps},
        "cpu_baseline": None,
    }
    sim.finalize()
    if rank == 0:
        print(json.dumps(line))
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
