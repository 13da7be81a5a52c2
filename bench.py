#!/usr/bin/env python
"""bench.py -- throughput of the Abelian-Higgs hot path (arXiv 1809.00995 Eqs. 4-7 + diagnostics) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--lattice 1024] [--precision f32]

One bench "step" is one pass of the whole hot path at BASELINE.json config 4's cadence: `--leapfrog` (50) fused
leapfrog launches (Eqs. 4-7) followed by one diagnostics pass (winding Eq. 11, <v^2>_L Eqs. 9-10,
Gauss residual) whose record is read back.  Default K = 10 -> the config's 500-step timed window.  The line printed
by rank 0 follows the driver's contract; see DESIGN.md "Measurement" for every field.

  value       site-updates/s, whole job, state resident in HBM, CUDA events on the handle's stream, max over ranks
  e2e         same metric through the C ABI with HOST buffers: ahs_set_fields_native_async (H2D of the 10 fields from pinned
              memory) + the same step + the diagnostics record read back (D2H), all inside the timing; two handles alternate so
              that one step's upload overlaps the other's evolution
  roofline    step kernel: 80 B (fp32) / 160 B (fp64) per site per launch / average launch duration (events around the
              back-to-back launches of each step), against MEASURED_PEAKS.json hbm_gbs
  cpu_baseline  the fp64 oracle (oracle/, test infrastructure) as it stands on this box's host cores, bounded sample

Multi-GPU: the path is one GPU per lattice (north_star); --gpus N runs N independent replicas (seed + rank), no
data-path collective ("replicas only"); torch.distributed is used for the barrier and the max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

COMMON = dict(dx=0.5, dt=0.1, lambda0=2.0, e0=1.0, sigma=1.0, tau0=1.0)
SEED = 180900995
BYTES_PER_SITE = {"f32": 80, "f64": 160}          # 10 values read + 10 written per site per step
FALLBACK_HBM_GBS = 6650.0                         # B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the step kernel from the committed `ncu --set full`
# captures (profiles/); keyed by (kernel, precision, lattice) -> (bytes, capture).  Absent = no capture for that configuration:
# the line then carries "traffic": null.  A capture is only listed while the kernel it was taken on is the one that ships
# (the capture names its commit).
NCU_TRAFFIC = {
    ("march", "f32", 1024): (89.21e9, "profiles/r6_step1024_f32_full.md (46.31 GB read + 42.90 GB written per launch; capture of the step kernel that ships)"),
    ("march", "f64", 512): (21.80e9, "profiles/r6_step512_f64_full.md (11.11 GB read + 10.69 GB written per launch; capture of the step kernel that ships)"),
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--lattice", type=int, default=1024, help="N of the N^3 lattice (config 4: 1024)")
    ap.add_argument("--precision", default="f32", choices=["f32", "f64"])
    ap.add_argument("--leapfrog", type=int, default=50, help="leapfrog launches per bench step (config 4: diagnostics every 50)")
    ap.add_argument("--m", type=float, default=1.0)
    ap.add_argument("--s", type=float, default=0.0)
    ap.add_argument("--tau-ref", type=float, default=0.0, help="a = (tau/tau_ref)^m; 0 = tau0 (DESIGN.md R3: s != 0 runs leave the "
                    "stability region after ~80 steps at m=1 unless tau_ref is the end time)")
    ap.add_argument("--kernel", default="auto", choices=["auto", "generic", "march"])
    ap.add_argument("--e2e-steps", type=int, default=10, help="timed end-to-end steps (each uploads the full state; the two-handle pipeline's "
                    "drain, one evolution without an upload behind it, is inside the timed region and is amortised over them)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--slabs", type=int, default=0, help="cut the lattice into this many z-slabs (ahs_group, DESIGN.md 10) driven by this one "
                    "process; 0 = one handle")
    ap.add_argument("--slab-devices", default="", help="comma-separated CUDA ordinals, one per slab (default: all on this rank's GPU)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the short runs of BASELINE configs 2, 3 and 5 that the default command adds")
    ap.add_argument("--cpu-lattice", type=int, default=128, help="lattice of the oracle's bounded sample")
    ap.add_argument("--cpu-leapfrog", type=int, default=10)
    return ap.parse_args()


# ------------------------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md recipe)
# ------------------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], None, [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for t, line in self.lines:
            if not (t0 <= t <= t1 + 0.3):
                continue
            c = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(c[0])); smax = float(c[1]); power.append(float(c[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax, "samples": len(sm),
                "power_w_max": max(power) if power else None, "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------------------------
# the oracle on the host cores: cpu_baseline leg and the --impl reference arm (the only places bench.py runs oracle/)
# ------------------------------------------------------------------------------------------------------------------
def oracle_sample(args, steps: int = 1, warmup: int = 0, threads: int = 1, lattice: int = 0) -> dict:
    """Time the fp64 oracle, as it stands, on a bounded sample of the workload: a lattice^3 lattice with the same physics,
    `cpu_leapfrog` leapfrog steps + one diagnostics pass per bench step, on `threads` host threads (0 = all cores online;
    the oracle's results do not depend on the thread count)."""
    import numpy as np
    from oracle import ahs_oracle as O
    N, L = lattice or args.cpu_lattice, args.cpu_leapfrog
    used = O.set_threads(threads)
    p = O.Params(N=N, m=args.m, s=args.s, tau_ref=args.tau_ref, **COMMON)
    f = O.initial_condition(p, SEED)
    if args.precision == "f32":
        f = np.ascontiguousarray(f.astype(np.float32).astype(np.float64))
    n = 0
    for _ in range(warmup):
        O.step(p, f, n, L); n += L
        O.diagnostics(p, f, n)
    t0 = time.perf_counter()
    for _ in range(steps):
        O.step(p, f, n, L); n += L
        d = O.diagnostics(p, f, n)
    dt = time.perf_counter() - t0
    O.set_threads(1)
    return {"value": N ** 3 * L * steps / dt, "unit": "site-updates/s", "cores": used, "kind": "oracle",
            "sample": "%d^3 lattice, same physics (m=%g, s=%g), %d x (%d leapfrog steps + 1 diagnostics), fp64, %d thread%s, %.1f s"
                      % (N, args.m, args.s, steps, L, used, "" if used == 1 else "s", dt),
            "seconds": dt, "n_pierced": int(d["n_pierced"]), "host_cores_online": os.cpu_count(), "cpu_model": cpu_model()}


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def run_reference(args):
    """--impl reference: for this tier the reference arm is the oracle on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    steps, warm = max(1, args.steps), max(0, args.warmup)
    # bound the whole run to a few minutes: ~0.3 us per site-update on one core, all cores are used
    while args.cpu_lattice ** 3 * args.cpu_leapfrog * (steps + warm) > 6e8 and args.cpu_leapfrog > 1:
        args.cpu_leapfrog = max(1, args.cpu_leapfrog // 2)
    while args.cpu_lattice ** 3 * args.cpu_leapfrog * (steps + warm) > 6e8 and args.cpu_lattice > 32:
        args.cpu_lattice //= 2
    r = oracle_sample(args, steps=steps, warmup=warm, threads=0)     # all host cores
    # the config names what this arm RAN (a bounded fp64 sample of the workload on the host cores), and which workload it samples
    target = workload_config(args)
    config = {"workload": "bounded sample on the host cores: %d^3 periodic lattice, f64, same physics, %d leapfrog steps + 1 diagnostics per "
                          "bench step -- a sample of: %s" % (args.cpu_lattice, args.cpu_leapfrog, target["workload"]),
              "lattice": args.cpu_lattice, "leapfrog_per_step": args.cpu_leapfrog, "diagnostics_per_step": 1,
              "sample": r["sample"], "workload_lattice": target["lattice"], "workload_leapfrog_per_step": target["leapfrog_per_step"],
              "parallelism": "host threads x%d (rank 0 only)" % r["cores"]}
    line = {
        "impl": "reference", "metric": "lattice site-updates/sec per leapfrog step", "value": r["value"], "unit": "site-updates/s",
        "n_gpus": args.gpus, "steps": steps, "warmup": warm, "ms_per_step": 1e3 * r["seconds"] / steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config,
        "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
        "e2e": {"value": r["value"], "unit": "site-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(args) -> dict:
    N = args.lattice
    name = {1024: "BASELINE.json configs[3]", 256: "BASELINE.json configs[1]", 512: "BASELINE.json configs[2]/[4]"}.get(N, "custom")
    return {"workload": "%d^3 periodic lattice, %s, dx=0.5 dt=0.1 lambda=2 e=1 sigma=1 tau0=1, a~tau^%g, s=%g, random-phase IC "
                        "(Philox seed %d); %d leapfrog steps + 1 diagnostics per bench step (%s)%s"
                        % (N, args.precision, args.m, args.s, SEED, args.leapfrog, name, ", tau_ref=%g" % args.tau_ref if args.tau_ref else ""),
            "lattice": N, "leapfrog_per_step": args.leapfrog, "diagnostics_per_step": 1,
            "l2": "inputs larger than L2 (%.1f GB of fields streamed per leapfrog launch)" % (N ** 3 * BYTES_PER_SITE[args.precision] / 1e9),
            "parallelism": ("z-slabs x%d on devices [%s] of one process (one lattice, exchange inside the step kernel)" % (args.slabs, args.slab_devices)
                            if args.gpus > 1 and int(os.environ.get("WORLD_SIZE", "1")) == 1 and args.slabs else
                            "replicas x%d" % args.gpus + (", each lattice cut into %d z-slabs on devices [%s]" % (args.slabs, args.slab_devices or "this rank's GPU")
                                                          if args.slabs else ""))}


# ------------------------------------------------------------------------------------------------------------------
# our arm: the CUDA path through the C ABI binding
# ------------------------------------------------------------------------------------------------------------------
def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy kernel)"
    except (OSError, KeyError, ValueError):
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------------------------------------------------------
# multi-rank host logic ("replicas only"): no data-path collective; torch.distributed carries the barrier
# and the max over ranks of the device-timed window.  Backend-agnostic so that tests/test_bench_host.py can run it with
# gloo, world_size 2, on CPU.
# ------------------------------------------------------------------------------------------------------------------
def max_over_ranks(x: float, world: int, device="cpu") -> float:
    if world == 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, sites: int, leapfrog: int, steps: int, total_ms: float) -> float:
    """site-updates/s of the whole job: every rank advanced its own replica by leapfrog*steps steps in total_ms (max over ranks)."""
    return world * sites * leapfrog * steps / (total_ms * 1e-3)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1809_00995_b200 import binding as ahs

    rank, world, local = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_ranks(x: float) -> float:
        return max_over_ranks(x, world, "cuda")

    N, L, K, W = args.lattice, args.leapfrog, args.steps, args.warmup
    sites = N ** 3
    # ONE process asked for several GPUs (no torchrun: WORLD_SIZE unset): the lattice is cut into z-slabs over them (ahs_group,
    # DESIGN.md 10) -- total work fixed, "strong" scaling.  Under torchrun every rank keeps a whole lattice of its own (replicas).
    strong = world == 1 and args.gpus > 1
    if strong:
        if torch.cuda.device_count() < args.gpus:
            raise SystemExit("bench.py --gpus %d in one process cuts the lattice into z-slabs over %d GPUs, but this box has %d; "
                             "launch it with torchrun for independent replicas" % (args.gpus, args.gpus, torch.cuda.device_count()))
        args.slabs = args.slabs or args.gpus
        if not args.slab_devices:
            args.slab_devices = ",".join(str(i * args.gpus // args.slabs) for i in range(args.slabs))   # contiguous blocks of slabs per GPU
    if args.slabs:
        devs = [int(d) for d in args.slab_devices.split(",")] if args.slab_devices else [local] * args.slabs
        sim = ahs.Group(N=N, nslabs=args.slabs, devices=devs, precision=args.precision, m=args.m, s=args.s, seed=SEED + rank,
                        tau_ref=args.tau_ref, **COMMON)
        sim.kernel_kind = "march"
        args.no_e2e = True                 # (the end-to-end leg is the single-handle path)
    else:
        sim = ahs.Simulation(N=N, precision=args.precision, m=args.m, s=args.s, seed=SEED + rank, kernel=args.kernel, tau_ref=args.tau_ref, **COMMON)
    diag = None
    for _ in range(W):
        sim.step(L)
        diag = sim.diagnostics()

    ev = lambda: torch.cuda.Event(enable_timing=True)
    marks = [(ev(), ev(), ev()) for _ in range(K)]
    barrier()
    clocks = ClockSampler(local)
    clocks.start()
    launches0 = sim.kernel_launches
    t0 = time.time()
    start, stop = ev(), ev()
    start.record()
    for a, b, c in marks:
        a.record()
        sim.step(L)                 # L fused leapfrog launches, asynchronous
        if args.slabs:
            sim.synchronize()       # the slabs run on their own streams: bring their work in front of the event
        b.record()
        diag = sim.diagnostics()    # diagnostics kernels + the record to the host (synchronises)
        c.record()
    stop.record()
    barrier()
    t1 = time.time()
    clk = clocks.stop(t0, t1)
    launches = sim.kernel_launches - launches0
    per_device = None
    if args.slabs:
        per_device = {}
        for d, n in zip(devs, sim.launches_per_slab()):
            per_device[str(d)] = per_device.get(str(d), 0) + int(n)     # (since creation: IC and warm-up launches included)
    total_ms = max_ranks(start.elapsed_time(stop))
    step_ms = sum(a.elapsed_time(b) for a, b, _ in marks)       # the leapfrog launches only
    diag_ms = sum(b.elapsed_time(c) for _, b, c in marks)
    value = whole_job_value(world, sites, L, K, total_ms)       # (z-slabs in one process: world = 1, ONE lattice on args.gpus GPUs)

    launch_s = step_ms * 1e-3 / (K * L)
    peak, peak_src = measured_peak()
    achieved = BYTES_PER_SITE[args.precision] * sites / launch_s / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": NCU_TRAFFIC.get((sim.kernel_kind, args.precision, N), (None, None))[0],
                "traffic_source": NCU_TRAFFIC.get((sim.kernel_kind, args.precision, N), (None, "no ncu capture for this configuration"))[1],
                "kernel": "fused leapfrog step (%s)" % sim.kernel_kind, "peak_source": peak_src,
                "bytes_per_launch": BYTES_PER_SITE[args.precision] * sites, "launch_ms": launch_s * 1e3,
                "frac_of_nominal_8TBps": achieved / 8000.0,
                "diagnostics_ms_per_call": diag_ms / K, "diagnostics_in_steps": (diag_ms / K) / (launch_s * 1e3),
                "diagnostics_GBps": (BYTES_PER_SITE[args.precision] // 2) * sites / (diag_ms / K * 1e-3) / 1e9,
                "diagnostics_overhead_at_this_cadence": diag_ms / step_ms}

    e2e = None
    if not args.no_e2e:
        e2e = run_e2e(args, sim, torch, max_ranks, barrier, world)

    line = {
        "metric": "lattice site-updates/sec per leapfrog step", "value": value, "unit": "site-updates/s", "n_gpus": args.gpus if strong else world,
        "steps": K, "warmup": W, "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "strong" if strong else "weak",
        "vs_baseline": None, "dtype": args.precision, "data": "synthetic", "config": workload_config(args),
        "roofline": roofline, "clocks": clk, "gpu_launches": int(launches),
        "ms_per_leapfrog_step": launch_s * 1e3, "step_only_site_updates_per_s": sites / launch_s,
        "kernel": sim.kernel_kind,
        "last_diagnostics": {k: diag[k] for k in ("step", "n_pierced", "xi", "v2", "gauss_max", "gauss_rhs_rms", "nonfinite")} if diag else None,
    }
    if e2e is not None:
        line["e2e"] = e2e
    if per_device is not None:
        line["gpu_launches_per_device_since_create"] = per_device
        line["slab_faces_by_copies"] = sim.copied_faces
    sim.destroy()
    default_workload = (N, args.precision, L, args.m, args.s, args.kernel, args.slabs) == (1024, "f32", 50, 1.0, 0.0, "auto", 0)
    if rank == 0 and world == 1 and default_workload and not args.no_other_configs:
        line["other_configs"] = other_configs(torch)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        # the oracle on all host cores (a sample twice as wide: ~10 s) and, beside it, on one core
        r = oracle_sample(args, threads=0, lattice=2 * args.cpu_lattice)
        one = oracle_sample(args, threads=1)
        line["cpu_baseline"] = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample", "host_cores_online", "cpu_model")}
        line["cpu_baseline"]["one_core"] = {k: one[k] for k in ("value", "unit", "cores", "sample")}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def other_configs(torch):
    """BASELINE.json's remaining marching configurations (2: 256^3 fp32, 3: 512^3 fp32 matter s = 1 Gaussian IC, 5: 512^3 fp64), each run whole
    at its own diagnostics cadence with the state resident in HBM and timed with CUDA events on the handle's stream, so that their step times stand
    beside the headline in the same driver-run line.  They are not the bench value (config 4 is): context, a few seconds in total.
    Config 3 takes a = (tau / tau_end)^m: read literally (tau_ref = tau0) its s = 1 leaves the leapfrog stability region after ~27 steps (R3)."""
    from paper_1809_00995_b200 import binding as ahs
    from paper_1809_00995_b200.synthetic import CONFIGS
    peak, _ = measured_peak()
    ev = lambda: torch.cuda.Event(enable_timing=True)
    out = []
    for c in (2, 3, 5):
        cfg = CONFIGS[c]
        steps, every, N = cfg["steps"], max(cfg["diag_every"], 1), cfg["N"]
        tau_ref = COMMON["tau0"] + steps * COMMON["dt"] if c == 3 else 0.0
        with ahs.Simulation(N=N, precision=cfg["precision"], m=cfg["m"], s=cfg["s"], ic=cfg["ic"], seed=SEED, tau_ref=tau_ref, **COMMON) as sim:
            sim.step(min(every, 10))                       # warm-up (part of the run: the step count goes on)
            sim.diagnostics()
            t_step = t_diag = 0.0
            done, calls, d = 0, 0, None
            while done < steps:
                n = min(every, steps - done)
                a, b, e = ev(), ev(), ev()
                a.record(); sim.step(n); b.record()
                d = sim.diagnostics()
                e.record()
                torch.cuda.synchronize()
                t_step += a.elapsed_time(b); t_diag += b.elapsed_time(e)
                done += n; calls += 1
                if d["nonfinite"]:
                    break
            bps = BYTES_PER_SITE[cfg["precision"]] * N ** 3 * done / (t_step * 1e-3) / 1e9
            out.append({"config": c, "lattice": N, "precision": cfg["precision"], "m": cfg["m"], "s": cfg["s"], "ic": cfg["ic"], "tau_ref": tau_ref or COMMON["tau0"],
                        "steps": done, "diagnostics_calls": calls, "kernel": sim.kernel_kind, "ms_per_leapfrog_step": t_step / done,
                        "site_updates_per_s": N ** 3 * done / (t_step * 1e-3), "achieved_GBps": bps, "frac_of_measured_copy": bps / peak,
                        "diagnostics_ms_per_call": t_diag / calls, "diagnostics_overhead_at_its_cadence": t_diag / t_step,
                        "nonfinite": int(d["nonfinite"]), "n_pierced_last": int(d["n_pierced"]), "gauss_max_last": d["gauss_max"]})
    return out


def run_e2e(args, sim, torch, max_over_ranks, barrier, world):
    """The same step through the C ABI with HOST buffers: every timed step uploads its 10 input fields from pinned host memory
    (ahs_set_fields_native_async), runs L leapfrog launches + diagnostics and reads the diagnostics record back to the host.
    With room for a second lattice in HBM the steps alternate between two handles on two streams, so the upload of step k+1
    overlaps the evolution of step k (an input pipeline through the public API); otherwise they run back to back on one handle."""
    from paper_1809_00995_b200 import binding as ahs
    N, L, E = args.lattice, args.leapfrog, max(1, args.e2e_steps)
    sites = N ** 3
    tdtype = torch.float32 if args.precision == "f32" else torch.float64
    try:
        host = torch.empty((10, N, N, N), dtype=tdtype, pin_memory=True)
    except RuntimeError as exc:
        return {"value": None, "unit": "site-updates/s", "error": "pinned host allocation failed: %s" % str(exc)[:120]}
    n0 = sim.step_count
    sim.get_fields_native(host.data_ptr())            # the resident state, downloaded once (untimed)
    h2d = host.numel() * host.element_size()
    import ctypes
    d2h = ctypes.sizeof(ahs.ahs_diag)

    sims = [sim]
    free, _ = torch.cuda.mem_get_info()
    if free > ahs.required_bytes(N, args.precision) + (4 << 30):
        with torch.cuda.stream(torch.cuda.Stream()):
            sims.append(ahs.Simulation(N=N, precision=args.precision, m=args.m, s=args.s, ic="none", kernel=args.kernel,
                                       tau_ref=args.tau_ref, **COMMON))

    def submit(k):
        sm = sims[k % len(sims)]
        sm.set_fields_native(host.data_ptr(), step=n0, wait=False)   # H2D of this step's inputs, asynchronous on the handle's stream
        sm.step(L)
        sm.diagnostics_launch()

    def collect(k):
        return sims[k % len(sims)].diagnostics_fetch()               # D2H of the record; synchronises that handle's stream

    def run(n):
        submit(0)
        for k in range(1, n):
            submit(k)
            collect(k - 1)
        return collect(n - 1)

    run(len(sims))                                    # warm-up on every handle
    barrier()
    w0 = time.perf_counter()
    last = run(E)
    torch.cuda.synchronize()
    wall = time.perf_counter() - w0
    barrier()
    ms = max_over_ranks(1e3 * wall)                   # host clock between two device synchronisations: the copies are part of it
    for sm in sims[1:]:
        sm.destroy()
    del host
    return {"value": world * sites * L * E / (ms * 1e-3), "unit": "site-updates/s", "h2d_bytes_per_step": h2d,
            "d2h_bytes_per_step": d2h, "steps": E, "ms_per_step": ms / E, "handles": len(sims), "n_pierced_last": int(last["n_pierced"]),
            "what": "per step: ahs_set_fields_native_async (pinned host -> HBM) + %d x ahs_step + ahs_diagnostics_launch/_fetch (record -> host); "
                    "%s" % (L, "two handles on two streams, upload of one step overlapping the evolution of the other"
                            if len(sims) == 2 else "one handle, back to back (no room for a second lattice)")}


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
