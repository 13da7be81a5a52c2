"""Sweep the launch-shape options of the z-marching kernels (ahs_set_option) on the current GPU.

    python -m paper_1809_00995_b200.tune --lattice 512 --precision f32
    python -m paper_1809_00995_b200.tune --lattice 1024 --step-chunks 0,16,32,64 --diag-chunks 0,8,16,32

For each candidate number of z-chunks per tile (0 = the library's default) the fused leapfrog step and the diagnostics pass
are timed with CUDA events on the handle's stream (best of `--reps` windows, candidates visited twice in opposite orders so
that clock drift does not favour a position) and one JSON line is printed per kernel:
{"kernel", "lattice", "precision", "us_per_launch": {chunks: microseconds}, "best", "of_measured_copy": {...}}.
Argument marshalling and timing only: every number comes from libahs.  The defaults compiled into the library
(ahs_step_march.cu / ahs_diag_march.cu: pick_chunks) were read off this sweep; profiles/r4_chunks.md keeps its output.
"""
from __future__ import annotations

import argparse
import json
import os

from . import binding as ahs
from .synthetic import COMMON, SEED_PRIMARY

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def measured_copy_gbs() -> float:
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"])
    except (OSError, KeyError, ValueError):
        return 6650.0          # B200_PROFILING.md fallback


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--lattice", type=int, default=512)
    ap.add_argument("--precision", default="f32", choices=["f32", "f64"])
    ap.add_argument("--step-chunks", default="0,8,16,32,64")
    ap.add_argument("--diag-chunks", default="0,8,16,32,64")
    ap.add_argument("--steps", type=int, default=0, help="leapfrog launches per timed window (0: ~30 ms worth)")
    ap.add_argument("--reps", type=int, default=3)
    args = ap.parse_args()

    import torch
    N, prec = args.lattice, args.precision
    bytes_step = N ** 3 * (80 if prec == "f32" else 160)
    nst = args.steps or max(2, int(30e-3 / (bytes_step / 5.5e12)))
    ev = lambda: torch.cuda.Event(enable_timing=True)
    peak = measured_copy_gbs()

    with ahs.Simulation(N=N, precision=prec, m=1.0, s=0.0, seed=SEED_PRIMARY, **COMMON) as sim:
        if sim.kernel_kind != "march":
            raise SystemExit("N = %d runs on the one-thread-per-site kernels: nothing to tune" % N)
        sim.step(20)

        def time_step():
            best = float("inf")
            for _ in range(args.reps):
                a, b = ev(), ev()
                a.record(); sim.step(nst); b.record()
                torch.cuda.synchronize()
                best = min(best, a.elapsed_time(b) / nst)
            return best * 1e3

        def time_diag():
            best = float("inf")
            for _ in range(args.reps):
                a, b = ev(), ev()
                a.record()
                for _ in range(4):
                    sim.diagnostics_launch()
                b.record()
                torch.cuda.synchronize()
                sim.diagnostics_fetch()
                best = min(best, a.elapsed_time(b) / 4)
            return best * 1e3

        for kernel, option, cands, timer, nbytes in (
                ("step", ahs.AHS_OPT_STEP_CHUNKS, args.step_chunks, time_step, bytes_step),
                ("diagnostics", ahs.AHS_OPT_DIAG_CHUNKS, args.diag_chunks, time_diag, bytes_step // 2)):
            cands = [int(c) for c in cands.split(",") if c != ""]
            us = {}
            for c in cands + cands[::-1]:
                if c > N:
                    continue
                sim.set_option(option, c)
                timer()                                      # settle
                us[c] = min(us.get(c, float("inf")), timer())
            sim.set_option(option, 0)
            best = min(us, key=us.get)
            print(json.dumps({"kernel": kernel, "lattice": N, "precision": prec, "launches_per_window": nst if kernel == "step" else 4,
                              "us_per_launch": {str(k): round(v, 1) for k, v in us.items()}, "best": best,
                              "of_measured_copy": {str(k): round(nbytes / v / 1e3 / peak, 4) for k, v in us.items()},
                              "peak_GBps": peak}), flush=True)


if __name__ == "__main__":
    main()
