"""Run one of the BASELINE.json configurations through the C ABI and print its diagnostics series.

    python -m paper_1809_00995_b200.run_config 2                 # 256^3 fp32, radiation, s=0, to tau=64, diagnostics every 20
    python -m paper_1809_00995_b200.run_config 3 --tau-ref end   # 512^3 fp32 matter s=1 with a normalised at the end time
    python -m paper_1809_00995_b200.run_config 5 --steps 60      # 512^3 fp64, step-only vs diagnostics after every step

One JSON line per diagnostics call ({"step", "tau", "xi", "v2", "n_pierced", "gauss_max", ...}) and a final summary line
with the device-timed window (CUDA events through torch on the handle's stream).  Argument marshalling and printing only:
every number comes from libahs.  s != 0 configurations read literally (a = (tau/tau0)^m) leave the leapfrog stability
region (R3); the run stops at the first non-finite diagnostics and says so.
"""
from __future__ import annotations

import argparse
import json
import math

from . import binding as ahs
from .synthetic import COMMON, CONFIGS, SEED_PRIMARY


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config", type=int, choices=sorted(CONFIGS))
    ap.add_argument("--steps", type=int, default=0, help="override the number of steps")
    ap.add_argument("--diag-every", type=int, default=0)
    ap.add_argument("--tau-ref", default="0", help="'end' = tau at the last step, or a number; 0 = tau0")
    ap.add_argument("--seed", type=int, default=SEED_PRIMARY)
    ap.add_argument("--quiet", action="store_true", help="only the summary line")
    args = ap.parse_args()

    import torch
    cfg = dict(CONFIGS[args.config])
    steps = args.steps or cfg["steps"]
    every = args.diag_every or cfg["diag_every"]
    tau_end = COMMON["tau0"] + steps * COMMON["dt"]
    tau_ref = tau_end if args.tau_ref == "end" else float(args.tau_ref)
    sim = ahs.Simulation(N=cfg["N"], precision=cfg["precision"], m=cfg["m"], s=cfg["s"], ic=cfg["ic"], seed=args.seed,
                         tau_ref=tau_ref, **COMMON)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    t_step, t_diag, series, stopped = 0.0, 0.0, [], None
    d = sim.diagnostics()
    series.append(d)
    done = 0
    while done < steps and stopped is None:
        n = min(every, steps - done)
        a, b, c = ev(), ev(), ev()
        a.record()
        sim.step(n)
        b.record()
        d = sim.diagnostics()
        c.record()
        torch.cuda.synchronize()
        t_step += a.elapsed_time(b)
        t_diag += b.elapsed_time(c)
        done += n
        series.append(d)
        if d["nonfinite"]:
            stopped = done
    if not args.quiet:
        for d in series:
            print(json.dumps({k: (None if isinstance(v, float) and not math.isfinite(v) else v) for k, v in d.items()}))
    sites = cfg["N"] ** 3
    bytes_site = 80 if cfg["precision"] == "f32" else 160
    last = next((x for x in reversed(series) if not x["nonfinite"]), series[0])
    print(json.dumps({
        "summary": "config %d" % args.config, "lattice": cfg["N"], "precision": cfg["precision"], "m": cfg["m"], "s": cfg["s"], "ic": cfg["ic"],
        "tau_ref": tau_ref or COMMON["tau0"], "steps_done": done, "diag_calls": len(series) - 1, "kernel": sim.kernel_kind,
        "first_nonfinite_step": stopped, "ms_per_step": t_step / max(done, 1), "ms_per_diag": t_diag / max(len(series) - 1, 1),
        "site_updates_per_s": sites * done / (t_step * 1e-3) if t_step else None,
        "step_GBps": bytes_site * sites * done / (t_step * 1e-3) / 1e9 if t_step else None,
        "diag_overhead": t_diag / t_step if t_step else None,
        "last_finite": {k: last[k] for k in ("step", "tau", "n_pierced", "xi", "v2", "mean_lagrangian", "gauss_max", "gauss_rhs_rms")},
    }))
    sim.destroy()


if __name__ == "__main__":
    main()
