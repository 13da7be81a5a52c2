"""The s = 0 rows of the paper's Table 4 through the C ABI: asymptotic slopes of the mean string
separation and late-time mean square velocities, 512^3, five seeds per era (L224).

    python -m paper_1809_00995_b200.table4 [--lattice 512] [--seeds 5] [--fit-from 64]

For each era (radiation a ~ tau, matter a ~ tau^2) and seed: random-phase initial condition, evolution to half a
light-crossing time (tau = 1 + N dx / 2 ... the paper's 1280 steps at 512^3, L64, L166), diagnostics every 10 steps;
d xi / d tau by a least-squares line over tau in [fit_from, tau_end] (the paper does not state its fit window: this one is
ours and is printed), velocities averaged over the same window.  Mean and sample standard deviation over the seeds, one
JSON line per era.  Printing and line fitting only: every number comes from libahs.
"""
from __future__ import annotations

import argparse
import json

import numpy as np

from . import binding as ahs
from .synthetic import COMMON

PAPER = {  # PAPER.md Table 4 (L211-222), s = 0 rows: context, five-run averages on a Quadro P5000
    "radiation": {"xi_L_dot": "0.30 +- 0.02", "xi_W_dot": "0.32 +- 0.03", "v2_V": "0.34 +- 0.01", "v2_L": "0.31 +- 0.01", "v2_omega": "0.32 +- 0.01"},   # L215
    "matter": {"xi_L_dot": "0.29 +- 0.01", "xi_W_dot": "0.29 +- 0.02", "v2_V": "0.26 +- 0.01", "v2_L": "0.27 +- 0.01", "v2_omega": "0.25 +- 0.01"},      # L222
}


def run(N, m, seed, steps, every, fit_from, precision, c_B, c_E=0.0, s_schedule=(), tau_ref=0.0, diag_trig=None):
    tau, series = [], {k: [] for k in ("xi", "xi_L", "v2", "v2_V", "v2_omega", "gauss_max")}
    with ahs.Simulation(N=N, precision=precision, m=m, s=0.0, seed=seed, c_B=c_B, c_E=c_E, tau_ref=tau_ref, **COMMON) as sim:
        if s_schedule:
            sim.set_s_schedule(s_schedule)
        if diag_trig is not None:
            sim.set_option(ahs.AHS_OPT_DIAG_TRIG, diag_trig)
        for n in range(0, steps + 1, every):
            if n:
                sim.step(every)
            d = sim.diagnostics()
            tau.append(d["tau"])
            for k in series:
                series[k].append(d[k])
    tau = np.array(tau)
    sel = tau >= fit_from
    out = {}
    for k in ("xi", "xi_L"):
        y = np.array(series[k])[sel]
        out[k + "_dot"] = float(np.polyfit(tau[sel], y, 1)[0])
    for k in ("v2", "v2_V", "v2_omega"):
        out[k] = float(np.mean(np.array(series[k])[sel]))
    out["gauss_max"] = float(np.max(series["gauss_max"]))
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--lattice", type=int, default=512)
    ap.add_argument("--seeds", type=int, default=5)
    ap.add_argument("--fit-from", type=float, default=64.0)
    ap.add_argument("--every", type=int, default=10)
    ap.add_argument("--precision", default="f32")
    ap.add_argument("--c-b", type=float, default=0.0, help="factor on the plaquette sum of Eq. 2 in the weight (0 = 1, DESIGN.md R2; Eq. 2 prints 0.5)")
    ap.add_argument("--c-e", type=float, default=0.0, help="factor on the electric term of Eq. 2 in the weight (0 = 1; 0.04 = (dt/dx)^2, L44 read literally, DESIGN.md R21)")
    ap.add_argument("--s-schedule", default="", help="'tau:s,tau:s,...' piecewise-linear s(tau) instead of s = 0 (ahs_set_s_schedule, DESIGN.md R23), "
                    "e.g. core growth then the true equations: '1:-1,40:-1,48:1'")
    ap.add_argument("--tau-ref", type=float, default=0.0, help="a = (tau/tau_ref)^m; 0 = tau0.  With s = 1 at the end use the end time (R3)")
    ap.add_argument("--eras", default="radiation,matter")
    ap.add_argument("--diag-trig", default="hardware", choices=["hardware", "polynomial"],
                    help="AHS_OPT_DIAG_TRIG: where an fp32 lattice's diagnostics evaluate the sines / cosines of their sums (DESIGN.md 7.2)")
    args = ap.parse_args()
    sched = tuple(tuple(float(v) for v in kv.split(":")) for kv in args.s_schedule.split(",") if kv)
    N = args.lattice
    steps = int(round(N * COMMON["dx"] / 2 / COMMON["dt"]))          # half a light-crossing time of the box
    steps -= steps % args.every
    for era, m in (("radiation", 1.0), ("matter", 2.0)):
        if era not in args.eras.split(","):
            continue
        trig = ahs.AHS_TRIG_HARDWARE if args.diag_trig == "hardware" else ahs.AHS_TRIG_POLYNOMIAL
        runs = [run(N, m, seed, steps, args.every, args.fit_from, args.precision, args.c_b, args.c_e, sched, args.tau_ref, trig) for seed in range(1, args.seeds + 1)]
        line = {"era": era, "m": m, "s": 0.0, "lattice": N, "precision": args.precision, "seeds": args.seeds, "steps": steps, "diag_trig": args.diag_trig, "c_B": args.c_b or 1.0,
                "c_E": args.c_e or 1.0, "s_schedule": sched or "s = 0", "tau_ref": args.tau_ref or COMMON["tau0"],
                "fit_window_tau": [args.fit_from, COMMON["tau0"] + steps * COMMON["dt"]], "paper_table4": PAPER[era]}
        for k, name in (("xi_L_dot", "xi_L_dot"), ("xi_dot", "xi_W_dot"), ("v2_V", "v2_V"), ("v2", "v2_L"), ("v2_omega", "v2_omega")):
            v = np.array([r[k] for r in runs])
            line[name] = {"mean": float(v.mean()), "std": float(v.std(ddof=1)) if len(v) > 1 else 0.0}
        line["gauss_max_over_all_runs"] = max(r["gauss_max"] for r in runs)
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
