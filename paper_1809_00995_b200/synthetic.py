"""Seeded synthetic inputs and the BASELINE.json configurations.

This module holds none of the method's arithmetic (no update, no estimator, no Philox): it only draws
generic random field snapshots with numpy's own generator and names the workloads, so both the CUDA path's
tests and the oracle's tests may use it.  The paper's workload is itself synthetic (random-phase field,
PAPER.md L72), produced on each side by its own Philox implementation; the snapshots below are for parity
tests that want a generic state (all ten fields non-zero) without running many steps first.
"""
from __future__ import annotations

import numpy as np

SEED_PRIMARY = 180900995

# BASELINE.json "configs", as parameter dictionaries (dx, dt, lambda0, e0, sigma, tau0 are common)
COMMON = dict(dx=0.5, dt=0.1, lambda0=2.0, e0=1.0, sigma=1.0, tau0=1.0)
CONFIGS = {
    1: dict(N=32, precision="f64", m=1.0, s=1.0, ic="random_phase", steps=100, diag_every=10),
    2: dict(N=256, precision="f32", m=1.0, s=0.0, ic="random_phase", steps=630, diag_every=20),
    3: dict(N=512, precision="f32", m=2.0, s=1.0, ic="gaussian", steps=1270, diag_every=20),
    4: dict(N=1024, precision="f32", m=1.0, s=0.0, ic="random_phase", steps=500, diag_every=50),
    5: dict(N=512, precision="f64", m=1.0, s=1.0, ic="random_phase", steps=60, diag_every=1),
}


def random_snapshot(N: int, seed: int, amp: float = 0.3) -> np.ndarray:
    """A generic smooth-ish snapshot, float64 (10, N, N, N): |phi| ~ 1 with random phase, Pi, theta, eps ~ amp * N(0,1)."""
    rng = np.random.default_rng(seed)
    shp = (N, N, N)
    mod = 1.0 + amp * rng.standard_normal(shp)
    ph = rng.uniform(0.0, 2.0 * np.pi, shp)
    f = np.empty((10,) + shp, dtype=np.float64)
    f[0] = mod * np.cos(ph)
    f[1] = mod * np.sin(ph)
    for k in range(2, 10):
        f[k] = amp * rng.standard_normal(shp)
    return f


def gauge_angles(N: int, seed: int, span: float = 10.0) -> np.ndarray:
    return np.random.default_rng(seed).uniform(-span, span, (N, N, N))
