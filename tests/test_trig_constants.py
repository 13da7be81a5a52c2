"""The polynomial constants compiled into csrc/ahs_trig.cuh (CUDA path), emulated in fp32 on the CPU by
csrc/fit_trig.py: a mistyped digit or a dropped reduction term fails here, without a GPU.  Host logic of the CUDA
path only -- nothing of oracle/ is involved."""
import importlib.util
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
spec = importlib.util.spec_from_file_location("fit_trig", os.path.join(HERE, "..", "paper_1809_00995_b200", "csrc", "fit_trig.py"))
fit_trig = importlib.util.module_from_spec(spec)
spec.loader.exec_module(fit_trig)


def test_sincos_fast_fp32_constants():
    rng = np.random.default_rng(3)
    x = np.concatenate([rng.uniform(-20, 20, 400_000), rng.uniform(-1e3, 1e3, 100_000), [0.0, np.pi / 4, -np.pi / 4, 1e-8]]).astype(np.float32)
    s, c = fit_trig.emu_sincos(x, fit_trig.header_constants("void sincos_core(W x"))
    xs = x.astype(np.float64)
    assert np.abs(s - np.sin(xs)).max() < 1.2e-7 and np.abs(c - np.cos(xs)).max() < 1.2e-7


def test_atan2_fast_constants_stay_inside_the_winding_error_budget():
    rng = np.random.default_rng(4)
    ph = rng.uniform(-np.pi, np.pi, 500_000)
    rad = np.exp(rng.uniform(-3, 3, ph.size))
    y, x = (rad * np.sin(ph)).astype(np.float32), (rad * np.cos(ph)).astype(np.float32)
    a = fit_trig.emu_atan2(y, x, fit_trig.header_constants("float atan2_fast(float y"))
    ref = np.arctan2(y.astype(np.float64), x.astype(np.float64))
    assert np.abs(a - ref).max() < 4.8e-7      # ahs_diag_march.cu budgets 6e-7 rad per phase
    # octants and axes
    for yy, xx in ((0.0, 1.0), (1.0, 0.0), (0.0, -1.0), (-1.0, 0.0), (1.0, 1.0), (-1.0, -1.0), (1.0, -1.0)):
        got = fit_trig.emu_atan2(np.array([yy]), np.array([xx]), fit_trig.header_constants("float atan2_fast(float y"))[0]
        assert abs(abs(got) - abs(np.arctan2(yy, xx))) < 4.8e-7
