"""The polynomial constants compiled into csrc/ahs_trig.cuh (CUDA path), emulated on the CPU by tests/tools/fit_trig.py:
a mistyped digit or a dropped reduction term fails here, without a GPU.  Host logic of the CUDA path only -- nothing of
oracle/ is involved."""
import importlib.util
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
spec = importlib.util.spec_from_file_location("fit_trig", os.path.join(HERE, "tools", "fit_trig.py"))
fit_trig = importlib.util.module_from_spec(spec)
spec.loader.exec_module(fit_trig)


def test_sincos_fast_fp32_constants():
    rng = np.random.default_rng(3)
    x = np.concatenate([rng.uniform(-20, 20, 400_000), rng.uniform(-1e3, 1e3, 100_000), [0.0, np.pi / 4, -np.pi / 4, 1e-8]]).astype(np.float32)
    s, c = fit_trig.emu_sincos(x, fit_trig.header_constants("void sincos_core(W x"))
    xs = x.astype(np.float64)
    assert np.abs(s - np.sin(xs)).max() < 1.2e-7 and np.abs(c - np.cos(xs)).max() < 1.2e-7


def test_sin_fast_fp32_constants():
    rng = np.random.default_rng(5)
    x = np.concatenate([rng.uniform(-20, 20, 400_000), rng.uniform(-1e3, 1e3, 100_000), [0.0, np.pi / 2, -np.pi / 2, 1e-8]]).astype(np.float32)
    s = fit_trig.emu_sin(x, fit_trig.header_constants("void sin_core(W x"))
    assert np.abs(s - np.sin(x.astype(np.float64))).max() < 1.8e-7            # <= 1.9 ulp at |sin| ~ 1 (ahs_trig.cuh)


def test_chord_is_the_sine_polynomial_with_power_of_two_scaled_constants():
    """chord_fast (the magnetic term of the diagnostics) = sin_core<W, 1>: the constants of sin_core scaled by the exact powers of
    two of HalfAngle<1> (read from the header).  Emulated, it must be twice sin_core at x/2 bit for bit up to its sign, hence
    |chord| = 2 |sin(x/2)| within twice the sine's bound."""
    import re
    src = open(os.path.join(fit_trig.CSRC, "ahs_trig.cuh")).read()
    m = re.search(r"inv = HALF \? ([\d.]+)f : 1\.0f, pi = HALF \? ([\d.]+)f : 1\.0f;\s*\n\s*static constexpr float q1 = HALF \? ([\d.]+)f : 1\.0f", src)
    inv, pi2, q1 = (float(g) for g in m.groups())
    assert (inv, pi2, q1) == (0.5, 2.0, 0.25)
    k = fit_trig.header_constants("void sin_core(W x")
    scaled = list(k)
    scaled[0] = k[0] * inv                                   # 1 / 2 pi
    scaled[3], scaled[4] = k[3] * pi2, k[4] * pi2            # the two-term split of 2 pi
    for j, power in zip((5, 6, 7, 8, 9), (5, 4, 3, 2, 1)):   # c_i / 4^i, highest degree first
        scaled[j] = k[j] * q1 ** power
    assert all(np.float32(v) == v or abs(np.float32(v) - v) <= abs(v) * 2.0 ** -24 for v in scaled)
    rng = np.random.default_rng(8)
    x = np.concatenate([rng.uniform(-20, 20, 400_000), rng.uniform(-300, 300, 100_000), [0.0, np.pi, -np.pi, 1e-8]]).astype(np.float32)
    chord = fit_trig.emu_sin(x, [np.float32(v) for v in scaled])
    half = fit_trig.emu_sin((x * np.float32(0.5)).astype(np.float32), k)
    assert np.array_equal(np.abs(chord), np.abs(2.0 * half).astype(np.float32))
    assert np.abs(np.abs(chord) - 2.0 * np.abs(np.sin(0.5 * x.astype(np.float64)))).max() < 3.6e-7


def test_atan2_turns_constants_stay_inside_the_winding_error_budget():
    rng = np.random.default_rng(4)
    ph = rng.uniform(-np.pi, np.pi, 500_000)
    rad = np.exp(rng.uniform(-3, 3, ph.size))
    y, x = (rad * np.sin(ph)).astype(np.float32), (rad * np.cos(ph)).astype(np.float32)
    k = fit_trig.header_constants("float2 atan2_turns(float2 y")[:10]      # 8 coefficients, 1/4, 1/2 (then the 0.0f of x < 0)
    assert k[8] == 0.25 and k[9] == 0.5
    a = fit_trig.emu_atan2_turns(y, x, k, rcp_ulps=1.0, rng=rng)
    ref = np.arctan2(y.astype(np.float64), x.astype(np.float64)) / (2 * np.pi)
    assert np.abs(a - ref).max() < 7.6e-8      # ahs_diag_march.cu budgets eps_a <= 7.6e-8 turns per phase
    # octants and axes
    for yy, xx in ((0.0, 1.0), (1.0, 0.0), (0.0, -1.0), (-1.0, 0.0), (1.0, 1.0), (-1.0, -1.0), (1.0, -1.0)):
        got = fit_trig.emu_atan2_turns(np.array([yy]), np.array([xx]), k)[0]
        assert abs(abs(got) - abs(np.arctan2(yy, xx)) / (2 * np.pi)) < 7.6e-8


def test_sincos_fast_fp64_polynomials():
    """The fp64 fits (sincos_fast(double), also the coefficient sets sin_fast(double) selects by quadrant parity): evaluated
    in long double so that only the polynomials are under test; <= 1e-16 absolute on the reduced interval."""
    rng = np.random.default_rng(6)
    x = np.concatenate([rng.uniform(-20, 20, 200_000), [0.0, np.pi / 4, -np.pi / 4, 1e-9, 3.0]])
    k = fit_trig.header_constants64("void sincos_fast(double x")
    # 6 sine coefficients, 6 cosine coefficients, then the -0.5 and 1.0 of the cosine's leading terms
    assert len(k) >= 14 and k[12] == -0.5 and k[13] == 1.0
    s, c = fit_trig.emu_sincos64(x, k[:12])
    ref_s, ref_c = np.sin(x.astype(np.longdouble)), np.cos(x.astype(np.longdouble))
    assert float(np.abs(s - ref_s).max()) < 1.2e-16 and float(np.abs(c - ref_c).max()) < 1.2e-16
    # sin_fast(double) carries the same ten constants, chosen by the parity of the quadrant
    k2 = fit_trig.header_constants64("double sin_fast(double x")
    assert sorted(k2[:12]) == sorted(k[:12])
