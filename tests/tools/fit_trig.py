#!/usr/bin/env python
"""fit_trig.py -- generator and checker of the polynomial coefficients in ahs_trig.cuh (CUDA path only).

    python tests/tools/fit_trig.py          # fit, print the constants, emulate and report max errors

The marching kernels use branch-free sine / cosine / arctangent (ahs_trig.cuh).  Their polynomials are fitted here by
Lawson-reweighted least squares on Chebyshev nodes (an approximation of the minimax fit) -- nothing is copied from a
library -- and each routine is then emulated in numpy with every operation rounded to fp32 (products and sums are
formed exactly in fp64 and rounded once, which is what an fp32 FMA does up to double rounding) and compared with the
fp64 numpy function.  tests/test_trig_constants.py runs the emulation against the constants that are compiled into
the header, so a mistyped digit fails on the CPU box.  This file is not imported by the library and shares nothing
with oracle/.
"""
from __future__ import annotations

import re
import os
import numpy as np

f32 = np.float32
HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "..", "..", "paper_1809_00995_b200", "csrc")


def lawson(fun, lo, hi, powers, n=4000, iters=80, rel=False):
    """c minimising max |sum_k c_k x^p_k - fun(x)| (relative to fun if rel) on [lo, hi]."""
    k = np.arange(n)
    x = 0.5 * (lo + hi) + 0.5 * (hi - lo) * np.cos(np.pi * (k + 0.5) / n)
    A = np.stack([x ** p for p in powers], 1)
    y = fun(x)
    if rel:
        A, y = A / y[:, None], np.ones_like(y)
    w = np.ones(n)
    for _ in range(iters):
        sw = np.sqrt(w)
        c = np.linalg.lstsq(A * sw[:, None], y * sw, rcond=None)[0]
        e = np.abs(A @ c - y)
        w = w * np.maximum(e, 1e-300)
        w /= w.sum()
    return c, float(np.abs(A @ c - y).max())


def fma(a, b, c):
    """fp32 fused multiply-add emulated through fp64 (exact product of two fp32 values, one rounding of the sum)."""
    return (a.astype(np.float64) * np.asarray(b, np.float64) + np.asarray(c, np.float64)).astype(f32)


def header_constants(name: str):
    """The float literals inside `name(...) { ... }` of ahs_trig.cuh, in order of appearance."""
    src = open(os.path.join(CSRC, "ahs_trig.cuh")).read()
    i = src.index(name)
    j = src.index("\n}\n", i)
    return [float(v) for v in re.findall(r"(-?\d+\.\d+(?:e[-+]?\d+)?)f\b", src[i:j])]


def header_constants64(name: str):
    """The double literals inside `name(...) { ... }` of ahs_trig.cuh, in order of appearance."""
    src = open(os.path.join(CSRC, "ahs_trig.cuh")).read()
    i = src.index(name)
    j = src.index("\n}\n", i)
    return [float(v) for v in re.findall(r"(?<![\w.])(-?\d+\.\d+(?:e[-+]?\d+)?)(?![\w.])", src[i:j])]


# ---- emulations of the device routines (same operation order as ahs_trig.cuh) -------------------------------------------
def emu_sincos(x, k):
    two_over_pi, magic, c1, c2, s3, s2, s1, q3, q2, q1, q0 = k[0], k[1], k[3], k[4], k[5], k[6], k[7], k[8], k[9], k[10], k[11]
    x = x.astype(f32)
    t = fma(x, f32(two_over_pi), f32(magic))
    q = t.view(np.int32)
    kk = (t - f32(magic)).astype(f32)
    r = fma(kk, f32(c1), x)
    r = fma(kk, f32(c2), r)
    z = (r * r).astype(f32)
    ps = fma(z, f32(s3), f32(s2))
    ps = fma(z, ps, f32(s1))
    sr = fma((r * z).astype(f32), ps, r)
    pc = fma(z, f32(q3), f32(q2))
    pc = fma(z, pc, f32(q1))
    pc = fma(z, pc, f32(q0))
    cr = fma(z, pc, f32(1.0))
    odd = (q & 1).astype(bool)
    so, co = np.where(odd, cr, sr), np.where(odd, sr, cr)
    s = np.where((q & 2) != 0, -so, so)
    c = np.where(((q + 1) & 2) != 0, -co, co)
    return s, c


def emu_sin(x, k):
    """sin_core + sign: k = constants of `void sin_core(W x`."""
    inv_pi, magic, c1, c2, p5, p4, p3, p2, p1 = k[0], k[1], k[3], k[4], k[5], k[6], k[7], k[8], k[9]
    x = x.astype(f32)
    t = fma(x, f32(inv_pi), f32(magic))
    q = t.view(np.int32)
    kk = (t - f32(magic)).astype(f32)
    r = fma(kk, f32(c1), x)
    r = fma(kk, f32(c2), r)
    z = (r * r).astype(f32)
    p = fma(z, f32(p5), f32(p4))
    for c in (p3, p2, p1):
        p = fma(z, p, f32(c))
    sr = fma((r * z).astype(f32), p, r)
    return np.where((q & 1) != 0, -sr, sr)


def emu_atan2_turns(y, x, k, rcp_ulps=1.0, rng=None):
    """atan2_turns: k = the float constants of `float2 atan2_turns(float2 y` (8 polynomial coefficients, 1/4, 1/2).
    The hardware reciprocal (MUFU.RCP, <= 1 ulp) is emulated as the rounded exact reciprocal perturbed by up to rcp_ulps."""
    y, x = y.astype(f32), x.astype(f32)
    ax, ay = np.abs(x), np.abs(y)
    mx, mn = np.maximum(ax, ay), np.minimum(ax, ay)
    rc = (1.0 / mx.astype(np.float64)).astype(f32)
    if rng is not None:
        rc = (rc.astype(np.float64) * (1.0 + rcp_ulps * 2.0 ** -23 * rng.uniform(-1, 1, rc.shape))).astype(f32)
    q = (mn * rc).astype(f32)
    z = (q * q).astype(f32)
    p = np.full_like(z, f32(k[0]))
    for c in k[1:8]:
        p = fma(z, p, f32(c))
    r = (q * p).astype(f32)
    r = np.where(ay > ax, (f32(k[8]) - r).astype(f32), r)
    r = np.where(x < 0, (f32(k[9]) - r).astype(f32), r)
    return np.copysign(r, y)


def emu_sincos64(x, ks):
    """sincos_fast(double): the reduction constants of trig64::reduce are exact splits of pi/2; the polynomial constants `ks`
    (6 sine, 6 cosine; the cosine's leading 1 - z/2 is separate) are evaluated here in long double so that only the FIT is tested."""
    ld = np.longdouble
    x = x.astype(ld)
    k = np.rint(x * ld(2) / ld(np.pi))
    r = (x - k * ld(1.5707963267948966) - k * ld(6.123233995736766e-17)).astype(ld)
    z = r * r
    ps = ld(ks[0])
    for c in ks[1:6]:
        ps = z * ps + ld(c)
    sr = r * z * ps + r
    pc = ld(ks[6])
    for c in ks[7:12]:
        pc = z * pc + ld(c)
    cr = z * z * pc + (ld(1) - z / 2)
    q = k.astype(np.int64)
    odd = (q & 1).astype(bool)
    so, co = np.where(odd, cr, sr), np.where(odd, sr, cr)
    return np.where((q & 2) != 0, -so, so), np.where(((q + 1) & 2) != 0, -co, co)


def main():
    rng = np.random.default_rng(1)
    # ---- fits -----------------------------------------------------------------------------------------------------
    c, e = lawson(lambda q: np.arctan(q) / (2 * np.pi), 0.0, 1.0, [2 * i + 1 for i in range(8)])
    print("atan(q) / 2 pi, q in [0,1], odd degree 15: max abs error %.2e turns" % e)
    print("  coefficients (highest power first):", ", ".join("%.17gf" % f32(v) for v in c[::-1]))
    c, e = lawson(lambda r: np.sin(r) / r, 1e-9, np.pi / 4, [0, 2, 4, 6], rel=True)
    print("sin(r)/r on [0, pi/4], even degree 6: max rel error %.2e" % e, c)
    c, e = lawson(np.cos, 0.0, np.pi / 4, [0, 2, 4, 6, 8])
    print("cos(r) on [0, pi/4], even degree 8: max abs error %.2e" % e, c)
    c, e = lawson(lambda r: np.sin(r) / r, 1e-9, np.pi / 2, [0, 2, 4, 6, 8, 10], rel=True)
    print("sin(r)/r on [0, pi/2], even degree 10: max rel error %.2e" % e, c)
    # ---- the constants that are compiled in, emulated ------------------------------------------------------------------
    x = np.concatenate([rng.uniform(-20, 20, 2_000_000), rng.uniform(-1e3, 1e3, 200_000)]).astype(f32)
    s, cc = emu_sincos(x, header_constants("void sincos_core(W x"))
    xs = x.astype(np.float64)
    print("sincos_fast fp32 emulation: max abs error sin %.2e cos %.2e" % (np.abs(s - np.sin(xs)).max(), np.abs(cc - np.cos(xs)).max()))
    ph = rng.uniform(-np.pi, np.pi, 4_000_000)
    rad = np.exp(rng.uniform(-3, 3, ph.size))
    yy, xx = (rad * np.sin(ph)).astype(f32), (rad * np.cos(ph)).astype(f32)
    a = emu_atan2_turns(yy, xx, header_constants("float2 atan2_turns(float2 y")[:10], rng=rng)
    ref = np.arctan2(yy.astype(np.float64), xx.astype(np.float64)) / (2 * np.pi)
    print("atan2_turns fp32 emulation: max abs error %.2e turns (the winding fast path assumes <= 7.6e-8)" % np.abs(a - ref).max())
    sn = emu_sin(x, header_constants("void sin_core(W x"))
    print("sin_fast fp32 emulation: max abs error %.2e" % np.abs(sn - np.sin(xs)).max())


if __name__ == "__main__":
    main()
