// ahs_trig.cuh -- branch-free sine / cosine for the marching kernels (fp32 and fp64), accurate to ~1-2 ulp.
//
// Why not libdevice sincosf/sinf: the step is issue-bound as much as HBM-bound, six
// transcendental evaluations per site are half of its instructions, and every libdevice call carries a
// Payne-Hanek slow path whose branch (BSSY/BSYNC) stalls instruction fetch and bloats the loop past the
// instruction cache (seen on the first marching kernel of round 1; no profile of that version was kept).  Why not
// the __sinf/__cosf intrinsics: their absolute
// error (2^-21) is what PAPER.md L142 reports as degrading the diagnostics.  So: Cody-Waite reduction with a
// two-term (fp32) / three-term (fp64) split of pi/2 (or pi) carried by FMAs, then minimax-style polynomials on the reduced interval.
//
//   sincos_fast(x): k = rint(x * 2/pi), r = x - k*pi/2 in [-pi/4, pi/4]; sin and cos polynomials; quadrant fix-up.
//   sin_fast(x)   : fp32: k = rint(x / pi), r in [-pi/2, pi/2], odd polynomial, sign (-1)^k;
//                   fp64: the quadrant form with the coefficient set chosen by the parity of k.
// Measured against fp64 references (tests/tools/fit_trig.py): fp32 sincos <= 0.9 ulp, fp32 sin <= 1.9 ulp
// (abs 1.2e-7), fp64 <= 1.3 ulp.  Domain: |x| < 2^22 * pi/2 (fp32: 6.5e6; fp64: |x| < 2^30); beyond it the result
// is finite garbage or NaN (a link angle that large has no phase information left in fp32 anyway); NaN and Inf
// inputs give NaN, so blown-up lattices still reach the diagnostics' non-finite flag.
// The polynomial coefficients were fitted by tests/tools/fit_trig.py (least squares on Chebyshev nodes, relative
// weighting), not copied from a library.
#pragma once
#include <cuda_runtime.h>

namespace ahs {

// ---- fp32 ---------------------------------------------------------------------------------------------------------------
// The arithmetic is written once over a lane type W: float, or float2 evaluated with Blackwell's packed fp32
// instructions (FFMA2 / FMUL2 / FADD2 on sm_100: two IEEE fp32 operations per issued instruction, constants broadcast from
// immediates).  Both give bit-identical results per lane; the marching kernels use the packed form on pairs of sites,
// which takes a quarter of the instructions out of the step kernel's trigonometry (profiles/HISTORY.md r3).
namespace lanes {
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ float mul_(float a, float b) { return a * b; }
__device__ __forceinline__ float add_(float a, float b) { return a + b; }
__device__ __forceinline__ float2 fma_(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 mul_(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 add_(float2 a, float2 b) { return __fadd2_rn(a, b); }
template <typename W> __device__ __forceinline__ W all(float v);
template <> __device__ __forceinline__ float all<float>(float v) { return v; }
template <> __device__ __forceinline__ float2 all<float2>(float v) { return make_float2(v, v); }
}  // namespace lanes

// t = x * 2/pi + 1.5 * 2^23 (its low mantissa bits hold k = rint(x * 2/pi)); sr = sin(r), cr = cos(r), r = x - k pi/2
template <typename W>
__device__ __forceinline__ void sincos_core(W x, W& t, W& sr, W& cr)
{
    using namespace lanes;
    t = fma_(x, all<W>(0.6366197466850281f), all<W>(12582912.0f));
    const W k = add_(t, all<W>(-12582912.0f));
    W r = fma_(k, all<W>(-1.5707963705062866f), x);
    r = fma_(k, all<W>(4.371138828673793e-08f), r);   // (a third term, 1.7e-15 k, is below fp32 resolution over the whole domain)
    const W z = mul_(r, r);
    W ps = fma_(z, all<W>(-0.00019513866573106498f), all<W>(0.00833214819431305f));
    ps = fma_(z, ps, all<W>(-0.16666653752326965f));
    sr = fma_(mul_(r, z), ps, r);
    W pc = fma_(z, all<W>(2.438912088109646e-05f), all<W>(-0.0013886747183278203f));
    pc = fma_(z, pc, all<W>(0.04166662320494652f));
    pc = fma_(z, pc, all<W>(-0.5f));
    cr = fma_(z, pc, all<W>(1.0f));
}
// quadrant k mod 4 = 0: (sr, cr), 1: (cr, -sr), 2: (-sr, -cr), 3: (-cr, sr): one sign word (bit 1 of k) on both, then the
// odd quadrants swap and negate -- the negation rides on the select
__device__ __forceinline__ void sincos_quadrant(float t, float sr, float cr, float& s, float& c)
{
    const int q = __float_as_int(t);
    const int sgn = (q << 30) & 0x80000000;
    const float X = __int_as_float(__float_as_int(sr) ^ sgn), Y = __int_as_float(__float_as_int(cr) ^ sgn);
    const bool odd = q & 1;
    s = odd ? Y : X;
    c = odd ? -X : Y;
}
__device__ __forceinline__ void sincos_fast(float x, float& s, float& c)
{
    float t, sr, cr;
    sincos_core<float>(x, t, sr, cr);
    sincos_quadrant(t, sr, cr, s, c);
}
__device__ __forceinline__ void sincos_fast(float2 x, float2& s, float2& c)
{
    float2 t, sr, cr;
    sincos_core<float2>(x, t, sr, cr);
    sincos_quadrant(t.x, sr.x, cr.x, s.x, c.x);
    sincos_quadrant(t.y, sr.y, cr.y, s.y, c.y);
}

// t = x / pi + 1.5 * 2^23; sr = sin(r), r = x - k pi in [-pi/2, pi/2]; sin x = (-1)^k sr.
// HALF = 1 evaluates the same polynomial at x/2 without ever forming x/2: every constant is scaled by an exact power of
// two (HalfAngle), k = rint(x / 2 pi), r = x - 2 pi k in [-pi, pi] and sr = 2 sin(r/2) -- bit for bit twice what HALF = 0
// returns for x/2; 2 sin(x/2) = (-1)^k sr.
template <int HALF> struct HalfAngle {
    static constexpr float inv = HALF ? 0.5f : 1.0f, pi = HALF ? 2.0f : 1.0f;
    static constexpr float q1 = HALF ? 0.25f : 1.0f, q2 = q1 * q1, q3 = q2 * q1, q4 = q3 * q1, q5 = q4 * q1;   // c_i -> c_i / 4^i
};
template <typename W, int HALF = 0>
__device__ __forceinline__ void sin_core(W x, W& t, W& sr)
{
    using namespace lanes;
    using H = HalfAngle<HALF>;
    t = fma_(x, all<W>(0.31830987334251404f * H::inv), all<W>(12582912.0f));
    const W k = add_(t, all<W>(-12582912.0f));
    W r = fma_(k, all<W>(-3.1415927410125732f * H::pi), x);
    r = fma_(k, all<W>(8.742277657347586e-08f * H::pi), r);
    const W z = mul_(r, r);
    W p = fma_(z, all<W>(-2.388586395341008e-08f * H::q5), all<W>(2.752518867055187e-06f * H::q4));
    p = fma_(z, p, all<W>(-0.00019840864115394652f * H::q3));
    p = fma_(z, p, all<W>(0.008333330973982811f * H::q2));
    p = fma_(z, p, all<W>(-0.1666666716337204f * H::q1));
    sr = fma_(mul_(r, z), p, r);
}
__device__ __forceinline__ float sin_fast(float x)
{
    float t, sr;
    sin_core<float>(x, t, sr);
    return __int_as_float(__float_as_int(sr) ^ (__float_as_int(t) << 31));
}
__device__ __forceinline__ float2 sin_fast(float2 x)
{
    float2 t, sr;
    sin_core<float2>(x, t, sr);
    return make_float2(__int_as_float(__float_as_int(sr.x) ^ (__float_as_int(t.x) << 31)),
                       __int_as_float(__float_as_int(sr.y) ^ (__float_as_int(t.y) << 31)));
}

// the chord of the angle x on the unit circle up to its sign: +- |exp(i x) - 1| = +- 2 sin(x/2).  Only its square
// 2 (1 - cos x) is used (the magnetic term of Eq. 2), so the sign fix-up of sin_fast and the halving of x are left out.
__device__ __forceinline__ float2 chord_fast(float2 x)
{
    float2 t, sr;
    sin_core<float2, 1>(x, t, sr);
    return sr;
}

// ---- the special-function unit's sine / cosine (MUFU.SIN / MUFU.COS behind one multiplication by 1/2pi), two lanes ------------
// Absolute error <= 2^-21.4 (sine) / 2^-21.2 (cosine) for |x| <= pi; beyond, the unit sees x / 2 pi rounded to fp32, i.e. a
// phase error of about |x| 2^-23 -- the rounding an fp32 angle of that size carries anyway.  NaN and Inf give NaN.  Used by the
// diagnostics' <v^2> sums only (AHS_TRIG_HARDWARE), never by the step or the winding.
__device__ __forceinline__ float2 sin_hw(float2 x)
{
    float2 r;
    asm("sin.approx.ftz.f32 %0, %1;" : "=f"(r.x) : "f"(x.x));
    asm("sin.approx.ftz.f32 %0, %1;" : "=f"(r.y) : "f"(x.y));
    return r;
}
__device__ __forceinline__ void sincos_hw(float2 x, float2& s, float2& c)
{
    s = sin_hw(x);
    asm("cos.approx.ftz.f32 %0, %1;" : "=f"(c.x) : "f"(x.x));
    asm("cos.approx.ftz.f32 %0, %1;" : "=f"(c.y) : "f"(x.y));
}

// arg(x + i y) / 2 pi, in turns, for the winding fast path (ahs_diag_march.cu): two values at once, branch-free.
// q = min/max in [0, 1] (MUFU.RCP and a multiply), odd polynomial of degree 15 in q fitted to atan(q) / 2 pi, then the
// octant fix-ups, whose constants 1/4 and 1/2 are exact in turns.  Absolute error <= 5e-8 turns in the fp32 emulation of
// tests/tools/fit_trig.py (the fast path's error budget assumes <= 7.6e-8 turns = 4.8e-7 rad).  atan2_turns(0, 0) and
// non-finite inputs give NaN, which sends the link to the fp64 evaluation.  Range: max(|x|, |y|) < 2^126 -- above it the approximate
// reciprocal flushes to zero and q = 0 comes out without a NaN, so such a link is NOT re-evaluated (field values of that size, 10^38
// times the vacuum expectation value, also overflow every sum of the pass; include/ahs.h states the range at n_pierced).
__device__ __forceinline__ float rcp_approx(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float2 atan2_turns(float2 y, float2 x)
{
    using namespace lanes;
    const float ax0 = fabsf(x.x), ay0 = fabsf(y.x), ax1 = fabsf(x.y), ay1 = fabsf(y.y);
    const float2 mn = make_float2(fminf(ax0, ay0), fminf(ax1, ay1));
    const float2 q = mul_(mn, make_float2(rcp_approx(fmaxf(ax0, ay0)), rcp_approx(fmaxf(ax1, ay1))));
    const float2 z = mul_(q, q);
    float2 p = fma_(z, all<float2>(-0.00064530421514064074f), all<float2>(0.0034795976243913174f));
    p = fma_(z, p, all<float2>(-0.0088987238705158234f));
    p = fma_(z, p, all<float2>(0.015346035361289978f));
    p = fma_(z, p, all<float2>(-0.022136272862553596f));
    p = fma_(z, p, all<float2>(0.031745944172143936f));
    p = fma_(z, p, all<float2>(-0.053046122193336487f));
    p = fma_(z, p, all<float2>(0.15915483236312866f));
    float2 r = mul_(q, p);
    const float2 r4 = add_(all<float2>(0.25f), make_float2(-r.x, -r.y));
    r = make_float2(ay0 > ax0 ? r4.x : r.x, ay1 > ax1 ? r4.y : r.y);
    const float2 r2 = add_(all<float2>(0.5f), make_float2(-r.x, -r.y));
    r = make_float2(x.x < 0.0f ? r2.x : r.x, x.y < 0.0f ? r2.y : r.y);
    return make_float2(copysignf(r.x, y.x), copysignf(r.y, y.y));
}

// ---- fp64 ---------------------------------------------------------------------------------------------------------------
namespace trig64 {
__device__ __forceinline__ double reduce(double x, int& q)
{
    const double t = fma(x, 0.6366197723675814, 6755399441055744.0);   // 1.5 * 2^52
    q = __double2loint(t);
    const double k = t - 6755399441055744.0;
    double r = fma(k, -1.5707963267948966, x);
    r = fma(k, -6.123233995736766e-17, r);
    r = fma(k, 1.4973849048591698e-33, r);
    return r;
}
__device__ __forceinline__ double flip(double v, int bit)   // negate v if bit 1 of `bit` is set
{
    return __hiloint2double(__double2hiint(v) ^ ((bit << 30) & 0x80000000), __double2loint(v));
}
}  // namespace trig64

__device__ __forceinline__ void sincos_fast(double x, double& s, double& c)
{
    int q;
    const double r = trig64::reduce(x, q);
    const double z = r * r;
    double ps = fma(z, 1.5895906110388965e-10, -2.505074159906586e-08);
    ps = fma(z, ps, 2.7557313577062805e-06);
    ps = fma(z, ps, -0.00019841269829441296);
    ps = fma(z, ps, 0.008333333333321893);
    ps = fma(z, ps, -0.1666666666666663);
    const double sr = fma(r * z, ps, r);
    double pc = fma(z, -1.1359191040163257e-11, 2.087571361252908e-09);
    pc = fma(z, pc, -2.755731427353126e-07);
    pc = fma(z, pc, 2.480158728917463e-05);
    pc = fma(z, pc, -0.0013888888888873554);
    pc = fma(z, pc, 0.041666666666666595);
    const double cr = fma(z * z, pc, fma(z, -0.5, 1.0));
    const double X = trig64::flip(sr, q), Y = trig64::flip(cr, q);   // same quadrant logic as the fp32 version
    const bool odd = q & 1;
    s = odd ? Y : X;
    c = odd ? -X : Y;
}

__device__ __forceinline__ double sin_fast(double x)
{
    int q;
    const double r = trig64::reduce(x, q);
    const double z = r * r;
    const bool odd = q & 1;
    double p = fma(z, odd ? -1.1359191040163257e-11 : 1.5895906110388965e-10, odd ? 2.087571361252908e-09 : -2.505074159906586e-08);
    p = fma(z, p, odd ? -2.755731427353126e-07 : 2.7557313577062805e-06);
    p = fma(z, p, odd ? 2.480158728917463e-05 : -0.00019841269829441296);
    p = fma(z, p, odd ? -0.0013888888888873554 : 0.008333333333321893);
    p = fma(z, p, odd ? 0.041666666666666595 : -0.1666666666666663);
    const double base = odd ? fma(z, -0.5, 1.0) : r;
    const double mult = (odd ? z : r) * z;
    return trig64::flip(fma(mult, p, base), q);
}

// ---- V values at once (the V sites of a thread): fp32 goes through the packed two-lane form, fp64 one by one ------------
template <int V>
__device__ __forceinline__ void sincos_vec(const float (&x)[V], float (&s)[V], float (&c)[V])
{
    static_assert(V % 2 == 0, "pairs");
#pragma unroll
    for (int v = 0; v < V; v += 2) {
        float2 s2, c2;
        sincos_fast(make_float2(x[v], x[v + 1]), s2, c2);
        s[v] = s2.x; s[v + 1] = s2.y; c[v] = c2.x; c[v + 1] = c2.y;
    }
}
template <int V>
__device__ __forceinline__ void sin_vec(const float (&x)[V], float (&y)[V])
{
#pragma unroll
    for (int v = 0; v < V; v += 2) {
        const float2 r = sin_fast(make_float2(x[v], x[v + 1]));
        y[v] = r.x; y[v + 1] = r.y;
    }
}
template <int V>
__device__ __forceinline__ void sincos_vec(const double (&x)[V], double (&s)[V], double (&c)[V])
{
#pragma unroll
    for (int v = 0; v < V; ++v) sincos_fast(x[v], s[v], c[v]);
}
template <int V>
__device__ __forceinline__ void sin_vec(const double (&x)[V], double (&y)[V])
{
#pragma unroll
    for (int v = 0; v < V; ++v) y[v] = sin_fast(x[v]);
}

// ---- pairs of sites (ahs_pack.cuh): fp32 through the packed form, fp64 element by element ------------------------------
__device__ __forceinline__ void sincos_pair(float2 x, float2& s, float2& c) { sincos_fast(x, s, c); }
__device__ __forceinline__ float2 sin_pair(float2 x) { return sin_fast(x); }
__device__ __forceinline__ void sincos_pair(double2 x, double2& s, double2& c)
{
    sincos_fast(x.x, s.x, c.x);
    sincos_fast(x.y, s.y, c.y);
}
__device__ __forceinline__ double2 sin_pair(double2 x) { return make_double2(sin_fast(x.x), sin_fast(x.y)); }
__device__ __forceinline__ float2 chord_pair(float2 x) { return chord_fast(x); }
__device__ __forceinline__ double2 chord_pair(double2 x) { return make_double2(2.0 * sin_fast(0.5 * x.x), 2.0 * sin_fast(0.5 * x.y)); }

}  // namespace ahs
