// ahs_pack.cuh -- arithmetic on PAIRS of lattice sites.
//
// sm_100 has packed fp32 instructions (FFMA2 / FMUL2 / FADD2: two IEEE fp32 operations per issued instruction, with
// negate / |.| / swap modifiers and scalar or immediate broadcast on the operands).  The diagnostics march is bound by
// instruction issue, not by HBM (profiles/HISTORY.md r2), so its arithmetic is written once over a pair type
// P = Pair<T>: for T = float the packed instructions on two neighbouring sites (x, x+1) of a thread's 16-byte vector,
// for T = double the same expressions element by element.  Every operation rounds exactly like its scalar
// counterpart, so results do not depend on how the sites are paired.
#pragma once
#include <cuda_runtime.h>

namespace ahs {
namespace pk {

template <typename T> struct PairOf;
template <> struct PairOf<float> { using type = float2; };
template <> struct PairOf<double> { using type = double2; };
template <typename T> using Pair = typename PairOf<T>::type;

// ---- fp32: packed ----------------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 mk(float x, float y) { return make_float2(x, y); }
__device__ __forceinline__ float2 splat(float v) { return make_float2(v, v); }
__device__ __forceinline__ float2 neg(float2 a) { return make_float2(-a.x, -a.y); }        // folds into an operand modifier
__device__ __forceinline__ float2 absv(float2 a) { return make_float2(fabsf(a.x), fabsf(a.y)); }   // likewise
__device__ __forceinline__ float2 add(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 sub(float2 a, float2 b) { return __fadd2_rn(a, neg(b)); }
__device__ __forceinline__ float2 mul(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }

// ---- fp64: the same names, element by element ---------------------------------------------------------------------------
__device__ __forceinline__ double2 mk(double x, double y) { return make_double2(x, y); }
__device__ __forceinline__ double2 splat(double v) { return make_double2(v, v); }
__device__ __forceinline__ double2 neg(double2 a) { return make_double2(-a.x, -a.y); }
__device__ __forceinline__ double2 absv(double2 a) { return make_double2(fabs(a.x), fabs(a.y)); }
__device__ __forceinline__ double2 add(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 sub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 mul(double2 a, double2 b) { return make_double2(a.x * b.x, a.y * b.y); }
__device__ __forceinline__ double2 fma(double2 a, double2 b, double2 c) { return make_double2(::fma(a.x, b.x, c.x), ::fma(a.y, b.y, c.y)); }

// pair h of a 16-byte vector's elements (2h, 2h+1), and the same shifted by one site: (2h+1, 2h+2) with element V = `edge`
template <typename T, int V>
__device__ __forceinline__ Pair<T> at(const T (&a)[V], int h) { return mk(a[2 * h], a[2 * h + 1]); }
template <typename T, int V>
__device__ __forceinline__ Pair<T> next(const T (&a)[V], int h, T edge) { return mk(a[2 * h + 1], 2 * h + 2 < V ? a[2 * h + 2 < V ? 2 * h + 2 : 0] : edge); }

}  // namespace pk
}  // namespace ahs
