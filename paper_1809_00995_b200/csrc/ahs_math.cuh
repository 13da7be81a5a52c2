// ahs_math.cuh -- precision-generic device math used by the step and diagnostics kernels.
// Accurate libdevice routines only: no --use_fast_math, no __sinf/__cosf intrinsics (PAPER.md L142 reports
// that reduced-precision intrinsics degrade the diagnostics).
#pragma once
#include <cuda_runtime.h>

namespace ahs {

__device__ __forceinline__ void sincos_t(float x, float& s, float& c) { sincosf(x, &s, &c); }
__device__ __forceinline__ void sincos_t(double x, double& s, double& c) { sincos(x, &s, &c); }
__device__ __forceinline__ float sin_t(float x) { return sinf(x); }
__device__ __forceinline__ double sin_t(double x) { return sin(x); }
__device__ __forceinline__ float cos_t(float x) { return cosf(x); }
__device__ __forceinline__ double cos_t(double x) { return cos(x); }
__device__ __forceinline__ bool finite_t(float x) { return isfinite(x); }
__device__ __forceinline__ bool finite_t(double x) { return isfinite(x); }

// complex helpers on (re, im) pairs; U = cos(theta) - i sin(theta)  (q = +1, R1)
template <typename T> struct Cx { T re, im; };

// The contraction into fused multiply-adds is written out (one rounded product, one fma) so that a hop is rounded the same
// way wherever the compiler inlines it: the step march forms conj(U_2) phi both in a chunk's prologue and in its loop, and
// the fields must not depend on where the chunk boundaries fall.
// U * z = (c - i s)(re + i im) = (c re + s im) + i (c im - s re)
template <typename T> __device__ __forceinline__ Cx<T> mulU(T c, T s, Cx<T> z) { return { fma(c, z.re, s * z.im), fma(c, z.im, -(s * z.re)) }; }
// conj(U) * z = (c + i s)(re + i im) = (c re - s im) + i (c im + s re)
template <typename T> __device__ __forceinline__ Cx<T> mulUc(T c, T s, Cx<T> z) { return { fma(c, z.re, -(s * z.im)), fma(c, z.im, s * z.re) }; }

}  // namespace ahs
