// ahs_ic.cu -- initial condition from a counter-based generator, and the
// precision-conversion helpers of ahs_get_fields / ahs_set_fields.
//
// "the scalar field phi is set to have a random phase, its norm is set to unity (given that sigma = 1) and
//  all other field variables are set to zero" (L72).  The paper draws the phase with cuRAND (L74); here it is
// Philox4x32-10 keyed by (seed) with counter = site index, so that the field does not depend on the launch
// shape and the CPU oracle can reproduce it from the specification alone (R9).
#include "ahs_internal.cuh"

namespace ahs {

namespace {

__device__ __forceinline__ void philox_round(uint32_t (&c)[4], uint32_t k0, uint32_t k1)
{
    const uint32_t hi0 = __umulhi(0xD2511F53u, c[0]), lo0 = 0xD2511F53u * c[0];
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c[2]), lo1 = 0xCD9E8D57u * c[2];
    const uint32_t a = hi1 ^ c[1] ^ k0, b = lo1, d = hi0 ^ c[3] ^ k1, e = lo0;
    c[0] = a; c[1] = b; c[2] = d; c[3] = e;
}

__device__ __forceinline__ void philox4x32_10(uint64_t counter, uint64_t seed, uint32_t (&r)[4])
{
    r[0] = (uint32_t)counter; r[1] = (uint32_t)(counter >> 32); r[2] = 0u; r[3] = 0u;
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        philox_round(r, k0, k1);
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
}

__device__ __forceinline__ double unit53(uint32_t hi, uint32_t lo)
{
    const uint64_t w = ((uint64_t)hi << 32) | (uint64_t)lo;
    return (double)(w >> 11) * 0x1.0p-53;
}

template <typename T>
__global__ void __launch_bounds__(256) ic_kernel(T* __restrict__ phi_re, T* __restrict__ phi_im, int64_t nsites,
                                                 int64_t plane_sites, int64_t lattice_sites, int64_t first_site,
                                                 double sigma, uint64_t seed, int kind)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t site = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; site < nsites; site += stride) {
        // site index of the full lattice (the Philox counter, R9): local planes map to global planes periodically
        int64_t gsite = first_site + site;
        while (gsite >= lattice_sites) gsite -= lattice_sites;
        uint32_t r[4];
        philox4x32_10((uint64_t)gsite, seed, r);
        double amp, ang;
        if (kind == AHS_IC_RANDOM_PHASE) {
            amp = sigma;
            ang = 6.283185307179586476925286766559 * unit53(r[0], r[1]);
        } else {  // Box-Muller: re, im ~ N(0, sigma^2/2)
            const double u1 = unit53(r[0], r[1]) + 0x1.0p-54;
            amp = (sigma / sqrt(2.0)) * sqrt(-2.0 * log(u1));
            ang = 6.283185307179586476925286766559 * unit53(r[2], r[3]);
        }
        double sn, cs;
        sincos(ang, &sn, &cs);
        phi_re[site] = (T)(amp * cs);
        phi_im[site] = (T)(amp * sn);
    }
}

template <typename S, typename D>
__global__ void __launch_bounds__(256) convert_kernel(const S* __restrict__ src, D* __restrict__ dst, int64_t n)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) dst[i] = (D)src[i];
}

inline int grid_for(int64_t n)
{
    int64_t b = (n + 255) / 256;
    const int64_t cap = 148 * 16;   // grid-stride; a multiple of the SM count
    return (int)(b < cap ? b : cap);
}

}  // namespace

template <typename T>
int launch_ic(T* phi_re, T* phi_im, int N, int nz_alloc, int z_first, double sigma, uint64_t seed, int kind, cudaStream_t st)
{
    const int64_t plane = (int64_t)N * N, nsites = plane * nz_alloc, lattice = plane * N;
    const int64_t first = plane * (((int64_t)z_first % N + N) % N);
    if (nz_alloc > N + 2) return AHS_ERR_INVALID_ARG;
    ic_kernel<T><<<grid_for(nsites), 256, 0, st>>>(phi_re, phi_im, nsites, plane, lattice, first, sigma, seed, kind);
    return cudaGetLastError() == cudaSuccess ? 1 : AHS_ERR_CUDA;
}

template <typename T>
int launch_convert_from_double(const double* src, T* dst, int64_t n, cudaStream_t st)
{
    convert_kernel<double, T><<<grid_for(n), 256, 0, st>>>(src, dst, n);
    return cudaGetLastError() == cudaSuccess ? 1 : AHS_ERR_CUDA;
}

template <typename T>
int launch_convert_to_double(const T* src, double* dst, int64_t n, cudaStream_t st)
{
    convert_kernel<T, double><<<grid_for(n), 256, 0, st>>>(src, dst, n);
    return cudaGetLastError() == cudaSuccess ? 1 : AHS_ERR_CUDA;
}

template int launch_ic<float>(float*, float*, int, int, int, double, uint64_t, int, cudaStream_t);
template int launch_ic<double>(double*, double*, int, int, int, double, uint64_t, int, cudaStream_t);
template int launch_convert_from_double<float>(const double*, float*, int64_t, cudaStream_t);
template int launch_convert_from_double<double>(const double*, double*, int64_t, cudaStream_t);
template int launch_convert_to_double<float>(const float*, double*, int64_t, cudaStream_t);
template int launch_convert_to_double<double>(const double*, double*, int64_t, cudaStream_t);

}  // namespace ahs
