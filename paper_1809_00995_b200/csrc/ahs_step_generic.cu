// ahs_step_generic.cu -- the fused leapfrog step (Eqs. 4-7) for ANY lattice size:
// one thread per site, periodic neighbours by index arithmetic, every link phase and plaquette sine
// recomputed where it is used.  It serves small lattices (N < 128) where the z-marching kernel does not
// apply, and is the on-device cross-check of that kernel (tests/test_gpu_parity.py).  All loads of the
// level-n fields hit L1/L2 at these sizes; performance work lives in ahs_step_march.cu.
#include "ahs_internal.cuh"
#include "ahs_math.cuh"

namespace ahs {

namespace {

template <typename T>
__global__ void __launch_bounds__(128) step_generic_kernel(FieldPtrs<T> f, int N, StepCoef k)
{
    const int64_t nsites = (int64_t)N * N * N;
    const int64_t site = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (site >= nsites) return;
    const int x = (int)(site % N), y = (int)((site / N) % N), z = (int)(site / ((int64_t)N * N));
    const int64_t sN = N, sNN = (int64_t)N * N;
    // neighbour offsets with periodic wrap: sp[j] = site + k_j, sm[j] = site - k_j
    const int64_t sp[3] = { site + (x == N - 1 ? 1 - sN : 1), site + (y == N - 1 ? sN - sNN : sN), site + (z == N - 1 ? sNN - nsites : sNN) };
    const int64_t sm[3] = { site - (x == 0 ? 1 - sN : 1), site - (y == 0 ? sN - sNN : sN), site - (z == 0 ? sNN - nsites : sNN) };

    const Cx<T> phi0 = { f.phi_re[site], f.phi_im[site] };
    const T th0[3] = { f.th[0][site], f.th[1][site], f.th[2][site] };

    // ---- Eq. 4: covariant Laplacian  sum_j [U_j^x phi^{x+k_j} - 2 phi^x + conj(U_j^{x-k_j}) phi^{x-k_j}] ------------
    T lap_re = T(0), lap_im = T(0);
    T cur[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        T s, c;
        sincos_t(th0[j], s, c);
        const Cx<T> fwd = mulU<T>(c, s, { f.phi_re[sp[j]], f.phi_im[sp[j]] });
        T sb, cb;
        sincos_t(f.th[j][sm[j]], sb, cb);
        const Cx<T> bwd = mulUc<T>(cb, sb, { f.phi_re[sm[j]], f.phi_im[sm[j]] });
        lap_re += (fwd.re - T(2) * phi0.re) + bwd.re;
        lap_im += (fwd.im - T(2) * phi0.im) + bwd.im;
        cur[j] = phi0.re * fwd.im - phi0.im * fwd.re;   // Im[conj(phi^x) U_j^x phi^{x+k_j}]  (Eq. 5, 2nd term)
    }
    const T mod2 = phi0.re * phi0.re + phi0.im * phi0.im;
    const T higgs = (T)k.c3 * (mod2 - (T)k.sigma2);
    const T pr = (T)k.c1 * f.pi_re[site] - higgs * phi0.re + (T)k.c2 * lap_re;
    const T pi = (T)k.c1 * f.pi_im[site] - higgs * phi0.im + (T)k.c2 * lap_im;

    // ---- Eq. 5: plaquette curl  sum_{j != i} [sin Xi_ij^x - sin Xi_ij^{x-k_j}],  Xi_ij^x per Eq. 3 --------------------
    T e_new[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        T curl = T(0);
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            if (j == i) continue;
            // Xi_ij^x = th_i^x + th_j^{x+k_i} - th_i^{x+k_j} - th_j^x
            const T xi0 = th0[i] + f.th[j][sp[i]] - f.th[i][sp[j]] - th0[j];
            // the same plaquette based at b = x - k_j:  th_i^b + th_j^{b+k_i} - th_i^{b+k_j} - th_j^b ,  b + k_j = x
            const int64_t b = sm[j];
            // b + k_i : shift sm[j] along i with wrap (i != j so the two wraps are independent)
            const int ci = (i == 0 ? x : (i == 1 ? y : z));
            const int64_t stride_i = (i == 0 ? 1 : (i == 1 ? sN : sNN));
            const int64_t bpi = b + (ci == N - 1 ? stride_i - stride_i * sN : stride_i);
            const T xim = f.th[i][b] + f.th[j][bpi] - th0[i] - f.th[j][b];
            curl += sin_t(xi0) - sin_t(xim);
        }
        e_new[i] = (T)k.d1 * f.eps[i][site] + (T)k.d2 * cur[i] - (T)k.d3 * curl;
    }

    // ---- in-place kicks, drift to the other buffer (Eqs. 6-7) ------------------------------------------------------------
    f.pi_re[site] = pr;
    f.pi_im[site] = pi;
    f.phi_re_out[site] = phi0.re + (T)k.dt * pr;
    f.phi_im_out[site] = phi0.im + (T)k.dt * pi;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        f.eps[i][site] = e_new[i];
        f.th_out[i][site] = th0[i] + (T)k.dt * e_new[i];
    }
}

}  // namespace

template <typename T>
int launch_step_generic(const FieldPtrs<T>& f, int N, const StepCoef& c, cudaStream_t st)
{
    const int64_t nsites = (int64_t)N * N * N;
    const int64_t blocks = (nsites + 127) / 128;
    if (blocks > 0x7fffffffLL) return AHS_ERR_INVALID_ARG;
    step_generic_kernel<T><<<(unsigned)blocks, 128, 0, st>>>(f, N, c);
    return cudaGetLastError() == cudaSuccess ? 1 : AHS_ERR_CUDA;
}

template int launch_step_generic<float>(const FieldPtrs<float>&, int, const StepCoef&, cudaStream_t);
template int launch_step_generic<double>(const FieldPtrs<double>&, int, const StepCoef&, cudaStream_t);

}  // namespace ahs
