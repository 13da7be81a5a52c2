// ahs_diag_generic.cu -- network diagnostics for ANY lattice size, one thread per site, plus the
// fixed-order finishing reduction shared with the z-marching diagnostics kernel.
//
//   winding   Eq. 11:  n_i^x = rint((arg phi^{x+k_i} - arg phi^x - theta_i^x) / 2 pi),
//             W_ij^x = -(n_i^x + n_j^{x+k_i} - n_i^{x+k_j} - n_j^x), integer arithmetic; the rint decision is taken
//             in fp64 whatever the storage type, so that the count is bit-exact against an fp64 evaluation
//             of the same snapshot.
//   <v^2>_L   Eqs. 9-10 with the weight of Eq. 2 (L40, L78-86): sums of K*Lag and G*Lag, fp64 accumulation.
//   Gauss     g^x = sum_i (eps_i^x - eps_i^{x-k_i}) - 2 dx^2 e0^2 a_h^(2s) Im[conj(phi) Pi]   (L72, L181; R4).
#include "ahs_internal.cuh"
#include "ahs_math.cuh"
#include "ahs_reduce.cuh"

namespace ahs {

namespace {

constexpr double kInv2Pi = 0.15915494309189535;

}  // namespace

namespace {

// second stage: ONE block sums the partials in a fixed order (thread t takes t, t+256, ...; then the block tree)
__global__ void __launch_bounds__(256) diag_finish_kernel(const DiagPartial* __restrict__ partials, int n, DiagPartial* __restrict__ result)
{
    DiagPartial t = {0ull, 0ull, 0.0, 0.0, 0.0, 0.0, 0.0, 0ull, 0.0, 0.0, 0.0, 0.0};
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const DiagPartial p = partials[i];
        t.n_pierced += p.n_pierced; t.sum_abs_w += p.sum_abs_w;
        t.num += p.num; t.den += p.den; t.lsum += p.lsum;
        t.gmax = fmax(t.gmax, p.gmax); t.rhs2 += p.rhs2; t.nonfinite += p.nonfinite;
        t.vnum += p.vnum; t.vden += p.vden; t.wnum += p.wnum; t.wden += p.wden;
    }
    block_reduce_store(t, result);
}

template <typename T>
__global__ void __launch_bounds__(128) diag_generic_kernel(DiagPtrs<T> f, int N, DiagCoef k, DiagPartial* __restrict__ partials)
{
    const int64_t nsites = (int64_t)N * N * N;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t sN = N, sNN = (int64_t)N * N;
    DiagPartial acc = {0ull, 0ull, 0.0, 0.0, 0.0, 0.0, 0.0, 0ull, 0.0, 0.0, 0.0, 0.0};

    for (int64_t site = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; site < nsites; site += stride) {
        const int x = (int)(site % N), y = (int)((site / N) % N), z = (int)(site / sNN);
        const int64_t wrap[3] = { 1 - sN, sN - sNN, sNN - nsites };
        const int64_t str[3] = { 1, sN, sNN };
        const int co[3] = { x, y, z };
        int64_t sp[3], sm[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            sp[i] = site + (co[i] == N - 1 ? wrap[i] : str[i]);
            sm[i] = site - (co[i] == 0 ? wrap[i] : str[i]);
        }
        const Cx<T> phi0 = { f.phi_re[site], f.phi_im[site] };
        const Cx<T> pi0 = { f.pi_re[site], f.pi_im[site] };
        const T th0[3] = { f.th[0][site], f.th[1][site], f.th[2][site] };
        const T ep0[3] = { f.eps[0][site], f.eps[1][site], f.eps[2][site] };

        bool ok = finite_t(phi0.re) && finite_t(phi0.im) && finite_t(pi0.re) && finite_t(pi0.im);
#pragma unroll
        for (int i = 0; i < 3; ++i) ok = ok && finite_t(th0[i]) && finite_t(ep0[i]);
        if (!ok) acc.nonfinite += 1ull;

        // ---- winding (fp64 decision) ---------------------------------------------------------------------------------
        // link number n_i at site s with forward neighbour t:  rint((arg_t - arg_s - theta_i^s) / 2 pi)
        auto arg = [&](int64_t s) { return atan2((double)f.phi_im[s], (double)f.phi_re[s]); };
        auto nlink = [&](double arg_s, double arg_t, T th) { return (int)rint((arg_t - arg_s - (double)th) * kInv2Pi); };
        const double a0 = arg(site);
        double ap[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) ap[i] = arg(sp[i]);
        int n0[3];
#pragma unroll
        for (int i = 0; i < 3; ++i) n0[i] = nlink(a0, ap[i], th0[i]);
        // plaquettes (i,j) = (0,1), (0,2), (1,2) based at this site
#pragma unroll
        for (int pl = 0; pl < 3; ++pl) {
            const int i = (pl == 2 ? 1 : 0), j = (pl == 0 ? 1 : 2);
            // corner x + k_i + k_j
            const int64_t spij = sp[i] + (co[j] == N - 1 ? wrap[j] : str[j]);
            const double aij = arg(spij);
            const int nj_pi = nlink(ap[i], aij, f.th[j][sp[i]]);   // n_j at x + k_i
            const int ni_pj = nlink(ap[j], aij, f.th[i][sp[j]]);   // n_i at x + k_j
            const int W = -(n0[i] + nj_pi - ni_pj - n0[j]);
            if (W != 0) acc.n_pierced += 1ull;
            acc.sum_abs_w += (unsigned long long)(W < 0 ? -W : W);
        }

        // ---- Eq. 2 pieces ---------------------------------------------------------------------------------------------
        T G = T(0);
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            T s, c;
            sincos_t(th0[i], s, c);
            const Cx<T> fwd = mulU<T>(c, s, { f.phi_re[sp[i]], f.phi_im[sp[i]] });
            const T dr = fwd.re - phi0.re, di = fwd.im - phi0.im;
            G += dr * dr + di * di;
        }
        G *= (T)k.inv_dx2;
        const T K = pi0.re * pi0.re + pi0.im * pi0.im;
        const T dm = phi0.re * phi0.re + phi0.im * phi0.im - (T)k.sigma2;
        const T Vp = (T)k.pot_coef * dm * dm;
        T mag = T(0);
#pragma unroll
        for (int pl = 0; pl < 3; ++pl) {
            const int i = (pl == 2 ? 1 : 0), j = (pl == 0 ? 1 : 2);
            const T xi = th0[i] + f.th[j][sp[i]] - f.th[i][sp[j]] - th0[j];
            mag += T(1) - cos_t(xi);
        }
        mag *= T(2);   // ordered pairs (i,j) and (j,i): cos is even (R12)
        const T e2 = ep0[0] * ep0[0] + ep0[1] * ep0[1] + ep0[2] * ep0[2];
        const T El = (T)k.gauge_norm * e2, Bm = (T)k.gauge_norm * (T)k.inv_dx2 * mag;   // electric / magnetic energy densities
        const T lag = ((T)k.cE * El - (T)k.cB * Bm) + K - G - Vp;
        acc.num += (double)K * (double)lag;
        acc.den += (double)G * (double)lag;
        acc.lsum += (double)lag;
        acc.vnum += (double)K * (double)Vp;   // potential-weighted estimator <v^2>_V (L86)
        acc.vden += (double)G * (double)Vp;
        // Eq. 12: rho = K + G + Vp + El + Bm, p = K - G/3 - Vp + (El + Bm)/3, weighted with the Lagrangian
        acc.wnum += (double)(K - G * (T)(1.0 / 3.0) - Vp + (El + Bm) * (T)(1.0 / 3.0)) * (double)lag;
        acc.wden += (double)(K + G + Vp + El + Bm) * (double)lag;

        // ---- Gauss residual ------------------------------------------------------------------------------------------
        T div = T(0);
#pragma unroll
        for (int i = 0; i < 3; ++i) div += ep0[i] - f.eps[i][sm[i]];
        const T rhs = (T)k.gauss_rhs * (phi0.re * pi0.im - phi0.im * pi0.re);
        const double g = fabs((double)(div - rhs));
        acc.gmax = fmax(acc.gmax, g);
        acc.rhs2 += (double)rhs * (double)rhs;
    }
    block_reduce_store(acc, partials + blockIdx.x);
}

}  // namespace

int launch_diag_finish(const DiagPartial* partials, int n, DiagPartial* result, cudaStream_t st)
{
    diag_finish_kernel<<<1, 256, 0, st>>>(partials, n, result);
    return cudaGetLastError() == cudaSuccess ? 1 : AHS_ERR_CUDA;
}

template <typename T>
int launch_diag_generic(const DiagPtrs<T>& f, int N, const DiagCoef& c, DiagPartial* partials, int max_partials,
                        DiagPartial* result, cudaStream_t st)
{
    const int64_t nsites = (int64_t)N * N * N;
    int64_t blocks = (nsites + 127) / 128;
    const int64_t cap = 148 * 32;
    if (blocks > cap) blocks = cap;
    if (blocks > max_partials) blocks = max_partials;
    diag_generic_kernel<T><<<(unsigned)blocks, 128, 0, st>>>(f, N, c, partials);
    if (cudaGetLastError() != cudaSuccess) return AHS_ERR_CUDA;
    const int r = launch_diag_finish(partials, (int)blocks, result, st);
    return r < 0 ? r : 2;
}

template int launch_diag_generic<float>(const DiagPtrs<float>&, int, const DiagCoef&, DiagPartial*, int, DiagPartial*, cudaStream_t);
template int launch_diag_generic<double>(const DiagPtrs<double>&, int, const DiagCoef&, DiagPartial*, int, DiagPartial*, cudaStream_t);

}  // namespace ahs
