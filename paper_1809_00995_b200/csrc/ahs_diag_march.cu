// ahs_diag_march.cu -- the fused network diagnostics (winding Eq. 11, <v^2>_L Eqs. 9-10 with the weight of Eq. 2,
// Gauss residual) as a 2.5D z-march for sm_100a: one read of the ten arrays per call.
//
// Same tile and staging as the step kernel (ahs_step_march.cu): a CTA owns TX x TY sites in (x, y) and marches over
// `zlen` planes; phi_re, phi_im, theta_0..2 of plane k+3 are streamed by cp.async.bulk into a 4-stage ring of halo'd
// shared-memory tiles while planes k, k+1 are in use; Pi and eps are read with streaming 16-byte loads.
// All the estimators need only FORWARD neighbours (x+k_i, x+k_i+k_j) of phi, theta -- except the divergence of eps,
// whose -x / -y / -z terms come by shuffle, one extra row load and a carried register.
//
// Winding, compute-once form.  arg phi is evaluated ONCE per site (phase A: plane k+1 -> a shared "arg tile", plus the
// forward halo row/column shared out over the threads), one CTA barrier, then (phase B) every link number
//     n_i^x = rint((arg^{x+k_i} - arg^x - theta_i^x) / 2 pi)
// a plaquette needs is formed from the arg tiles of planes k and k+1 and W_ij = -(n_i^x + n_j^{x+k_i} - n_i^{x+k_j} - n_j^x)
// is summed exactly.  The decision is the fp64 one: the arg tile holds atan2f values (error
// <= 2 ulp(pi) = 5e-7 rad), the quotient is formed in fp32 from them, and any link whose quotient lies within
// 1e-5 (1 + |t|) of a half-integer -- thirty times the worst-case error -- is redone with fp64 atan2 of both ends, so every
// rint is the one an all-fp64 evaluation takes (probability of the slow path: 4e-5 per link at |theta| <~ 1).
// <v^2>_L sums: products and the sum over the 16-byte vector of a thread in the storage type, then fp64 accumulation.
// The paper runs Winding and VelRWLag as two kernels over raw fields with a CUB block sum and a host-side final sum
// (L140); this is a different design.
#include <cstdlib>

#include "ahs_internal.cuh"
#include "ahs_math.cuh"
#include "ahs_reduce.cuh"
#include "ahs_stage.cuh"
#include "ahs_trig.cuh"

namespace ahs {

namespace {

constexpr double kInv2Pi = 0.15915494309189535;
constexpr float kTieMargin = 4e-6f;   // in units of a full turn, relative to 1 + |t|: ten times the error bound

template <typename T, int TY_>
struct DiagCfg {
    static constexpr int V = 16 / sizeof(T);
    static constexpr int TY = TY_;
    static constexpr int NSTAGE = 4;
    using G = TileGeom<T, V, TY, 5, NSTAGE>;                 // a stage: phi_re, phi_im, theta_0, theta_1, theta_2 of one plane
    static constexpr int TX = G::TX;
    static constexpr int NTHREADS = TY * 32;
    static constexpr int APITCH = TX + 4;                    // arg tile: rows 0 .. TY, columns 0 .. TX (floats)
    static constexpr int ATILE = (TY + 1) * APITCH;
    static constexpr int NARG = 3;                           // planes k, k+1 in use while k+2's slot may still be read
    static constexpr int NJOBS = TX + 1 + TY;                // forward halo: row TY (TX+1 sites) and column TX (TY sites)
    static constexpr size_t SMEM = 128 + sizeof(T) * (size_t)(NSTAGE * G::STAGE_ELEMS) + sizeof(float) * (size_t)(NARG * ATILE);
};

template <int V> struct FVec;
template <> struct FVec<4> { using type = float4; };
template <> struct FVec<2> { using type = float2; };

// Link number of the link s -> t with angle th, fast path, all in fp32: t = (arg_t - arg_s - th) / 2 pi from the
// atan2_fast phases of the arg tile, n = rint(t) (ties to even) as a float.  |t - t_exact| <= 3.5e-7 + 2.5e-7 |t| turns
// (6e-7 rad per phase, three roundings, the fp32 constant), so whenever |t - n| < 1/2 - kTieMargin (1 + |t|), n IS the
// fp64 decision.  `slack` keeps the smallest margin seen; the caller redoes the whole thread-plane in fp64
// (winding_fp64, out of line) when it is not positive.  Everything here is branch-free.
__device__ __forceinline__ float link_number(float as, float at, float th, float& slack)
{
    const float t = ((at - as) - th) * 0.15915494309189535f;
    const float n = (t + 12582912.0f) - 12582912.0f;   // 1.5 * 2^23
    slack = fminf(slack, (0.5f - kTieMargin) - fmaf(kTieMargin, fabsf(t), fabsf(t - n)));
    return n;
}

// The winding of the V sites of one thread in one plane, every phase and every quotient in fp64, straight from the
// staged raw fields (same arithmetic as diag_generic_kernel).  Returns n_pierced | sum|W| << 16.  Out of line on purpose:
// it runs for ~4e-4 of the thread-planes, and thirty inlined copies of the fp64 atan2 made the loop overflow the
// instruction cache (profiles/r2).
template <typename T, typename G>
__device__ __noinline__ unsigned winding_fp64(const T* sc, const T* sn, int w, int xi)
{
    constexpr int V = G::V;
    double a[2][2][V + 1];
    for (int pl = 0; pl < 2; ++pl)
        for (int r = 0; r < 2; ++r)
            for (int c = 0; c <= V; ++c) {
                const T* st = pl ? sn : sc;
                a[pl][r][c] = atan2((double)st[G::idx(1, w + r, xi + c)], (double)st[G::idx(0, w + r, xi + c)]);
            }
    auto ln = [](double as, double at, T th) { return (int)rint((at - as - (double)th) * kInv2Pi); };
    unsigned pierced = 0u, absw = 0u;
    for (int v = 0; v < V; ++v) {
        const int n0 = ln(a[0][0][v], a[0][0][v + 1], sc[G::idx(2, w, xi + v)]);
        const int n1 = ln(a[0][0][v], a[0][1][v], sc[G::idx(3, w, xi + v)]);
        const int n2 = ln(a[0][0][v], a[1][0][v], sc[G::idx(4, w, xi + v)]);
        const int n1x = ln(a[0][0][v + 1], a[0][1][v + 1], sc[G::idx(3, w, xi + v + 1)]);
        const int n2x = ln(a[0][0][v + 1], a[1][0][v + 1], sc[G::idx(4, w, xi + v + 1)]);
        const int n0y = ln(a[0][1][v], a[0][1][v + 1], sc[G::idx(2, w + 1, xi + v)]);
        const int n2y = ln(a[0][1][v], a[1][1][v], sc[G::idx(4, w + 1, xi + v)]);
        const int n0z = ln(a[1][0][v], a[1][0][v + 1], sn[G::idx(2, w, xi + v)]);
        const int n1z = ln(a[1][0][v], a[1][1][v], sn[G::idx(3, w, xi + v)]);
        const int W01 = -(n0 + n1x - n0y - n1), W02 = -(n0 + n2x - n0z - n2), W12 = -(n1 + n2y - n1z - n2);
        pierced += (W01 != 0) + (W02 != 0) + (W12 != 0);
        absw += (unsigned)(abs(W01) + abs(W02) + abs(W12));
    }
    return pierced | (absw << 16);
}

template <typename T, int TY, int MINB>
__global__ void __launch_bounds__(DiagCfg<T, TY>::NTHREADS, MINB)
diag_march_kernel(DiagPtrs<T> f, int N, int zlen, DiagCoef kd, DiagPartial* __restrict__ partials)
{
    using C = DiagCfg<T, TY>;
    using G = typename C::G;
    using VecT = Vec<T, C::V>;
    using FV = typename FVec<C::V>::type;
    constexpr int V = C::V, TX = C::TX, NS = C::NSTAGE, SE = G::STAGE_ELEMS, ARR = G::ARR_ELEMS, AP = C::APITCH;

    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);
    T* stages = reinterpret_cast<T*>(smem + 128);
    float* argt = reinterpret_cast<float*>(stages + NS * SE);

    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int tiles_x = N / TX, tiles_y = N / TY;
    int bid = blockIdx.x;
    const int tx = bid % tiles_x;
    bid /= tiles_x;
    const int ty = bid % tiles_y, zc = bid / tiles_y;
    const int x0 = tx * TX, y0 = ty * TY, z0 = zc * zlen;
    const int xi = V * lane;

    const T* const src[5] = { f.phi_re, f.phi_im, f.th[0], f.th[1], f.th[2] };
    const T inv_dx2 = (T)kd.inv_dx2, gauge_norm = (T)kd.gauge_norm, cB = (T)kd.cB_inv_dx2, pot = (T)kd.pot_coef;
    const T sigma2 = (T)kd.sigma2, grhs = (T)kd.gauss_rhs;

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();

    // plane index p of this CTA's march = lattice plane z0 + p (periodic); planes 0 .. zlen are needed
    auto plane_of = [&](int p) { const int z = z0 + p; return z >= N ? z - N : z; };
    if (w == 0 && elect_one()) {
#pragma unroll
        for (int p = 0; p < NS - 1; ++p) {
            if (p <= zlen) {
                mbar_arrive_expect_tx(&full[p], G::STAGE_BYTES);
                issue_rows<G, 5>(stages + p * SE, &full[p], src, N, x0, y0, plane_of(p));
            }
        }
    }

    // phase A of a plane: arg phi of the tile (own sites, then the forward halo row and column) -> arg tile `dst`
    auto fill_args = [&](const T* st, float* dst, int rot) {
        const VecT pr = lds_vec<T, V>(st + G::idx(0, w, xi)), pi = lds_vec<T, V>(st + G::idx(1, w, xi));
        float a[V];
#pragma unroll
        for (int v = 0; v < V; ++v) a[v] = atan2_fast((float)pi.v[v], (float)pr.v[v]);
        FV av;
        memcpy(&av, a, sizeof(av));
        *reinterpret_cast<FV*>(dst + w * AP + xi) = av;
        const int t = (threadIdx.x + 32 * rot) % C::NTHREADS;   // the halo jobs rotate over the warps
        for (int j = t; j < C::NJOBS; j += C::NTHREADS) {
            const int r = j <= TX ? TY : j - (TX + 1), c = j <= TX ? j : TX;
            dst[r * AP + c] = atan2_fast((float)st[G::idx(1, r, c)], (float)st[G::idx(0, r, c)]);
        }
    };

    mbar_wait(&full[0], 0);
    fill_args(stages, argt, 0);
    __syncthreads();
    // n_0, n_1 of the current plane (own sites; n_1 also right of the vector), carried along the march, with their margin
    float n0c[V], n1c[V + 1], slack_c = 1.0f;
    {
        const VecT t0 = lds_vec<T, V>(stages + G::idx(2, w, xi)), t1 = lds_vec<T, V>(stages + G::idx(3, w, xi));
        const T t1x_e = stages[G::idx(3, w, xi + V)];
#pragma unroll
        for (int v = 0; v <= V; ++v) {
            const float as = argt[w * AP + xi + v], ay = argt[(w + 1) * AP + xi + v];
            n1c[v] = link_number(as, ay, (float)(v < V ? t1.v[v < V ? v : 0] : t1x_e), slack_c);
            if (v < V) n0c[v < V ? v : 0] = link_number(as, argt[w * AP + xi + v + 1], (float)t0.v[v < V ? v : 0], slack_c);
        }
    }

    // eps_2 of the plane below, carried in registers along the march
    VecT E2m;
    {
        const int zm = z0 == 0 ? N - 1 : z0 - 1;
        E2m = ldg_vec<T, V>(f.eps[2] + ((size_t)zm * N + (size_t)(y0 + w)) * N + (size_t)(x0 + xi));
    }

    double num = 0.0, den = 0.0, lsum = 0.0, rhs2 = 0.0, gmax = 0.0;
    unsigned n_pierced = 0u, nonfinite = 0u;
    unsigned sum_abs_w = 0u;
    T gmax_t = T(0);

    for (int it = 0; it < zlen; ++it) {
        const T* sc = stages + (it % NS) * SE;
        const T* sn = stages + ((it + 1) % NS) * SE;
        const float* ac = argt + (it % C::NARG) * C::ATILE;
        float* an = argt + ((it + 1) % C::NARG) * C::ATILE;

        const int z = z0 + it, y = y0 + w;
        const size_t grow = ((size_t)z * N + (size_t)y) * N;
        const size_t g = grow + (size_t)(x0 + xi);
        const VecT Pr = ldg_vec<T, V>(f.pi_re + g), Pi = ldg_vec<T, V>(f.pi_im + g);
        const VecT E0 = ldg_vec<T, V>(f.eps[0] + g), E1 = ldg_vec<T, V>(f.eps[1] + g), E2 = ldg_vec<T, V>(f.eps[2] + g);
        const int ym = y == 0 ? N - 1 : y - 1;
        const VecT E1m = ldg_vec<T, V>(f.eps[1] + ((size_t)z * N + (size_t)ym) * N + (size_t)(x0 + xi));
        T e0_halo = T(0);
        if (lane == 0) e0_halo = f.eps[0][grow + (size_t)(x0 == 0 ? N - 1 : x0 - 1)];

        mbar_wait(&full[(it + 1) % NS], ((it + 1) / NS) & 1);
        fill_args(sn, an, it + 1);
        __syncthreads();

        // plane it+3 -> the stage that held plane it-1 (its last readers, phase B of iteration it-1, passed the barrier above)
        if (((w + it) % TY) == 0 && it + NS - 1 <= zlen && elect_one()) {
            const int s = (it + NS - 1) % NS;
            mbar_arrive_expect_tx(&full[s], G::STAGE_BYTES);
            issue_rows<G, 5>(stages + s * SE, &full[s], src, N, x0, y0, plane_of(it + NS - 1));
        }

        // ---- phase B: everything of plane `it` ---------------------------------------------------------------------------
        const VecT pr = lds_vec<T, V>(sc + G::idx(0, w, xi)), pi = lds_vec<T, V>(sc + G::idx(1, w, xi));
        const VecT t0 = lds_vec<T, V>(sc + G::idx(2, w, xi)), t1 = lds_vec<T, V>(sc + G::idx(3, w, xi)), t2 = lds_vec<T, V>(sc + G::idx(4, w, xi));
        const VecT pry = lds_vec<T, V>(sc + G::idx(0, w + 1, xi)), piy = lds_vec<T, V>(sc + G::idx(1, w + 1, xi));
        const VecT t0y = lds_vec<T, V>(sc + G::idx(2, w + 1, xi)), t2y = lds_vec<T, V>(sc + G::idx(4, w + 1, xi));
        const VecT prz = lds_vec<T, V>(sn + G::idx(0, w, xi)), piz = lds_vec<T, V>(sn + G::idx(1, w, xi));
        const VecT t0z = lds_vec<T, V>(sn + G::idx(2, w, xi)), t1z = lds_vec<T, V>(sn + G::idx(3, w, xi));
        const T prx_e = sc[G::idx(0, w, xi + V)], pix_e = sc[G::idx(1, w, xi + V)];
        const T t1x_e = sc[G::idx(3, w, xi + V)], t2x_e = sc[G::idx(4, w, xi + V)];
        // arg tiles: this plane (rows w, w+1) and the next (rows w, w+1), each with the element right of the vector
        float a[V + 1], ay[V + 1], az[V + 1], azy[V + 1];
        {
            const FV va = *reinterpret_cast<const FV*>(ac + w * AP + xi), vy = *reinterpret_cast<const FV*>(ac + (w + 1) * AP + xi);
            const FV vz = *reinterpret_cast<const FV*>(an + w * AP + xi), vzy = *reinterpret_cast<const FV*>(an + (w + 1) * AP + xi);
            memcpy(a, &va, sizeof(va)); memcpy(ay, &vy, sizeof(vy)); memcpy(az, &vz, sizeof(vz)); memcpy(azy, &vzy, sizeof(vzy));
            a[V] = ac[w * AP + xi + V]; ay[V] = ac[(w + 1) * AP + xi + V];
            az[V] = an[w * AP + xi + V]; azy[V] = an[(w + 1) * AP + xi + V];
        }
        // E0 of the site to the left: previous element, else lane-1's last element, else (lane 0) the halo value
        T e0_left = __shfl_up_sync(0xffffffffu, E0.v[V - 1], 1);
        if (lane == 0) e0_left = e0_halo;

        // ---- winding (Eq. 11), fast path: the link numbers this thread-plane needs.  n_0, n_1 of this plane were formed
        //      one iteration ago (as the +z links); n_1, n_2 are also taken at the site right of the vector (n_j^{x+k_0}).
        float slack = slack_c;                               // margins of the carried n0c, n1c
        float n2[V + 1], n0y[V], n2y[V], n0z[V], n1z[V + 1];
        slack_c = 1.0f;
        {
            const T t1z_e = sn[G::idx(3, w, xi + V)];
#pragma unroll
            for (int v = 0; v <= V; ++v) {
                n2[v] = link_number(a[v], az[v], (float)(v < V ? t2.v[v < V ? v : 0] : t2x_e), slack);
                n1z[v] = link_number(az[v], azy[v], (float)(v < V ? t1z.v[v < V ? v : 0] : t1z_e), slack_c);
            }
#pragma unroll
            for (int v = 0; v < V; ++v) {
                n0y[v] = link_number(ay[v], ay[v + 1], (float)t0y.v[v], slack);
                n2y[v] = link_number(ay[v], azy[v], (float)t2y.v[v], slack);
                n0z[v] = link_number(az[v], az[v + 1], (float)t0z.v[v], slack_c);
            }
        }
        unsigned pierced = 0u;
        float abs_w = 0.0f;                              // small integers: exact in fp32
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const float W01 = (n0c[v] + n1c[v + 1]) - (n0y[v] + n1c[v]);   // -W_ij
            const float W02 = (n0c[v] + n2[v + 1]) - (n0z[v] + n2[v]);
            const float W12 = (n1c[v] + n2y[v]) - (n1z[v] + n2[v]);
            pierced += (W01 != 0.0f) + (W02 != 0.0f) + (W12 != 0.0f);
            abs_w += (fabsf(W01) + fabsf(W02)) + fabsf(W12);
        }
        unsigned absw_u = (unsigned)abs_w;
        if (!(fminf(slack, slack_c) > 0.0f) || !(abs_w < 1.0e6f)) {   // a link too close to a tie (or NaN / huge): fp64 decides
            const unsigned r = winding_fp64<T, G>(sc, sn, w, xi);
            pierced = r & 0xffffu;
            absw_u = r >> 16;
        }
        n_pierced += pierced;
        sum_abs_w += absw_u;
#pragma unroll
        for (int v = 0; v < V; ++v) n0c[v] = n0z[v];
#pragma unroll
        for (int v = 0; v <= V; ++v) n1c[v] = n1z[v];

        T p_num = T(0), p_den = T(0), p_l = T(0), p_r2 = T(0);   // per thread and plane (V sites), then into the fp64 sums
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const Cx<T> ph = { pr.v[v], pi.v[v] };
            const Cx<T> pm = { Pr.v[v], Pi.v[v] };
            const T th0 = t0.v[v], th1 = t1.v[v], th2 = t2.v[v];
            const T ep0 = E0.v[v], ep1 = E1.v[v], ep2 = E2.v[v];
            // ---- Eq. 2 pieces ---------------------------------------------------------------------------------------------------
            T s, c;
            sincos_fast(th0, s, c);
            const Cx<T> f0 = mulU<T>(c, s, { next_x<T, V>(pr, v, prx_e), next_x<T, V>(pi, v, pix_e) });
            sincos_fast(th1, s, c);
            const Cx<T> f1 = mulU<T>(c, s, { pry.v[v], piy.v[v] });
            sincos_fast(th2, s, c);
            const Cx<T> f2 = mulU<T>(c, s, { prz.v[v], piz.v[v] });
            T Gd = (f0.re - ph.re) * (f0.re - ph.re) + (f0.im - ph.im) * (f0.im - ph.im);
            Gd += (f1.re - ph.re) * (f1.re - ph.re) + (f1.im - ph.im) * (f1.im - ph.im);
            Gd += (f2.re - ph.re) * (f2.re - ph.re) + (f2.im - ph.im) * (f2.im - ph.im);
            Gd *= inv_dx2;
            const T K = pm.re * pm.re + pm.im * pm.im;
            const T dm = ph.re * ph.re + ph.im * ph.im - sigma2;
            const T Vp = pot * dm * dm;
            // 1 - cos Xi = 2 sin^2(Xi/2), without the cancellation of the literal form at small Xi
            const T h01 = sin_fast(T(0.5) * (th0 + next_x<T, V>(t1, v, t1x_e) - t0y.v[v] - th1));
            const T h02 = sin_fast(T(0.5) * (th0 + next_x<T, V>(t2, v, t2x_e) - t0z.v[v] - th2));
            const T h12 = sin_fast(T(0.5) * (th1 + t2y.v[v] - t1z.v[v] - th2));
            const T mag = T(4) * (h01 * h01 + h02 * h02 + h12 * h12);   // ordered pairs: 2 x [2 sin^2] per plaquette (R12)
            const T e2 = ep0 * ep0 + ep1 * ep1 + ep2 * ep2;
            const T lag = (e2 - cB * mag) * gauge_norm + K - Gd - Vp;
            p_num += K * lag;
            p_den += Gd * lag;
            p_l += lag;
            nonfinite += finite_t(lag) ? 0u : 1u;   // every one of the ten values feeds lag: NaN or Inf in, NaN or Inf out

            // ---- Gauss residual ---------------------------------------------------------------------------------------------------
            const T e0m = v > 0 ? E0.v[v > 0 ? v - 1 : 0] : e0_left;
            const T div = ((ep0 - e0m) + (ep1 - E1m.v[v])) + (ep2 - E2m.v[v]);
            const T rhs = grhs * (ph.re * pm.im - ph.im * pm.re);
            const T gabs = fabs(div - rhs);
            gmax_t = gabs > gmax_t ? gabs : gmax_t;   // (a NaN residual is reported through `nonfinite`)
            p_r2 += rhs * rhs;
        }
        num += (double)p_num; den += (double)p_den; lsum += (double)p_l; rhs2 += (double)p_r2;
        E2m = E2;
    }

    gmax = (double)gmax_t;
    DiagPartial acc = { (unsigned long long)n_pierced, (unsigned long long)sum_abs_w, num, den, lsum, gmax, rhs2, (unsigned long long)nonfinite };
    block_reduce_store(acc, partials + blockIdx.x);
}

template <typename T, int TY>
int pick_zlen(int N, int ctas_per_sm, int max_partials)
{
    using C = DiagCfg<T, TY>;
    const long tiles = (long)(N / C::TX) * (N / TY);
    const int cands[5] = { 128, 64, 32, 16, 8 };
    for (int c : cands)   // the longest march that still gives >= 4 waves of resident CTAs (the prologue costs one plane)
        if (N % c == 0 && tiles * (N / c) <= max_partials && tiles * (N / c) >= 4L * ctas_per_sm * 148) return c;
    for (int c : cands)
        if (N % c == 0 && tiles * (N / c) <= max_partials) return c;
    return N;
}

template <typename T, int TY, int MINB>
int launch_cfg(const DiagPtrs<T>& f, int N, const DiagCoef& c, DiagPartial* partials, int max_partials, DiagPartial* result, cudaStream_t st)
{
    using C = DiagCfg<T, TY>;
    auto kern = diag_march_kernel<T, TY, MINB>;
    static bool configured = false;
    if (!configured) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM) != cudaSuccess) return AHS_ERR_CUDA;
        configured = true;
    }
    static const int zlen_env = [] { const char* e = getenv("AHS_DIAG_ZLEN"); return e ? atoi(e) : 0; }();
    const int zlen = (zlen_env > 0 && N % zlen_env == 0) ? zlen_env : pick_zlen<T, TY>(N, MINB, max_partials);
    const long blocks = (long)(N / C::TX) * (N / TY) * (N / zlen);
    if (blocks > max_partials) return AHS_ERR_INVALID_ARG;
    kern<<<(unsigned)blocks, C::NTHREADS, C::SMEM, st>>>(f, N, zlen, c, partials);
    if (cudaGetLastError() != cudaSuccess) return AHS_ERR_CUDA;
    const int r = launch_diag_finish(partials, (int)blocks, result, st);
    return r < 0 ? r : 2;
}

}  // namespace

template <typename T>
int launch_diag_march(const DiagPtrs<T>& f, int N, const DiagCoef& c, DiagPartial* partials, int max_partials, DiagPartial* result, cudaStream_t st)
{
    if (!march_supported<T>(N)) return AHS_ERR_INVALID_ARG;
    // 4-row tiles (3 CTAs/SM) by default; AHS_DIAG_TY=8 selects 8-row tiles, two CTAs per SM (experiments)
    static const int ty = [] { const char* e = getenv("AHS_DIAG_TY"); return e ? atoi(e) : 4; }();
    if (ty == 8) return launch_cfg<T, 8, 2>(f, N, c, partials, max_partials, result, st);
    return launch_cfg<T, 4, 3>(f, N, c, partials, max_partials, result, st);
}

template int launch_diag_march<float>(const DiagPtrs<float>&, int, const DiagCoef&, DiagPartial*, int, DiagPartial*, cudaStream_t);
template int launch_diag_march<double>(const DiagPtrs<double>&, int, const DiagCoef&, DiagPartial*, int, DiagPartial*, cudaStream_t);

}  // namespace ahs
