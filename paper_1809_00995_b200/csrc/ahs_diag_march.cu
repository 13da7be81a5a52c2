// ahs_diag_march.cu -- the fused network diagnostics (winding Eq. 11, <v^2>_L Eqs. 9-10 with the weight of Eq. 2,
// Gauss residual) as a 2.5D z-march for sm_100a: one read of the ten arrays per call.
//
// Same tile and staging as the step kernel (ahs_step_march.cu): a CTA owns TX x TY sites in (x, y) and marches over
// `zlen` planes; phi_re, phi_im, theta_0..2 of plane k+3 are streamed by cp.async.bulk into a 4-stage ring of halo'd
// shared-memory tiles (full / empty mbarrier pairs) while planes k, k+1 are in use; Pi and eps are read with streaming 16-byte loads.
// All the estimators need only FORWARD neighbours (x+k_i, x+k_i+k_j) of phi, theta -- except the divergence of eps,
// whose -x / -y / -z terms come by shuffle, one extra row load and a carried register.
//
// Winding.  Every thread evaluates arg phi (branch-free atan2_fast) at the ten points of plane k+1 its V sites need and
// carries them to the next plane in registers; there is NO exchange between warps and therefore no CTA barrier in the
// march: the warps of a CTA drift freely and meet only at the stage ring's full / empty mbarriers (an earlier version
// computed each phase once into a shared arg tile and lost 31 % of its issue slots at the per-plane barrier, profiles/r2).
// The link numbers n_i^x = rint((arg^{x+k_i} - arg^x - theta_i^x) / 2 pi) are formed in fp32 and
// W_ij = -(n_i^x + n_j^{x+k_i} - n_i^{x+k_j} - n_j^x) is summed exactly.  The decision is the fp64 one:
// a phase is off by <= 6e-7 rad, a quotient by <= 3.5e-7 + 2.5e-7 |t| turns, and whenever a link of a thread-plane lies
// within 4e-6 (1 + |t|) turns of a half-integer -- ten times that bound -- the thread redoes the plane's plaquettes with
// fp64 atan2 in a second pass over a device-side doubt list (diag_resolve_kernel; ~4e-4 of the thread-planes), so every
// rint is the one an all-fp64 evaluation takes and the march itself never diverges.
// <v^2>_L sums: products and the sum over the 16-byte vector of a thread in the storage type, then fp64 accumulation.
// The paper runs Winding and VelRWLag as two kernels over raw fields with a CUB block sum and a host-side final sum
// (L140); this is a different design.
#include <cstdlib>
#include <cstring>

#include "ahs_internal.cuh"
#include "ahs_math.cuh"
#include "ahs_reduce.cuh"
#include "ahs_stage.cuh"
#include "ahs_tma.cuh"
#include "ahs_trig.cuh"

namespace ahs {

namespace {

constexpr double kInv2Pi = 0.15915494309189535;
constexpr float kTieMargin = 4e-6f;   // in units of a full turn, relative to 1 + |t|: ten times the error bound

template <typename T, int TY_, int NS_ = 4>
struct DiagCfg {
    static constexpr int V = 16 / sizeof(T);
    static constexpr int TY = TY_;
    static constexpr int NSTAGE = NS_;
    using G = TileGeom<T, V, TY, 5, NSTAGE, 0, 0>;           // a stage: phi_re, phi_im, theta_0..2 of one plane, forward halo only
    static constexpr int TX = G::TX;
    static constexpr int NTHREADS = TY * 32;
    static constexpr int STAGE_STRIDE = (int)(((G::STAGE_BYTES + 127u) & ~127u) / sizeof(T));   // tensor copies land 128-byte aligned
    // right-edge tiles under TMA: the wrapped forward halo column (x = 0 .. V-1) of a plane lands in a side buffer
    static constexpr int WRAP_STRIDE = (int)(((5 * G::ROWS * V * sizeof(T) + 127) & ~(size_t)127) / sizeof(T));
    static constexpr size_t SMEM = 128 + sizeof(T) * (size_t)(NSTAGE * (STAGE_STRIDE + WRAP_STRIDE));
};

// Link number of the link s -> t with angle th, fast path, all in fp32: t = (arg_t - arg_s - th) / 2 pi from the
// atan2_fast phases of the arg tile, n = rint(t) (ties to even) as a float.  |t - t_exact| <= 3.5e-7 + 2.5e-7 |t| turns
// (6e-7 rad per phase, three roundings, the fp32 constant), so whenever |t - n| < 1/2 - kTieMargin (1 + |t|), n IS the
// fp64 decision.  `slack` keeps the smallest margin seen; when it is not positive the caller drops the thread-plane's
// fast count and appends the thread-plane to the doubt list (diag_resolve_kernel).  Everything here is branch-free.
__device__ __forceinline__ float link_number(float as, float at, float th, float& slack)
{
    const float t = ((at - as) - th) * 0.15915494309189535f;
    const float n = (t + 12582912.0f) - 12582912.0f;   // 1.5 * 2^23
    slack = fminf(slack, (0.5f - kTieMargin) - fmaf(kTieMargin, fabsf(t), fabsf(t - n)));
    return n;
}

// Second pass over the doubt list: the winding of the V sites of each listed (x/V, y, z), every phase and every quotient
// in fp64 straight from global memory (same arithmetic as diag_generic_kernel), added to one extra partial record.
// Integer sums: the order of the atomics does not matter.  ~4e-4 of the thread-planes end up here on smooth or random
// fields; resolving them in-line (an out-of-line call inside the march) made every warp of the CTA wait for the one
// that took the slow path (profiles/r2: 30 % of the issue slots), a separate pass costs ~0.1 ms at 1024^3.
template <typename T>
__global__ void __launch_bounds__(128) diag_resolve_kernel(DiagPtrs<T> f, int N, const unsigned* __restrict__ list,
                                                           const unsigned long long* __restrict__ count, DiagPartial* __restrict__ extra)
{
    constexpr int V = 16 / sizeof(T);
    const unsigned long long n = *count;
    unsigned pierced = 0u, absw = 0u;
    for (unsigned long long e = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned u = list[e];
        const int xv = (int)(u & 1023u), y = (int)((u >> 10) & 2047u), z = (int)(u >> 21);
        const int yp = y + 1 == N ? 0 : y + 1, zp = z + 1 == N ? 0 : z + 1;
        auto at = [&](int x, int yy, int zz) { return ((size_t)zz * N + (size_t)yy) * N + (size_t)x; };
        auto arg = [&](size_t i) { return atan2((double)f.phi_im[i], (double)f.phi_re[i]); };
        auto ln = [](double as, double a_t, T th) { return (int)rint((a_t - as - (double)th) * kInv2Pi); };
        for (int v = 0; v < V; ++v) {
            const int x = xv * V + v, xp = x + 1 == N ? 0 : x + 1;
            const size_t s0 = at(x, y, z), sx = at(xp, y, z), sy = at(x, yp, z), sz = at(x, y, zp);
            const double a0 = arg(s0), ax = arg(sx), ay = arg(sy), az = arg(sz);
            const double axy = arg(at(xp, yp, z)), axz = arg(at(xp, y, zp)), ayz = arg(at(x, yp, zp));
            const int n0 = ln(a0, ax, f.th[0][s0]), n1 = ln(a0, ay, f.th[1][s0]), n2 = ln(a0, az, f.th[2][s0]);
            const int n1x = ln(ax, axy, f.th[1][sx]), n2x = ln(ax, axz, f.th[2][sx]);
            const int n0y = ln(ay, axy, f.th[0][sy]), n2y = ln(ay, ayz, f.th[2][sy]);
            const int n0z = ln(az, axz, f.th[0][sz]), n1z = ln(az, ayz, f.th[1][sz]);
            const int W01 = -(n0 + n1x - n0y - n1), W02 = -(n0 + n2x - n0z - n2), W12 = -(n1 + n2y - n1z - n2);
            pierced += (W01 != 0) + (W02 != 0) + (W12 != 0);
            absw += (unsigned)(abs(W01) + abs(W02) + abs(W12));
        }
    }
    unsigned long long p64 = warp_sum((unsigned long long)pierced), w64 = warp_sum((unsigned long long)absw);
    if ((threadIdx.x & 31) == 0 && (p64 | w64)) {
        atomicAdd(&extra->n_pierced, p64);
        atomicAdd(&extra->sum_abs_w, w64);
    }
}

template <typename T, int TY, int MINB, int NSTAGES>
__global__ void __launch_bounds__(DiagCfg<T, TY, NSTAGES>::NTHREADS, MINB)
diag_march_kernel(DiagPtrs<T> f, int N, int zlen, DiagCoef kd, DiagPartial* __restrict__ partials, unsigned* __restrict__ doubt_list,
                  unsigned long long* __restrict__ doubt_count, const __grid_constant__ CUtensorMap tmap,
                  const __grid_constant__ CUtensorMap wmap, int use_tma, int rotate)
{
    using C = DiagCfg<T, TY, NSTAGES>;
    using G = typename C::G;
    using VecT = Vec<T, C::V>;
    constexpr int V = C::V, TX = C::TX, NS = C::NSTAGE, SE = C::STAGE_STRIDE;

    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);    // full[s]: the bulk copies of stage s have landed
    uint64_t* empty = full + NS;                           // empty[s]: all TY warps have finished reading stage s
    T* stages = reinterpret_cast<T*>(smem + 128);
    T* wraps = stages + NS * SE;                           // side buffers of the wrapped column (right-edge tiles under TMA)

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
        for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], TY); }
        mbar_fence_init();
    }
    __syncthreads();

    // plane index p of this CTA's march = lattice plane z0 + p (periodic); planes 0 .. zlen are needed
    auto plane_of = [&](int p) { const int z = z0 + p; return z >= N ? z - N : z; };
    // One tensor copy per plane for tiles away from the periodic boundary.  Tiles on the right edge get the main box
    // (zero-filled out of bounds) plus a V-wide tensor copy of the wrapped column x = 0 .. V-1 into a side buffer, which the
    // readers of column TX use instead; tiles on the top edge in y (2 of N/TY tile rows) keep the row copies.
    const bool right_edge = x0 + TX == N;
    const bool tma_tile = use_tma && (y0 + TY < N);
    const bool wrapR = tma_tile && right_edge;
    auto issue_plane = [&](int s, int p) {
        mbar_arrive_expect_tx(&full[s], G::STAGE_BYTES + (wrapR ? (uint32_t)(5 * G::ROWS * V * sizeof(T)) : 0u));
        if (tma_tile) {
            tma_load_4d(stages + s * SE, &tmap, x0, y0, plane_of(p), 0, &full[s]);
            if (wrapR) tma_load_4d(wraps + s * C::WRAP_STRIDE, &wmap, 0, y0, plane_of(p), 0, &full[s]);
        } else {
            issue_rows<G, 5>(stages + s * SE, &full[s], src, N, x0, y0, plane_of(p));
        }
    };
    // element (array a, row r) right of this thread's vector: column xi + V (= TX for the last lane)
    auto edge = [&](const T* st, int a, int r) -> T {
        return (wrapR && lane == 31) ? (wraps + (st - stages) / SE * C::WRAP_STRIDE)[(a * G::ROWS + r) * V] : st[G::idx(a, r, xi + V)];
    };
    if (w == 0 && elect_one()) {
#pragma unroll
        for (int p = 0; p < NS - 1; ++p)
            if (p <= zlen) issue_plane(p, p);
    }

    // arg phi at the V sites of this thread and at the site right of them, rows w and w+1 of a staged plane.  Every
    // thread evaluates the ten phases it needs itself (2.5 per site instead of 1): no exchange, hence no CTA barrier
    // anywhere in the march -- the warps of a CTA drift freely and only meet at the stage ring's mbarriers.
    auto args_of = [&](const T* st, float (&a0)[V + 1], float (&a1)[V + 1]) {
        const VecT pr = lds_vec<T, V>(st + G::idx(0, w, xi)), pi = lds_vec<T, V>(st + G::idx(1, w, xi));
        const VecT pry = lds_vec<T, V>(st + G::idx(0, w + 1, xi)), piy = lds_vec<T, V>(st + G::idx(1, w + 1, xi));
#pragma unroll
        for (int v = 0; v < V; ++v) {
            a0[v] = atan2_fast((float)pi.v[v], (float)pr.v[v]);
            a1[v] = atan2_fast((float)piy.v[v], (float)pry.v[v]);
        }
        a0[V] = atan2_fast((float)edge(st, 1, w), (float)edge(st, 0, w));
        a1[V] = atan2_fast((float)edge(st, 1, w + 1), (float)edge(st, 0, w + 1));
    };

    mbar_wait(&full[0], 0);
    // phases of the current plane and n_0, n_1 of its links (own sites; n_1 also right of the vector), carried along
    // the march together with the smallest margin of those link numbers
    float a[V + 1], ay[V + 1], n0c[V], n1c[V + 1], slack_c = 1.0f;
    args_of(stages, a, ay);
    {
        const VecT t0 = lds_vec<T, V>(stages + G::idx(2, w, xi)), t1 = lds_vec<T, V>(stages + G::idx(3, w, xi));
        const T t1x_e = edge(stages, 3, w);
#pragma unroll
        for (int v = 0; v <= V; ++v) {
            n1c[v] = link_number(a[v], ay[v], (float)(v < V ? t1.v[v < V ? v : 0] : t1x_e), slack_c);
            if (v < V) n0c[v < V ? v : 0] = link_number(a[v], a[v < V ? v + 1 : v], (float)t0.v[v < V ? v : 0], slack_c);
        }
    }

    // eps_2 of the plane below, carried in registers along the march
    VecT E2m;
    {
        const int zm = z0 == 0 ? N - 1 : z0 - 1;
        E2m = ldg_vec<T, V>(f.eps[2] + ((size_t)zm * N + (size_t)(y0 + w)) * N + (size_t)(x0 + xi));
    }

    double num = 0.0, den = 0.0, lsum = 0.0, rhs2 = 0.0, gmax = 0.0, vnum = 0.0, vden = 0.0;
    unsigned n_pierced = 0u, nonfinite = 0u;
    unsigned sum_abs_w = 0u;
    T gmax_t = T(0);

    for (int it = 0; it < zlen; ++it) {
        const T* sc = stages + (it % NS) * SE;
        const T* sn = stages + ((it + 1) % NS) * SE;

        // plane it+3 -> the stage that held plane it-1, once all TY warps have released it
        if (w == (rotate ? it % TY : 0) && it + NS - 1 <= zlen && elect_one()) {
            const int s = (it + NS - 1) % NS;
            if (it > 0) mbar_wait(&empty[s], ((it - 1) / NS) & 1);
            issue_plane(s, it + NS - 1);
        }

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
        float az[V + 1], azy[V + 1];
        args_of(sn, az, azy);

        // ---- phase B: everything of plane `it` ---------------------------------------------------------------------------
        const VecT pr = lds_vec<T, V>(sc + G::idx(0, w, xi)), pi = lds_vec<T, V>(sc + G::idx(1, w, xi));
        const VecT t0 = lds_vec<T, V>(sc + G::idx(2, w, xi)), t1 = lds_vec<T, V>(sc + G::idx(3, w, xi)), t2 = lds_vec<T, V>(sc + G::idx(4, w, xi));
        const VecT pry = lds_vec<T, V>(sc + G::idx(0, w + 1, xi)), piy = lds_vec<T, V>(sc + G::idx(1, w + 1, xi));
        const VecT t0y = lds_vec<T, V>(sc + G::idx(2, w + 1, xi)), t2y = lds_vec<T, V>(sc + G::idx(4, w + 1, xi));
        const VecT prz = lds_vec<T, V>(sn + G::idx(0, w, xi)), piz = lds_vec<T, V>(sn + G::idx(1, w, xi));
        const VecT t0z = lds_vec<T, V>(sn + G::idx(2, w, xi)), t1z = lds_vec<T, V>(sn + G::idx(3, w, xi));
        const T prx_e = edge(sc, 0, w), pix_e = edge(sc, 1, w);
        const T t1x_e = edge(sc, 3, w), t2x_e = edge(sc, 4, w);
        // E0 of the site to the left: previous element, else lane-1's last element, else (lane 0) the halo value
        T e0_left = __shfl_up_sync(0xffffffffu, E0.v[V - 1], 1);
        if (lane == 0) e0_left = e0_halo;

        // ---- winding (Eq. 11), fast path: the link numbers this thread-plane needs.  n_0, n_1 of this plane were formed
        //      one iteration ago (as the +z links); n_1, n_2 are also taken at the site right of the vector (n_j^{x+k_0}).
        float slack = slack_c;                               // margins of the carried n0c, n1c
        float n2[V + 1], n0y[V], n2y[V], n0z[V], n1z[V + 1];
        slack_c = 1.0f;
        {
            const T t1z_e = edge(sn, 3, w);
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
            const unsigned long long e = atomicAdd(doubt_count, 1ull);
            doubt_list[e] = (unsigned)((x0 + xi) / V) | ((unsigned)(y0 + w) << 10) | ((unsigned)(z0 + it) << 21);
            pierced = 0u;
            absw_u = 0u;
        }
        n_pierced += pierced;
        sum_abs_w += absw_u;
#pragma unroll
        for (int v = 0; v < V; ++v) n0c[v] = n0z[v];
#pragma unroll
        for (int v = 0; v <= V; ++v) { n1c[v] = n1z[v]; a[v] = az[v]; ay[v] = azy[v]; }

        T p_num = T(0), p_den = T(0), p_l = T(0), p_r2 = T(0), p_vn = T(0), p_vd = T(0);   // per thread and plane (V sites), then into the fp64 sums
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
            p_vn += K * Vp;   // potential-weighted estimator <v^2>_V (L86)
            p_vd += Gd * Vp;
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
        vnum += (double)p_vn; vden += (double)p_vd;
        E2m = E2;
        // this warp is done with stage `sc` (plane it): release it to the copy-issuing thread
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[it % NS]);
    }

    gmax = (double)gmax_t;
    DiagPartial acc = { (unsigned long long)n_pierced, (unsigned long long)sum_abs_w, num, den, lsum, gmax, rhs2, (unsigned long long)nonfinite, vnum, vden };
    block_reduce_store(acc, partials + blockIdx.x);
}

template <typename T, int TY>
int pick_zlen(int N, int ctas_per_sm, int max_partials)
{
    using C = DiagCfg<T, TY>;
    const long tiles = (long)(N / C::TX) * (N / TY);
    const int cands[5] = { 128, 64, 32, 16, 8 };
    for (int c : cands)   // the longest march that still gives >= 4 waves of resident CTAs (the prologue costs one plane)
        if (N % c == 0 && tiles * (N / c) + 2 <= max_partials && tiles * (N / c) >= 4L * ctas_per_sm * 148) return c;
    for (int c : cands)
        if (N % c == 0 && tiles * (N / c) + 2 <= max_partials) return c;
    return N;
}

template <typename T, int TY, int MINB, int NSTAGES = 4>
int launch_cfg(const DiagPtrs<T>& f, int N, const DiagCoef& c, DiagPartial* partials, int max_partials, DiagPartial* result,
               void* list, size_t list_bytes, const DiagMaps* tmap, cudaStream_t st)
{
    using C = DiagCfg<T, TY, NSTAGES>;
    auto kern = diag_march_kernel<T, TY, MINB, NSTAGES>;
    static bool configured = false;
    if (!configured) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM) != cudaSuccess) return AHS_ERR_CUDA;
        configured = true;
    }
    static const int zlen_env = [] { const char* e = getenv("AHS_DIAG_ZLEN"); return e ? atoi(e) : 0; }();
    const int zlen = (zlen_env > 0 && N % zlen_env == 0) ? zlen_env : pick_zlen<T, TY>(N, MINB, max_partials);
    const long blocks = (long)(N / C::TX) * (N / TY) * (N / zlen);
    // partials[blocks] collects the second pass, partials[blocks + 1].n_pierced is the length of the doubt list
    if (blocks + 2 > max_partials || list_bytes < sizeof(unsigned) * ((size_t)N * N * N / C::V)) return AHS_ERR_INVALID_ARG;
    DiagPartial* extra = partials + blocks;
    unsigned long long* count = &partials[blocks + 1].n_pierced;
    if (cudaMemsetAsync(extra, 0, 2 * sizeof(DiagPartial), st) != cudaSuccess) return AHS_ERR_CUDA;
    static const bool tma_off = getenv("AHS_NO_TMA") != nullptr;
    static const int rot = [] { const char* e = getenv("AHS_DIAG_ROT"); return e ? atoi(e) : 1; }();
    DiagMaps none;
    memset(&none, 0, sizeof(none));
    const bool use_tma = tmap && !tma_off;
    const DiagMaps& mp = use_tma ? *tmap : none;
    kern<<<(unsigned)blocks, C::NTHREADS, C::SMEM, st>>>(f, N, zlen, c, partials, (unsigned*)list, count, mp.tile, mp.wrap, use_tma ? 1 : 0, rot);
    if (cudaGetLastError() != cudaSuccess) return AHS_ERR_CUDA;
    diag_resolve_kernel<T><<<148 * 8, 128, 0, st>>>(f, N, (const unsigned*)list, count, extra);
    if (cudaGetLastError() != cudaSuccess) return AHS_ERR_CUDA;
    const int r = launch_diag_finish(partials, (int)blocks + 1, result, st);
    return r < 0 ? r : 3;
}

}  // namespace

template <typename T>
int launch_diag_march(const DiagPtrs<T>& f, int N, const DiagCoef& c, DiagPartial* partials, int max_partials, DiagPartial* result,
                      void* list, size_t list_bytes, const DiagMaps* tmap, cudaStream_t st)
{
    if (!march_supported<T>(N)) return AHS_ERR_INVALID_ARG;
    // 4-row tiles (3 CTAs/SM) by default; AHS_DIAG_TY=8 selects 8-row tiles, two CTAs per SM (experiments)
    static const int ty = [] { const char* e = getenv("AHS_DIAG_TY"); return e ? atoi(e) : 4; }();
    if (ty == 8) return launch_cfg<T, 8, 2>(f, N, c, partials, max_partials, result, list, list_bytes, nullptr, st);
    static const int ns = [] { const char* e = getenv("AHS_DIAG_NS"); return e ? atoi(e) : 4; }();
    if (ns == 5) return launch_cfg<T, 4, 3, 5>(f, N, c, partials, max_partials, result, list, list_bytes, tmap, st);
    if (ns == 3) return launch_cfg<T, 4, 3, 3>(f, N, c, partials, max_partials, result, list, list_bytes, tmap, st);
    return launch_cfg<T, 4, 3>(f, N, c, partials, max_partials, result, list, list_bytes, tmap, st);
}

// the tensor map of one (phi, theta) buffer for the default tile shape (4 rows): box (TX + V, TY + 1, 1, 5)
template <typename T>
bool make_diag_march_map(DiagMaps* out, const void* phi_re_base, int N, size_t array_bytes)
{
    using G = typename DiagCfg<T, 4>::G;
    if (!march_supported<T>(N)) return false;
    return make_tile_map<T>(&out->tile, phi_re_base, N, array_bytes, 5, G::PITCH, G::ROWS, 5) &&
           make_tile_map<T>(&out->wrap, phi_re_base, N, array_bytes, 5, G::V, G::ROWS, 5);
}
template bool make_diag_march_map<float>(DiagMaps*, const void*, int, size_t);
template bool make_diag_march_map<double>(DiagMaps*, const void*, int, size_t);

template int launch_diag_march<float>(const DiagPtrs<float>&, int, const DiagCoef&, DiagPartial*, int, DiagPartial*, void*, size_t, const DiagMaps*, cudaStream_t);
template int launch_diag_march<double>(const DiagPtrs<double>&, int, const DiagCoef&, DiagPartial*, int, DiagPartial*, void*, size_t, const DiagMaps*, cudaStream_t);

}  // namespace ahs
