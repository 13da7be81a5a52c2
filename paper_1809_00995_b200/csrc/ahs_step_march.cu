// ahs_step_march.cu -- the fused leapfrog step (Eqs. 4-7) as a 2.5D z-march for sm_100a.
//
// One CTA owns a tile of TX x TY sites in (x, y) (TX = 32 lanes x one 16-byte vector, TY = 8 rows = 8 compute
// warps) and marches over `zlen` planes.  A ninth warp is the producer: it streams the level-n fields phi, theta
// (5 arrays) of plane k+2 into a 3-stage ring of halo'd shared-memory tiles with cp.async.bulk (UBLKCP) + mbarrier
// while planes k, k+1 are in use (ahs_stage.cuh); Pi and eps (no halo) are read with streaming 16-byte loads and
// all ten outputs leave as 16-byte stores.
//
// Compute-once form.  Each site owner computes, from raw phi, theta of the site and of its FORWARD neighbours only,
//   U_j = exp(-i theta_j)                         3 sincos       (link phases, Eq. 3 / L46-51, q = +1)
//   f_j = U_j phi^{x+k_j}, b_j = conj(U_j) phi^x, J_j = Im[conj(phi^x) f_j]
//   S_01, S_02, S_12 = sin Xi_ij^x                3 sin          (plaquettes based at x, Eq. 3)
// and receives the six products owned by its BACKWARD neighbours:
//   -x : b_0, S_01, S_02   through a small shared-memory exchange (slot lane-1; slot "-1" = halo column)
//   -y : b_1, S_01, S_12   through a shared-memory exchange row (row -1 = halo row)
//   -z : b_2, S_02, S_12   in the thread's own registers from the previous plane of the march.
// The products of the halo row y0-1 and of the halo column x0-1 are recomputed by the producer warp (same
// function, same inputs => bit-identical link phases on both sides of a tile edge, which is what keeps the Gauss
// law at roundoff: it needs the same U in Eq. 4 and Eq. 5).  Then
//   Lap    = sum_j (f_j + b_j^{x-k_j}) - 6 phi                                              (Eq. 4)
//   curl_0 = (S01 - S01^{-y}) + (S02 - S02^{-z}),  curl_1 = (S01^{-x} - S01) + (S12 - S12^{-z}),
//   curl_2 = (S02^{-x} - S02) + (S12^{-y} - S12)                                            (Eq. 5)
// followed by the kicks and the drift into the other (phi, theta) buffer (Eqs. 6-7).
// The paper's kernels stage raw fields per kernel and recompute every phase (L107-109); this is a different design.
#include <cstdlib>
#include <cstring>

#include "ahs_internal.cuh"
#include "ahs_math.cuh"
#include "ahs_stage.cuh"

namespace ahs {

namespace {

template <typename T> struct StepCoefT { T c1, c2, c3, d1, d2, d3, dt, sigma2; };

template <typename T> struct NativeVec;
template <> struct NativeVec<float> { using type = float4; };
template <> struct NativeVec<double> { using type = double2; };

template <typename T>
struct MarchCfg {
    static constexpr int V = 16 / sizeof(T);
    static constexpr int TY = 8;
    static constexpr int NSTAGE = 3;
    using G = TileGeom<T, V, TY, 5, NSTAGE>;
    static constexpr int TX = G::TX;
    static constexpr int NTHREADS = (TY + 1) * 32;
    static constexpr int XP = 33;                         // x-exchange pitch: slot 0 = halo column, slot l+1 = lane l
    static constexpr int YEX_ELEMS = 4 * (TY + 1) * TX;   // b1.re, b1.im, S01, S12 for rows -1 .. TY-1
    static constexpr int XEX_ELEMS = 4 * TY * XP;         // b0.re, b0.im, S01, S02
    static constexpr size_t SMEM = 128 + sizeof(T) * (size_t)(NSTAGE * G::STAGE_ELEMS + YEX_ELEMS + XEX_ELEMS);
};

template <typename T, int V>
__device__ __forceinline__ Vec<T, V> lds_vec(const T* p) { return *reinterpret_cast<const Vec<T, V>*>(p); }
template <typename T, int V>
__device__ __forceinline__ void sts_vec(T* p, const Vec<T, V>& v) { *reinterpret_cast<Vec<T, V>*>(p) = v; }

// streaming 16-byte global load / store (each momentum value is read once and written once per step)
template <typename T, int V>
__device__ __forceinline__ Vec<T, V> ldg_vec(const T* p)
{
    using NV = typename NativeVec<T>::type;
    const NV n = __ldcs(reinterpret_cast<const NV*>(p));
    Vec<T, V> r;
    memcpy(&r, &n, sizeof(r));
    return r;
}
template <typename T, int V>
__device__ __forceinline__ void stg_vec(T* p, const Vec<T, V>& v)
{
    using NV = typename NativeVec<T>::type;
    NV n;
    memcpy(&n, &v, sizeof(n));
    *reinterpret_cast<NV*>(p) = n;
}

// Barrier over the whole CTA, executed from warp-specialised (warp-uniform) branches: a named barrier with an
// explicit thread count, as the producer warp and the compute warps reach it from different code.
template <int NT>
__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 1, %0;" ::"n"(NT) : "memory"); }

template <typename T, int MINB>
__global__ void __launch_bounds__(MarchCfg<T>::NTHREADS, MINB) step_march_kernel(FieldPtrs<T> f, int N, int zlen, StepCoefT<T> k)
{
    using C = MarchCfg<T>;
    using G = typename C::G;
    using VecT = Vec<T, C::V>;
    constexpr int V = C::V, TX = C::TX, TY = C::TY, NS = C::NSTAGE, XP = C::XP, SE = G::STAGE_ELEMS;

    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);
    T* stages = reinterpret_cast<T*>(smem + 128);
    T* yex = stages + NS * SE;
    T* xex = yex + C::YEX_ELEMS;

    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int tiles_x = N / TX, tiles_y = N / TY;
    int bid = blockIdx.x;
    const int tx = bid % tiles_x;
    bid /= tiles_x;
    const int ty = bid % tiles_y, zc = bid / tiles_y;
    const int x0 = tx * TX, y0 = ty * TY, z0 = zc * zlen;
    const int xi = V * lane;

    const T* const src[5] = { f.phi_re, f.phi_im, f.th[0], f.th[1], f.th[2] };

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();

    // plane index i of this CTA's march = lattice plane z0 - 1 + i (periodic)
    auto plane_of = [&](int i) { const int z = z0 - 1 + i; return z < 0 ? z + N : (z >= N ? z - N : z); };
    if (w == TY) {
#pragma unroll
        for (int i = 0; i < NS; ++i) issue_plane<G>(stages + i * SE, &full[i], src, N, x0, y0, plane_of(i), lane);
    }

    // products of the previous plane, carried in registers: b_2 = conj(U_2) phi, S_02, S_12
    T cb2r[V], cb2i[V], cS02[V], cS12[V];

    // ---- prologue: z-products of plane z0-1 (needs planes z0-1 and z0) ---------------------------------------------
    mbar_wait(&full[0], 0);
    mbar_wait(&full[1], 0);
    if (w < TY) {
        const T* sc = stages;
        const T* sn = stages + SE;
        const VecT pr = lds_vec<T, V>(sc + G::idx(0, w, xi)), pi = lds_vec<T, V>(sc + G::idx(1, w, xi));
        const VecT t0 = lds_vec<T, V>(sc + G::idx(2, w, xi)), t1 = lds_vec<T, V>(sc + G::idx(3, w, xi)), t2 = lds_vec<T, V>(sc + G::idx(4, w, xi));
        const VecT t2y = lds_vec<T, V>(sc + G::idx(4, w + 1, xi));
        const VecT t0z = lds_vec<T, V>(sn + G::idx(2, w, xi)), t1z = lds_vec<T, V>(sn + G::idx(3, w, xi));
        const T t2x_edge = sc[G::idx(4, w, xi + V)];
#pragma unroll
        for (int v = 0; v < V; ++v) {
            T s, c;
            sincos_t(t2.v[v], s, c);
            const Cx<T> b = mulUc<T>(c, s, { pr.v[v], pi.v[v] });
            cb2r[v] = b.re;
            cb2i[v] = b.im;
            const T t2x = (v < V - 1) ? t2.v[v + 1 < V ? v + 1 : v] : t2x_edge;
            cS02[v] = sin_t(t0.v[v] + t2x - t0z.v[v] - t2.v[v]);
            cS12[v] = sin_t(t1.v[v] + t2y.v[v] - t1z.v[v] - t2.v[v]);
        }
    }
    __syncthreads();

    // ---- the march -----------------------------------------------------------------------------------------------------
    for (int it = 1; it <= zlen; ++it) {
        const T* sc = stages + (it % NS) * SE;
        const T* sn = stages + ((it + 1) % NS) * SE;

        if (w == TY) {
            // ------------------------------- producer + halo warp -------------------------------------------------------
            if (it + 2 <= zlen + 1) {
                const int s = (it + 2) % NS;   // held plane it-1: every thread finished it before the last barrier
                issue_plane<G>(stages + s * SE, &full[s], src, N, x0, y0, plane_of(it + 2), lane);
            }
            mbar_wait(&full[(it + 1) % NS], ((it + 1) / NS) & 1);
            {   // halo row y0-1: b_1, S_01, S_12 -> exchange row 0
                const VecT pr = lds_vec<T, V>(sc + G::idx(0, -1, xi)), pi = lds_vec<T, V>(sc + G::idx(1, -1, xi));
                const VecT t0 = lds_vec<T, V>(sc + G::idx(2, -1, xi)), t1 = lds_vec<T, V>(sc + G::idx(3, -1, xi)), t2 = lds_vec<T, V>(sc + G::idx(4, -1, xi));
                const VecT t0y = lds_vec<T, V>(sc + G::idx(2, 0, xi)), t2y = lds_vec<T, V>(sc + G::idx(4, 0, xi));
                const VecT t1z = lds_vec<T, V>(sn + G::idx(3, -1, xi));
                const T t1x_edge = sc[G::idx(3, -1, xi + V)];
                VecT b1r, b1i, s01, s12;
#pragma unroll
                for (int v = 0; v < V; ++v) {
                    T s, c;
                    sincos_t(t1.v[v], s, c);
                    const Cx<T> b = mulUc<T>(c, s, { pr.v[v], pi.v[v] });
                    b1r.v[v] = b.re;
                    b1i.v[v] = b.im;
                    const T t1x = (v < V - 1) ? t1.v[v + 1 < V ? v + 1 : v] : t1x_edge;
                    s01.v[v] = sin_t(t0.v[v] + t1x - t0y.v[v] - t1.v[v]);
                    s12.v[v] = sin_t(t1.v[v] + t2y.v[v] - t1z.v[v] - t2.v[v]);
                }
                sts_vec<T, V>(yex + (0 * (TY + 1) + 0) * TX + xi, b1r);
                sts_vec<T, V>(yex + (1 * (TY + 1) + 0) * TX + xi, b1i);
                sts_vec<T, V>(yex + (2 * (TY + 1) + 0) * TX + xi, s01);
                sts_vec<T, V>(yex + (3 * (TY + 1) + 0) * TX + xi, s12);
            }
            if (lane < TY) {   // halo column x0-1, row r = lane: b_0, S_01, S_02 -> exchange slot 0
                const int r = lane;
                const T pr = sc[G::idx(0, r, -1)], pi = sc[G::idx(1, r, -1)];
                const T t0 = sc[G::idx(2, r, -1)], t1 = sc[G::idx(3, r, -1)], t2 = sc[G::idx(4, r, -1)];
                const T t1x = sc[G::idx(3, r, 0)], t2x = sc[G::idx(4, r, 0)];
                const T t0y = sc[G::idx(2, r + 1, -1)], t0z = sn[G::idx(2, r, -1)];
                T s, c;
                sincos_t(t0, s, c);
                const Cx<T> b = mulUc<T>(c, s, { pr, pi });
                xex[(0 * TY + r) * XP] = b.re;
                xex[(1 * TY + r) * XP] = b.im;
                xex[(2 * TY + r) * XP] = sin_t(t0 + t1x - t0y - t1);
                xex[(3 * TY + r) * XP] = sin_t(t0 + t2x - t0z - t2);
            }
            cta_sync<C::NTHREADS>();   // (A) products visible
            cta_sync<C::NTHREADS>();   // (B) exchange buffers, and the stage of plane it, are free again
            continue;
        }

        // ----------------------------------- compute warps ---------------------------------------------------------------
        const int z = z0 + it - 1;
        const size_t g = ((size_t)z * N + (size_t)(y0 + w)) * N + (size_t)(x0 + xi);
        const VecT Pr = ldg_vec<T, V>(f.pi_re + g), Pi = ldg_vec<T, V>(f.pi_im + g);
        const VecT E0 = ldg_vec<T, V>(f.eps[0] + g), E1 = ldg_vec<T, V>(f.eps[1] + g), E2 = ldg_vec<T, V>(f.eps[2] + g);

        mbar_wait(&full[(it + 1) % NS], ((it + 1) / NS) & 1);

        const VecT pr = lds_vec<T, V>(sc + G::idx(0, w, xi)), pi = lds_vec<T, V>(sc + G::idx(1, w, xi));
        const VecT t0 = lds_vec<T, V>(sc + G::idx(2, w, xi)), t1 = lds_vec<T, V>(sc + G::idx(3, w, xi)), t2 = lds_vec<T, V>(sc + G::idx(4, w, xi));
        T lfr[V], lfi[V], ep0[V], ep1[V], ep2[V], b0r[V], b0i[V], S01[V], S02[V], S12[V], nb2r[V], nb2i[V];
        {
            const VecT pry = lds_vec<T, V>(sc + G::idx(0, w + 1, xi)), piy = lds_vec<T, V>(sc + G::idx(1, w + 1, xi));
            const VecT t0y = lds_vec<T, V>(sc + G::idx(2, w + 1, xi)), t2y = lds_vec<T, V>(sc + G::idx(4, w + 1, xi));
            const VecT prz = lds_vec<T, V>(sn + G::idx(0, w, xi)), piz = lds_vec<T, V>(sn + G::idx(1, w, xi));
            const VecT t0z = lds_vec<T, V>(sn + G::idx(2, w, xi)), t1z = lds_vec<T, V>(sn + G::idx(3, w, xi));
            const T prx_e = sc[G::idx(0, w, xi + V)], pix_e = sc[G::idx(1, w, xi + V)];
            const T t1x_e = sc[G::idx(3, w, xi + V)], t2x_e = sc[G::idx(4, w, xi + V)];
            VecT yb1r, yb1i, yS01, yS12;
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const int vn = v + 1 < V ? v + 1 : v;
                const T prx = (v < V - 1) ? pr.v[vn] : prx_e, pix = (v < V - 1) ? pi.v[vn] : pix_e;
                const T t1x = (v < V - 1) ? t1.v[vn] : t1x_e, t2x = (v < V - 1) ? t2.v[vn] : t2x_e;
                const Cx<T> ph = { pr.v[v], pi.v[v] };
                T s, c;
                sincos_t(t0.v[v], s, c);
                const Cx<T> f0 = mulU<T>(c, s, { prx, pix });
                const Cx<T> b0 = mulUc<T>(c, s, ph);
                sincos_t(t1.v[v], s, c);
                const Cx<T> f1 = mulU<T>(c, s, { pry.v[v], piy.v[v] });
                const Cx<T> b1 = mulUc<T>(c, s, ph);
                sincos_t(t2.v[v], s, c);
                const Cx<T> f2 = mulU<T>(c, s, { prz.v[v], piz.v[v] });
                const Cx<T> b2 = mulUc<T>(c, s, ph);
                lfr[v] = (f0.re + f1.re) + f2.re;
                lfi[v] = (f0.im + f1.im) + f2.im;
                // J_j = Im[conj(phi^x) U_j phi^{x+k_j}]  (Eq. 5, 2nd term)
                ep0[v] = k.d1 * E0.v[v] + k.d2 * (ph.re * f0.im - ph.im * f0.re);
                ep1[v] = k.d1 * E1.v[v] + k.d2 * (ph.re * f1.im - ph.im * f1.re);
                ep2[v] = k.d1 * E2.v[v] + k.d2 * (ph.re * f2.im - ph.im * f2.re);
                b0r[v] = b0.re; b0i[v] = b0.im;
                yb1r.v[v] = b1.re; yb1i.v[v] = b1.im;
                nb2r[v] = b2.re; nb2i[v] = b2.im;
                // Xi_ij^x = th_i^x + th_j^{x+k_i} - th_i^{x+k_j} - th_j^x  (Eq. 3)
                S01[v] = sin_t(t0.v[v] + t1x - t0y.v[v] - t1.v[v]);
                S02[v] = sin_t(t0.v[v] + t2x - t0z.v[v] - t2.v[v]);
                S12[v] = sin_t(t1.v[v] + t2y.v[v] - t1z.v[v] - t2.v[v]);
                yS01.v[v] = S01[v];
                yS12.v[v] = S12[v];
            }
            sts_vec<T, V>(yex + (0 * (TY + 1) + w + 1) * TX + xi, yb1r);
            sts_vec<T, V>(yex + (1 * (TY + 1) + w + 1) * TX + xi, yb1i);
            sts_vec<T, V>(yex + (2 * (TY + 1) + w + 1) * TX + xi, yS01);
            sts_vec<T, V>(yex + (3 * (TY + 1) + w + 1) * TX + xi, yS12);
            xex[(0 * TY + w) * XP + lane + 1] = b0r[V - 1];
            xex[(1 * TY + w) * XP + lane + 1] = b0i[V - 1];
            xex[(2 * TY + w) * XP + lane + 1] = S01[V - 1];
            xex[(3 * TY + w) * XP + lane + 1] = S02[V - 1];
        }
        cta_sync<C::NTHREADS>();   // (A)
        {
            const VecT yb1r = lds_vec<T, V>(yex + (0 * (TY + 1) + w) * TX + xi), yb1i = lds_vec<T, V>(yex + (1 * (TY + 1) + w) * TX + xi);
            const VecT yS01 = lds_vec<T, V>(yex + (2 * (TY + 1) + w) * TX + xi), yS12 = lds_vec<T, V>(yex + (3 * (TY + 1) + w) * TX + xi);
            const T xb0r = xex[(0 * TY + w) * XP + lane], xb0i = xex[(1 * TY + w) * XP + lane];
            const T xS01 = xex[(2 * TY + w) * XP + lane], xS02 = xex[(3 * TY + w) * XP + lane];
            VecT oPr, oPi, oE0, oE1, oE2, oFr, oFi, oT0, oT1, oT2;
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const int vp = v > 0 ? v - 1 : 0;
                const T mb0r = v > 0 ? b0r[vp] : xb0r, mb0i = v > 0 ? b0i[vp] : xb0i;
                const T mS01 = v > 0 ? S01[vp] : xS01, mS02 = v > 0 ? S02[vp] : xS02;
                const T lap_re = (lfr[v] - T(6) * pr.v[v]) + ((mb0r + yb1r.v[v]) + cb2r[v]);
                const T lap_im = (lfi[v] - T(6) * pi.v[v]) + ((mb0i + yb1i.v[v]) + cb2i[v]);
                const T higgs = k.c3 * (pr.v[v] * pr.v[v] + pi.v[v] * pi.v[v] - k.sigma2);
                const T npr = k.c1 * Pr.v[v] - higgs * pr.v[v] + k.c2 * lap_re;     // Eq. 4
                const T npi = k.c1 * Pi.v[v] - higgs * pi.v[v] + k.c2 * lap_im;
                const T curl0 = (S01[v] - yS01.v[v]) + (S02[v] - cS02[v]);
                const T curl1 = (mS01 - S01[v]) + (S12[v] - cS12[v]);
                const T curl2 = (mS02 - S02[v]) + (yS12.v[v] - S12[v]);
                const T ne0 = ep0[v] - k.d3 * curl0, ne1 = ep1[v] - k.d3 * curl1, ne2 = ep2[v] - k.d3 * curl2;   // Eq. 5
                oPr.v[v] = npr; oPi.v[v] = npi; oE0.v[v] = ne0; oE1.v[v] = ne1; oE2.v[v] = ne2;
                oFr.v[v] = pr.v[v] + k.dt * npr;                                      // Eq. 6
                oFi.v[v] = pi.v[v] + k.dt * npi;
                oT0.v[v] = t0.v[v] + k.dt * ne0;                                      // Eq. 7
                oT1.v[v] = t1.v[v] + k.dt * ne1;
                oT2.v[v] = t2.v[v] + k.dt * ne2;
                cb2r[v] = nb2r[v]; cb2i[v] = nb2i[v]; cS02[v] = S02[v]; cS12[v] = S12[v];
            }
            stg_vec<T, V>(f.pi_re + g, oPr); stg_vec<T, V>(f.pi_im + g, oPi);
            stg_vec<T, V>(f.eps[0] + g, oE0); stg_vec<T, V>(f.eps[1] + g, oE1); stg_vec<T, V>(f.eps[2] + g, oE2);
            stg_vec<T, V>(f.phi_re_out + g, oFr); stg_vec<T, V>(f.phi_im_out + g, oFi);
            stg_vec<T, V>(f.th_out[0] + g, oT0); stg_vec<T, V>(f.th_out[1] + g, oT1); stg_vec<T, V>(f.th_out[2] + g, oT2);
        }
        cta_sync<C::NTHREADS>();   // (B)
    }
}

template <typename T>
int pick_zlen(int N)
{
    using C = MarchCfg<T>;
    const long tiles = (long)(N / C::TX) * (N / C::TY);
    const int cands[4] = { 64, 32, 16, 8 };
    for (int c : cands)
        if (N % c == 0 && tiles * (N / c) >= 8 * 148) return c;   // enough CTAs for >= 4 waves at 2 CTAs per SM
    return 8;
}

}  // namespace

template <typename T>
bool march_supported(int N)
{
    using C = MarchCfg<T>;
    return N >= C::TX && N % C::TX == 0 && N % C::TY == 0;
}

template <typename T>
int launch_step_march(const FieldPtrs<T>& f, int N, const StepCoef& c, cudaStream_t st)
{
    using C = MarchCfg<T>;
    if (!march_supported<T>(N)) return AHS_ERR_INVALID_ARG;
    // tuning knob (experiments only): AHS_MARCH_MINB=1 compiles for one resident CTA per SM (more registers)
    static const int minb = [] { const char* e = getenv("AHS_MARCH_MINB"); return (e && e[0] == '1') ? 1 : 2; }();
    auto kern = minb == 1 ? step_march_kernel<T, 1> : step_march_kernel<T, 2>;
    static bool configured = false;
    if (!configured) {
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM) != cudaSuccess) return AHS_ERR_CUDA;
        configured = true;
    }
    const int zlen = pick_zlen<T>(N);
    const long blocks = (long)(N / C::TX) * (N / C::TY) * (N / zlen);
    StepCoefT<T> k = { (T)c.c1, (T)c.c2, (T)c.c3, (T)c.d1, (T)c.d2, (T)c.d3, (T)c.dt, (T)c.sigma2 };
    kern<<<(unsigned)blocks, C::NTHREADS, C::SMEM, st>>>(f, N, zlen, k);
    return cudaGetLastError() == cudaSuccess ? 1 : AHS_ERR_CUDA;
}

// the marching diagnostics kernel lives in ahs_diag_march.cu
template bool march_supported<float>(int);
template bool march_supported<double>(int);
template int launch_step_march<float>(const FieldPtrs<float>&, int, const StepCoef&, cudaStream_t);
template int launch_step_march<double>(const FieldPtrs<double>&, int, const StepCoef&, cudaStream_t);

}  // namespace ahs
