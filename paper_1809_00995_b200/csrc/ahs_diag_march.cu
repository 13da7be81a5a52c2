// ahs_diag_march.cu -- the fused network diagnostics (winding Eq. 11, <v^2>_L Eqs. 9-10 with the weight of Eq. 2,
// Gauss residual) as a 2.5D z-march for sm_100a: one read of the ten arrays per call.
//
// Same tile and staging as the step kernel (ahs_step_march.cu): a CTA owns TX x TY sites in (x, y) and marches over a
// z-chunk; phi_re, phi_im, theta_0..2 of plane k+3 are streamed by the copy engine (one tensor-map TMA copy per plane, row
// copies on the periodic edge in y) into a 4-slot ring of halo'd shared-memory tiles (one `full` mbarrier per slot; the last
// warp to finish with a slot re-fills it) while planes k, k+1 are in use; eps_1 and the row below it ride in the same slot
// (one more tensor copy); Pi, eps_0, eps_2 are read with streaming 16-byte loads.  Inside a CTA the four warps sit side by side
// along x and a warp's lanes are 8 vectors along x by 4 rows.
// All the estimators need only FORWARD neighbours (x+k_i, x+k_i+k_j) of phi, theta -- except the divergence of eps,
// whose -x / -y / -z terms come by one scalar load, the staged row below and a carried register.
//
// The kernel is bound by fp32 arithmetic, not by HBM (profiles/r5_diag1024_f32_full.md), so ALL its arithmetic runs on pairs
// of neighbouring sites with sm_100's packed fp32 instructions (ahs_pack.cuh; for fp64 lattices the same expressions element
// by element), and the sines / cosines inside the <v^2> sums may go to the special-function unit (SumsTrig below).
//
// Winding.  arg phi / 2 pi (branch-free atan2_turns) is needed at the ten points of plane k+1 around a thread's V sites.  On
// fp32 lattices a warp evaluates each phase of its 32 x 4 region and of that region's halo once and hands them round through
// a private shared-memory tile (__syncwarp only); on fp64 lattices every thread evaluates its ten itself.  Either way there is
// NO exchange between warps and therefore no CTA barrier in the march: the warps of a CTA drift freely and meet only at the
// stage ring's `full` mbarriers (an earlier version computed each phase once per CTA into a shared arg tile and lost 31 % of
// its issue slots at the per-plane barrier, profiles/HISTORY.md r2).  The phases are carried to the next plane in registers.
// The link numbers n_i^x = rint(t), t = arg^{x+k_i}/2pi - arg^x/2pi - theta_i^x/2pi, are formed in fp32 and
// W_ij = -(n_i^x + n_j^{x+k_i} - n_i^{x+k_j} - n_j^x) is summed exactly.  The decision is the fp64 one:
//   |t - t_exact| <= 2 eps_a + 3e-8 + 1.6e-7 (1 + |t|) turns with eps_a <= 7.6e-8 turns per phase (atan2_turns, ahs_trig.cuh;
//   the remaining terms: rounding of the difference, of the fma, of 1/2pi in fp32 and of theta when the lattice is fp64),
//   i.e. <= 2.4e-7 + 1.6e-7 |t|;
// whenever some link of a thread-plane lies within kTieMargin (1 + |t|) = 4e-6 (1 + |t|) turns of a half-integer -- more
// than ten times that bound -- or a plaquette has |W| >= 2 (never seen on physical fields), the thread drops the plane's fast
// count and appends it to a device-side doubt list, which diag_resolve_kernel redoes with fp64 atan2 (~4e-4 of the
// thread-planes), so every rint is the one an all-fp64 evaluation takes and the march itself never diverges.
// <v^2>_L sums: products and the sum over the 16-byte vector of a thread in the storage type, then fp64 accumulation.
// The paper runs Winding and VelRWLag as two kernels over raw fields with a CUB block sum and a host-side final sum
// (L140); this is a different design.
#include <cstring>

#include "ahs_internal.cuh"
#include "ahs_math.cuh"
#include "ahs_pack.cuh"
#include "ahs_reduce.cuh"
#include "ahs_stage.cuh"
#include "ahs_tma.cuh"
#include "ahs_trig.cuh"

namespace ahs {

namespace {

constexpr double kInv2Pi = 0.15915494309189535;
constexpr float kTieMargin = 4e-6f;   // in units of a full turn, relative to 1 + |t|: more than ten times the error bound

template <typename T>
struct DiagCfg {
    static constexpr int V = 16 / sizeof(T);
    static constexpr int TY = 4;                             // 4-row tiles (4 warps)
    static constexpr int MINB = sizeof(T) == 8 ? 2 : 3;      // CTAs per SM the register budget is cut for (fp64: 255 registers, no spills)
    static constexpr int NSTAGE = 4;
    using G = TileGeom<T, V, TY, 5, NSTAGE, 0, 0>;           // a stage: phi_re, phi_im, theta_0..2 of one plane, forward halo only
    static constexpr int TX = G::TX;
    static constexpr int NTHREADS = TY * 32;
    static constexpr int STAGE_STRIDE = (int)(((G::STAGE_BYTES + 127u) & ~127u) / sizeof(T));   // tensor copies land 128-byte aligned
    // right-edge tiles under TMA: the wrapped forward halo column (x = 0 .. V-1) of a plane lands in a side buffer
    static constexpr int WRAP_STRIDE = (int)(((5 * G::ROWS * V * sizeof(T) + 127) & ~(size_t)127) / sizeof(T));
    // eps_1 (rows y0-1 .. y0+TY-1, no halo in x) of the same plane rides in the slot too: the divergence needs the row below, and a
    // register-held global load of it was consumed right at the top of the plane by the compiler (profiles/r5_diag1024_f32_full.md)
    static constexpr int E1_OFF = STAGE_STRIDE + WRAP_STRIDE;
    static constexpr int E1_ELEMS = (TY + 1) * TX;
    static constexpr uint32_t E1_BYTES = E1_ELEMS * sizeof(T);
    static_assert(E1_BYTES % 128 == 0, "slots stay 128-byte aligned");
    static constexpr int SLOT_STRIDE = E1_OFF + E1_ELEMS;   // a ring slot = a stage, its side buffer, the eps_1 rows
    // A warp covers WX columns x TY rows of the tile (lane = 8 vectors in x by 4 rows).  Its phase tile holds arg phi / 2 pi of one plane at
    // those sites plus the row above and the column to the right ((TY + 1) x (WX + 1) values, rows PP apart): each phase is evaluated
    // once per warp instead of by every thread that needs it.
    static constexpr int NWARPS = NTHREADS / 32;
    static constexpr int WX = 8 * V;
    static constexpr int PP = WX + 4;                          // row pitch: the row vectors stay 16-byte aligned, rows fall in different banks
    static constexpr int PT_FLOATS = (TY + 1) * PP;
    static constexpr int NEXTRA = WX + 1 + TY;                 // the halo of a warp's region: row TY (WX + 1 values), column WX of rows 0 .. TY-1
    static constexpr bool SHARE_PHASES = sizeof(T) == 4;       // fp64 lattices (half as many sites per warp) are faster without: 3.48 vs 3.57 ms at 512^3
    static_assert(TY == 4 && TX == NWARPS * WX, "4 rows of 8 lanes; the warps side by side span the tile");
    static_assert(NEXTRA <= 64, "two halo phases per lane");
    static constexpr size_t RING_BYTES = sizeof(T) * (size_t)(NSTAGE * SLOT_STRIDE);
    static constexpr size_t SMEM = 128 + RING_BYTES + sizeof(float) * (size_t)(NWARPS * PT_FLOATS);
};

// Link numbers of two links s -> t with angles th, fast path, all in fp32 and in turns: t = (at - as) - th / 2 pi from the
// atan2_turns phases, n = rint(t) (ties to even) as floats.  rmax / tmax collect max |t - n| and max |t| over the links of
// a thread-plane: whenever rmax < 1/2 - kTieMargin (1 + tmax) every n IS the fp64 decision (error bound in the header).
// Everything here is branch-free; NaN never raises rmax (fmaxf drops it) but makes the plaquette sums NaN, which the
// caller tests.
__device__ __forceinline__ float2 link_numbers(float2 as, float2 at, float2 th, float& rmax_x, float& rmax_y, float& tmax)
{
    const float2 t = pk::fma(th, pk::splat(-0.15915494309189535f), pk::sub(at, as));
    const float2 n = pk::add(pk::add(t, pk::splat(12582912.0f)), pk::splat(-12582912.0f));   // 1.5 * 2^23
    const float2 r = pk::sub(t, n);
    rmax_x = fmaxf(rmax_x, fabsf(r.x));
    rmax_y = fmaxf(rmax_y, fabsf(r.y));
    tmax = fmaxf(tmax, fmaxf(fabsf(t.x), fabsf(t.y)));
    return n;
}
// The trigonometry of the <v^2> sums (link phases of the gradient term, plaquette chords of the magnetic term), by TRIG:
//   AHS_TRIG_POLYNOMIAL  the Cody-Waite + polynomial routines of ahs_trig.cuh (<= 1-2 ulp), as in the step kernel;
//   AHS_TRIG_HARDWARE    (fp32 lattices only) the special-function unit's sine / cosine, |error| <= 2^-21.4 / 2^-21.2 for |x| <= pi
//                        and about |x| 2^-23 beyond (the unit takes x / 2 pi rounded to fp32): a quarter of the kernel's FMA-pipe
//                        time moves to the otherwise idle XU pipe.  The winding never uses it.
// sum over the ordered pairs (R12) of 1 - cos Xi = sum over the three plaquettes of |exp(i Xi) - 1|^2 = 4 sin^2(Xi/2): no
// cancellation at small Xi
template <int TRIG> struct SumsTrig {
    template <typename P> __device__ __forceinline__ static void link_phase(P th, P& s, P& c) { sincos_pair(th, s, c); }
    template <typename P> __device__ __forceinline__ static P plaquettes(P X01, P X02, P X12)
    {
        const P h01 = chord_pair(X01), h02 = chord_pair(X02), h12 = chord_pair(X12);   // +- 2 sin(Xi/2)
        return pk::fma(h01, h01, pk::fma(h02, h02, pk::mul(h12, h12)));
    }
};
template <> struct SumsTrig<AHS_TRIG_HARDWARE> {
    __device__ __forceinline__ static void link_phase(float2 th, float2& s, float2& c) { sincos_hw(th, s, c); }
    __device__ __forceinline__ static float2 plaquettes(float2 X01, float2 X02, float2 X12)
    {
        const float2 half = pk::splat(0.5f);
        const float2 h01 = sin_hw(pk::mul(half, X01)), h02 = sin_hw(pk::mul(half, X02)), h12 = sin_hw(pk::mul(half, X12));
        return pk::mul(pk::splat(4.0f), pk::fma(h01, h01, pk::fma(h02, h02, pk::mul(h12, h12))));
    }
};
__device__ __forceinline__ float2 to_float2(float2 v) { return v; }
__device__ __forceinline__ float2 to_float2(double2 v) { return make_float2((float)v.x, (float)v.y); }

// Second pass over the doubt list: the winding of the V sites of each listed (x/V, y, z), every phase and every quotient
// in fp64 straight from global memory (same arithmetic as diag_generic_kernel), added to one extra partial record.
// Integer sums: the order of the atomics does not matter.  ~4e-4 of the thread-planes end up here on smooth or random
// fields; resolving them in-line (an out-of-line call inside the march) made every warp of the CTA wait for the one
// that took the slow path (profiles/HISTORY.md r2: 30 % of the issue slots), a separate pass costs ~0.1 ms at 1024^3.
template <typename T>
__global__ void __launch_bounds__(128) diag_resolve_kernel(DiagPtrs<T> f, int N, int periodic_z, const unsigned* __restrict__ list,
                                                           const unsigned long long* __restrict__ count, DiagPartial* __restrict__ extra)
{
    constexpr int V = 16 / sizeof(T);
    const unsigned long long n = *count;
    unsigned pierced = 0u, absw = 0u;
    for (unsigned long long e = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned u = list[e];
        const int xv = (int)(u & 1023u), y = (int)((u >> 10) & 2047u), z = (int)(u >> 21);
        const int yp = y + 1 == N ? 0 : y + 1, zp = (periodic_z && z + 1 == N) ? 0 : z + 1;   // (z is the LOCAL plane index: a slab has its ghost above)
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

template <typename T, int TRIG>
__global__ void __launch_bounds__(DiagCfg<T>::NTHREADS, DiagCfg<T>::MINB)
diag_march_kernel(DiagPtrs<T> f, int N, ZRange zr, int nchunks, DiagCoef kd, DiagPartial* __restrict__ partials, unsigned* __restrict__ doubt_list,
                  unsigned long long* __restrict__ doubt_count, const __grid_constant__ CUtensorMap tmap,
                  const __grid_constant__ CUtensorMap wmap, const __grid_constant__ CUtensorMap emap, int use_tma)
{
    using C = DiagCfg<T>;
    using G = typename C::G;
    using VecT = Vec<T, C::V>;
    using P = pk::Pair<T>;
    constexpr int V = C::V, NP = V / 2, TX = C::TX, TY = C::TY, NS = C::NSTAGE, SE = C::SLOT_STRIDE;

    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);    // full[s]: the bulk copies of stage s have landed
    unsigned* released = reinterpret_cast<unsigned*>(full + NS);   // released[s]: how many of the CTA's warps have finished reading stage s
    T* stages = reinterpret_cast<T*>(smem + 128);          // ring slot s at stages + s SE: the stage, then (right-edge tiles under
                                                           // TMA) the side buffer of the wrapped column at + STAGE_STRIDE

    // lane -> (lx, w): 8 vectors along x by 4 rows; the CTA's warps sit side by side along x.  A quarter-warp reads 128 contiguous bytes.
    const int lane = threadIdx.x & 31, wq = threadIdx.x >> 5;
    const int lx = lane & 7, w = lane >> 3;
    float* const ptile = reinterpret_cast<float*>(smem + 128 + C::RING_BYTES) + wq * C::PT_FLOATS;   // this warp's phase tile
    const int tiles_x = N / TX, tiles_y = N / TY;
    int bid = blockIdx.x;
    const int tx = bid % tiles_x;
    bid /= tiles_x;
    const int ty = bid % tiles_y, zc = bid / tiles_y;
    // z-chunk zc of nchunks: own planes [zc nz / nchunks, (zc + 1) nz / nchunks)
    const int x0 = tx * TX, y0 = ty * TY, z0 = (int)((long long)zc * zr.nz / nchunks);
    const int zlen = (int)((long long)(zc + 1) * zr.nz / nchunks) - z0;
    const int xi = wq * C::WX + V * lx;   // column of this thread's vector inside the tile

    const T* const src[5] = { f.phi_re, f.phi_im, f.th[0], f.th[1], f.th[2] };
    const P inv_dx2 = pk::splat((T)kd.inv_dx2), g_el = pk::splat((T)kd.gauge_norm), g_mag = pk::splat((T)(kd.gauge_norm * kd.inv_dx2));
    const P ncB = pk::splat(-(T)kd.cB), cE = pk::splat((T)kd.cE), third = pk::splat((T)(1.0 / 3.0));
    const P pot = pk::splat((T)kd.pot_coef), nsigma2 = pk::splat(-(T)kd.sigma2), grhs = pk::splat((T)kd.gauss_rhs);

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 1); released[s] = 0u; }
        mbar_fence_init();
    }
    __syncthreads();

    // plane index p of this CTA's march = own plane z0 + p (periodic in a whole lattice, the ghost above in a slab); planes 0 .. zlen are needed
    auto plane_of = [&](int p) { const int z = z0 + p; return ((zr.periodic && z >= N) ? z - N : z) + zr.zbase; };
    // One tensor copy per plane for tiles away from the periodic boundary.  Tiles on the right edge get the main box
    // (zero-filled out of bounds) plus a V-wide tensor copy of the wrapped column x = 0 .. V-1 into a side buffer, which the
    // readers of column TX use instead; tiles on the top edge in y (1 of N/TY tile rows) keep the row copies.
    const bool right_edge = x0 + TX == N;
    const bool tma_tile = use_tma && (y0 + TY < N);
    const bool wrapR = tma_tile && right_edge;
    // eps_1 of own plane z0 + p, rows y0-1 .. y0+TY-1: one tensor copy, except on the bottom tile row (the row below wraps)
    const bool e1_tma = use_tma && y0 > 0;
    auto issue_plane = [&](int s, int p) {
        const bool own = p < zlen;   // (plane zlen is only read as the +z neighbour: no momenta)
        mbar_arrive_expect_tx(&full[s], G::STAGE_BYTES + (wrapR ? (uint32_t)(5 * G::ROWS * V * sizeof(T)) : 0u) + (own ? C::E1_BYTES : 0u));
        if (own && e1_tma) {
            tma_load_4d(stages + s * SE + C::E1_OFF, &emap, x0, y0 - 1, zr.zbase + z0 + p, 0, &full[s]);
        } else if (own) {
            const T* pl = f.eps[1] + (size_t)(zr.zbase + z0 + p) * N * N + (size_t)x0;
#pragma unroll 1
            for (int r = 0; r <= TY; ++r) {
                const int y = (y0 + r == 0) ? N - 1 : y0 + r - 1;
                bulk_g2s(stages + s * SE + C::E1_OFF + r * TX, pl + (size_t)y * N, TX * sizeof(T), &full[s]);
            }
        }
        if (tma_tile) {
            tma_load_4d(stages + s * SE, &tmap, x0, y0, plane_of(p), 0, &full[s]);
            if (wrapR) tma_load_4d(stages + s * SE + C::STAGE_STRIDE, &wmap, 0, y0, plane_of(p), 0, &full[s]);
        } else {
            issue_rows<G, 5>(stages + s * SE, &full[s], src, N, x0, y0, plane_of(p));
        }
    };
    // element (array a, row w + dr) right of this thread's vector: column xi + V (= TX for the last vector of a row, which on a
    // right-edge tile under TMA reads the side buffer instead).  The offsets from the slot base are per-thread constants.
    const bool side = wrapR && xi + V == TX;
    auto edge_off = [&](int a, int r) { return side ? C::STAGE_STRIDE + (a * G::ROWS + r) * V : G::idx(a, r, xi + V); };
    const int eo_re = edge_off(0, w), eo_im = edge_off(1, w), eo_rey = edge_off(0, w + 1), eo_imy = edge_off(1, w + 1);
    const int eo_t1 = edge_off(3, w), eo_t2 = edge_off(4, w);
    if (wq == 0 && elect_one()) {
#pragma unroll
        for (int p = 0; p < NS; ++p)
            if (p <= zlen) issue_plane(p, p);
    }
    // The halo of this warp's region, two sites per lane: halo site e <= WX is (row TY, column e), the others (row e - WX - 1, column WX).
    // Offsets of phi_re of those sites inside a slot (phi_im is one array further) and where their phases go in the tile (-1: nothing).
    int hx_src[2], hx_im[2], hx_dst[2];
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        const int e = 2 * lane + j;
        const bool used = e < C::NEXTRA;
        const int r = !used ? 0 : (e <= C::WX ? TY : e - C::WX - 1), c = !used ? 0 : (e <= C::WX ? e : C::WX);
        const int col = wq * C::WX + c;   // column inside the CTA's tile (TX = the wrapped column of a right-edge tile)
        hx_src[j] = (wrapR && col == TX) ? C::STAGE_STRIDE + r * V : G::idx(0, r, col);
        hx_im[j] = (wrapR && col == TX) ? G::ROWS * V : G::ARR_ELEMS;
        hx_dst[j] = used ? r * C::PP + c : -1;
    }

    // arg phi / 2 pi of one plane at the V sites of this thread (p0), in the row above (p1) and right of the vector (pe = rows w, w+1).
    // fp32 lattices: every thread evaluates the phases of its own sites and of two sites of the warp's halo, the warp exchanges them through
    // its phase tile and the thread reads p1, pe back: 1.5 evaluations per site instead of the 2.5 of every thread for itself, and still
    // no exchange between warps -- the warps of a CTA drift freely and only meet at the stage ring's mbarriers.
    auto phases_of = [&](const T* st, float2 (&p0)[NP], float2 (&p1)[NP], float2& pe) {
        const VecT pr = lds_vec<T, V>(st + G::idx(0, w, xi)), pi = lds_vec<T, V>(st + G::idx(1, w, xi));
        if constexpr (!C::SHARE_PHASES) {   // fp64 lattices: every thread evaluates the ten phases it needs itself (measured faster there)
            const VecT pry = lds_vec<T, V>(st + G::idx(0, w + 1, xi)), piy = lds_vec<T, V>(st + G::idx(1, w + 1, xi));
#pragma unroll
            for (int h = 0; h < NP; ++h) {
                p0[h] = atan2_turns(to_float2(pk::at<T, V>(pi.v, h)), to_float2(pk::at<T, V>(pr.v, h)));
                p1[h] = atan2_turns(to_float2(pk::at<T, V>(piy.v, h)), to_float2(pk::at<T, V>(pry.v, h)));
            }
            pe = atan2_turns(make_float2((float)st[eo_im], (float)st[eo_imy]), make_float2((float)st[eo_re], (float)st[eo_rey]));
            return;
        }
        __syncwarp();   // every lane has read the previous plane's phases before anyone overwrites the tile
#pragma unroll
        for (int h = 0; h < NP; ++h) {
            p0[h] = atan2_turns(to_float2(pk::at<T, V>(pi.v, h)), to_float2(pk::at<T, V>(pr.v, h)));
            *reinterpret_cast<float2*>(ptile + w * C::PP + V * lx + 2 * h) = p0[h];
        }
        const float2 hx = atan2_turns(make_float2((float)st[hx_src[0] + hx_im[0]], (float)st[hx_src[1] + hx_im[1]]),
                                      make_float2((float)st[hx_src[0]], (float)st[hx_src[1]]));
        if (hx_dst[0] >= 0) ptile[hx_dst[0]] = hx.x;
        if (hx_dst[1] >= 0) ptile[hx_dst[1]] = hx.y;
        __syncwarp();
        const float* up = ptile + (w + 1) * C::PP + V * lx;
#pragma unroll
        for (int h = 0; h < NP; ++h) p1[h] = *reinterpret_cast<const float2*>(up + 2 * h);
        pe = make_float2(ptile[w * C::PP + V * lx + V], up[V]);
    };
    // the pair of phases one site to the right of pair h: (p[2h+1], p[2h+2]), the last one being the edge phase
    auto shifted = [&](const float2 (&p)[NP], int h, float e) { return make_float2(p[h].y, h + 1 < NP ? p[h + 1 < NP ? h + 1 : h].x : e); };

    mbar_wait(&full[0], 0);
    // phases of the current plane and n_0, n_1 of its links (own sites; n_1 also right of the vector), carried along
    // the march together with the margins of those link numbers
    float2 a[NP], ay[NP], ae, n0c[NP], n1c[NP];
    float n1c_e, rmax_c = 0.0f, tmax_c = 0.0f;
    phases_of(stages, a, ay, ae);
    {
        const VecT t0 = lds_vec<T, V>(stages + G::idx(2, w, xi)), t1 = lds_vec<T, V>(stages + G::idx(3, w, xi));
        float dummy = 0.0f;
#pragma unroll
        for (int h = 0; h < NP; ++h) {
            n1c[h] = link_numbers(a[h], ay[h], to_float2(pk::at<T, V>(t1.v, h)), rmax_c, rmax_c, tmax_c);
            n0c[h] = link_numbers(a[h], shifted(a, h, ae.x), to_float2(pk::at<T, V>(t0.v, h)), rmax_c, rmax_c, tmax_c);
        }
        const float th_e = (float)stages[eo_t1];
        n1c_e = link_numbers(make_float2(ae.x, ae.x), make_float2(ae.y, ae.y), make_float2(th_e, th_e), rmax_c, dummy, tmax_c).x;
    }

    // The momenta (no halo) come straight from global memory: g = element offset of this thread's vector in plane z0 + it, a
    // running offset; the site left of the vector (eps_0^{x-k_0}; wrapped for the first vector of the lattice) sits at a fixed distance.
    const size_t plane_stride = (size_t)N * N;
    size_t g = ((size_t)(zr.zbase + z0) * N + (size_t)(y0 + w)) * N + (size_t)(x0 + xi);
    const ptrdiff_t d_site_left = (x0 + xi == 0) ? (ptrdiff_t)(N - 1) : -(ptrdiff_t)1;
    // eps_2 of the plane below, carried in registers along the march
    VecT E2m = ldg_vec<T, V>(f.eps[2] + ((zr.periodic && z0 == 0) ? g + (size_t)(N - 1) * plane_stride : g - plane_stride));   // (slab: the ghost below)

    double num = 0.0, den = 0.0, lsum = 0.0, rhs2 = 0.0, vnum = 0.0, vden = 0.0, wnum = 0.0, wden = 0.0;
    float pierced_f = 0.0f;   // plaquettes with W != 0 on the fast path (all |W| <= 1 there, so this is sum |W| as well); exact below 2^24
    unsigned nonfinite = 0u;
    T gmax_t = T(0);

    const T* sc = stages;             // slot of plane it (walks the ring with running pointers: no index arithmetic per plane)
    int ring = 0;                     // it % NS
    for (int it = 0; it < zlen; ++it) {
        const int ring_n = ring + 1 == NS ? 0 : ring + 1;
        const T* sn = ring_n ? sc + SE : stages;

        const VecT Pr = ldg_vec<T, V>(f.pi_re + g), Pi = ldg_vec<T, V>(f.pi_im + g);
        const VecT E0 = ldg_vec<T, V>(f.eps[0] + g), E2 = ldg_vec<T, V>(f.eps[2] + g);
        // eps_0 of the site left of the vector: its own scalar load (the line is in flight for the neighbouring lane's vector anyway);
        // a shuffle of E0 would tie the first use of the streamed loads to the top of the plane
        const T e0_left = __ldg(f.eps[0] + (g + d_site_left));

        mbar_wait(&full[ring_n], ((it + 1) / NS) & 1);
        float2 az[NP], azy[NP], aze;
        phases_of(sn, az, azy, aze);

        const VecT pr = lds_vec<T, V>(sc + G::idx(0, w, xi)), pi = lds_vec<T, V>(sc + G::idx(1, w, xi));
        const VecT t0 = lds_vec<T, V>(sc + G::idx(2, w, xi)), t1 = lds_vec<T, V>(sc + G::idx(3, w, xi)), t2 = lds_vec<T, V>(sc + G::idx(4, w, xi));
        const VecT pry = lds_vec<T, V>(sc + G::idx(0, w + 1, xi)), piy = lds_vec<T, V>(sc + G::idx(1, w + 1, xi));
        const VecT t0y = lds_vec<T, V>(sc + G::idx(2, w + 1, xi)), t2y = lds_vec<T, V>(sc + G::idx(4, w + 1, xi));
        const VecT prz = lds_vec<T, V>(sn + G::idx(0, w, xi)), piz = lds_vec<T, V>(sn + G::idx(1, w, xi));
        const VecT t0z = lds_vec<T, V>(sn + G::idx(2, w, xi)), t1z = lds_vec<T, V>(sn + G::idx(3, w, xi));
        const T prx_e = sc[eo_re], pix_e = sc[eo_im];
        const T t1x_e = sc[eo_t1], t2x_e = sc[eo_t2];
        const VecT E1 = lds_vec<T, V>(sc + C::E1_OFF + (w + 1) * TX + xi), E1m = lds_vec<T, V>(sc + C::E1_OFF + w * TX + xi);   // eps_1 here and one row below

        // ---- winding (Eq. 11), fast path: the link numbers this thread-plane needs.  n_0, n_1 of this plane were formed
        //      one iteration ago (as the +z links); n_1, n_2 are also taken at the site right of the vector (n_j^{x+k_0}).
        float rmax = rmax_c, tmax = tmax_c;                  // margins of the carried n0c, n1c
        float2 n2[NP], n0y[NP], n2y[NP], n0z[NP], n1z[NP];
        rmax_c = 0.0f;
        tmax_c = 0.0f;
#pragma unroll
        for (int h = 0; h < NP; ++h) {
            n2[h] = link_numbers(a[h], az[h], to_float2(pk::at<T, V>(t2.v, h)), rmax, rmax, tmax);
            n2y[h] = link_numbers(ay[h], azy[h], to_float2(pk::at<T, V>(t2y.v, h)), rmax, rmax, tmax);
            n0y[h] = link_numbers(ay[h], shifted(ay, h, ae.y), to_float2(pk::at<T, V>(t0y.v, h)), rmax, rmax, tmax);
            n1z[h] = link_numbers(az[h], azy[h], to_float2(pk::at<T, V>(t1z.v, h)), rmax_c, rmax_c, tmax_c);
            n0z[h] = link_numbers(az[h], shifted(az, h, aze.x), to_float2(pk::at<T, V>(t0z.v, h)), rmax_c, rmax_c, tmax_c);
        }
        // right of the vector: (n_2 of this plane, n_1 of the next) in one packed evaluation
        float tmax_e = 0.0f;
        const float2 ne = link_numbers(make_float2(ae.x, aze.x), make_float2(aze.x, aze.y), make_float2((float)t2x_e, (float)sn[eo_t1]),
                                       rmax, rmax_c, tmax_e);
        tmax = fmaxf(tmax, tmax_e);
        tmax_c = fmaxf(tmax_c, tmax_e);
        float2 sabs = pk::splat(0.0f), ssq = pk::splat(0.0f);   // small integers: exact in fp32
#pragma unroll
        for (int h = 0; h < NP; ++h) {
            const float2 n1x = make_float2(n1c[h].y, h + 1 < NP ? n1c[h + 1 < NP ? h + 1 : h].x : n1c_e);   // n_1^{x+k_0}
            const float2 n2x = make_float2(n2[h].y, h + 1 < NP ? n2[h + 1 < NP ? h + 1 : h].x : ne.x);      // n_2^{x+k_0}
            const float2 W01 = pk::sub(pk::add(n0c[h], n1x), pk::add(n0y[h], n1c[h]));   // -W_ij
            const float2 W02 = pk::sub(pk::add(n0c[h], n2x), pk::add(n0z[h], n2[h]));
            const float2 W12 = pk::sub(pk::add(n1c[h], n2y[h]), pk::add(n1z[h], n2[h]));
            sabs = pk::add(pk::add(sabs, pk::absv(W01)), pk::add(pk::absv(W02), pk::absv(W12)));
            ssq = pk::fma(W01, W01, pk::fma(W02, W02, pk::fma(W12, W12, ssq)));
        }
        {
            const float cnt = sabs.x + sabs.y;
            // sure: every link is far from a tie and every |W| <= 1 (integers: sum W^2 == sum |W|); NaN fails both
            // (n_0, n_1 of the next plane enter this plane's W_02, W_12 as the +z links: their margins count here too)
            const bool sure = (fmaxf(rmax, rmax_c) < 0.5f - kTieMargin * (1.0f + fmaxf(tmax, tmax_c))) && (ssq.x + ssq.y == cnt);
            if (!sure) {   // fp64 decides (diag_resolve_kernel)
                const unsigned long long e = atomicAdd(doubt_count, 1ull);
                doubt_list[e] = (unsigned)((x0 + xi) / V) | ((unsigned)(y0 + w) << 10) | ((unsigned)(zr.zbase + z0 + it) << 21);   // N <= 2048, local plane index
            }
            pierced_f += sure ? cnt : 0.0f;
        }
#pragma unroll
        for (int h = 0; h < NP; ++h) { n0c[h] = n0z[h]; n1c[h] = n1z[h]; a[h] = az[h]; ay[h] = azy[h]; }
        n1c_e = ne.y;
        ae = aze;

        // ---- Eq. 2 pieces, <v^2> sums and the Gauss residual, two sites at a time --------------------------------------------
        P p_num = pk::splat(T(0)), p_den = p_num, p_l = p_num, p_r2 = p_num, p_vn = p_num, p_vd = p_num, p_wn = p_num, p_wd = p_num;   // per thread and plane, then into the fp64 sums
#pragma unroll
        for (int h = 0; h < NP; ++h) {
            const P phr = pk::at<T, V>(pr.v, h), phi = pk::at<T, V>(pi.v, h), pmr = pk::at<T, V>(Pr.v, h), pmi = pk::at<T, V>(Pi.v, h);
            const P th0 = pk::at<T, V>(t0.v, h), th1 = pk::at<T, V>(t1.v, h), th2 = pk::at<T, V>(t2.v, h);
            const P ep0 = pk::at<T, V>(E0.v, h), ep1 = pk::at<T, V>(E1.v, h), ep2 = pk::at<T, V>(E2.v, h);
            P s0, c0, s1, c1, s2, c2;
            SumsTrig<TRIG>::link_phase(th0, s0, c0);
            SumsTrig<TRIG>::link_phase(th1, s1, c1);
            SumsTrig<TRIG>::link_phase(th2, s2, c2);
            // forward hops U_j phi^{x+k_j} - phi^x, U = cos - i sin:  (c re + s im, c im - s re)
            const P nxr = pk::next<T, V>(pr.v, h, prx_e), nxi = pk::next<T, V>(pi.v, h, pix_e);
            const P d0r = pk::sub(pk::fma(c0, nxr, pk::mul(s0, nxi)), phr), d0i = pk::sub(pk::fma(pk::neg(s0), nxr, pk::mul(c0, nxi)), phi);
            const P nyr = pk::at<T, V>(pry.v, h), nyi = pk::at<T, V>(piy.v, h);
            const P d1r = pk::sub(pk::fma(c1, nyr, pk::mul(s1, nyi)), phr), d1i = pk::sub(pk::fma(pk::neg(s1), nyr, pk::mul(c1, nyi)), phi);
            const P nzr = pk::at<T, V>(prz.v, h), nzi = pk::at<T, V>(piz.v, h);
            const P d2r = pk::sub(pk::fma(c2, nzr, pk::mul(s2, nzi)), phr), d2i = pk::sub(pk::fma(pk::neg(s2), nzr, pk::mul(c2, nzi)), phi);
            P Gd = pk::fma(d0r, d0r, pk::mul(d0i, d0i));
            Gd = pk::fma(d1r, d1r, pk::fma(d1i, d1i, Gd));
            Gd = pk::fma(d2r, d2r, pk::fma(d2i, d2i, Gd));
            Gd = pk::mul(Gd, inv_dx2);
            const P K = pk::fma(pmr, pmr, pk::mul(pmi, pmi));
            const P dm = pk::fma(phr, phr, pk::fma(phi, phi, nsigma2));
            const P Vp = pk::mul(pot, pk::mul(dm, dm));
            const P X01 = pk::sub(pk::add(th0, pk::next<T, V>(t1.v, h, t1x_e)), pk::add(pk::at<T, V>(t0y.v, h), th1));
            const P X02 = pk::sub(pk::add(th0, pk::next<T, V>(t2.v, h, t2x_e)), pk::add(pk::at<T, V>(t0z.v, h), th2));
            const P X12 = pk::sub(pk::add(th1, pk::at<T, V>(t2y.v, h)), pk::add(pk::at<T, V>(t1z.v, h), th2));
            const P mag = SumsTrig<TRIG>::plaquettes(X01, X02, X12);
            const P e2 = pk::fma(ep0, ep0, pk::fma(ep1, ep1, pk::mul(ep2, ep2)));
            const P El = pk::mul(g_el, e2), Bm = pk::mul(g_mag, mag);   // electric / magnetic energy densities
            const P lag = pk::sub(pk::sub(pk::fma(cE, El, pk::fma(ncB, Bm, K)), Gd), Vp);
            p_num = pk::fma(K, lag, p_num);
            p_den = pk::fma(Gd, lag, p_den);
            p_l = pk::add(p_l, lag);
            p_vn = pk::fma(K, Vp, p_vn);   // potential-weighted estimator <v^2>_V (L86)
            p_vd = pk::fma(Gd, Vp, p_vd);
            // equation of state (Eq. 12): rho = K + G + Vp + El + Bm, p = K - G/3 - Vp + (El + Bm)/3, Lagrangian weighted
            const P EB = pk::add(El, Bm);
            p_wn = pk::fma(pk::fma(pk::sub(EB, Gd), third, pk::sub(K, Vp)), lag, p_wn);
            p_wd = pk::fma(pk::add(pk::add(K, Gd), pk::add(Vp, EB)), lag, p_wd);

            // ---- Gauss residual: sum_i (eps_i^x - eps_i^{x-k_i}) - gauss_rhs Im[conj(phi) Pi] ----------------------------------
            const P e0m = pk::mk(h > 0 ? E0.v[h > 0 ? 2 * h - 1 : 0] : e0_left, E0.v[2 * h]);
            const P div = pk::add(pk::add(pk::sub(ep0, e0m), pk::sub(ep1, pk::at<T, V>(E1m.v, h))), pk::sub(ep2, pk::at<T, V>(E2m.v, h)));
            const P rhs = pk::mul(grhs, pk::fma(phr, pmi, pk::neg(pk::mul(phi, pmr))));
            const P gabs = pk::absv(pk::sub(div, rhs));
            const T g2 = gabs.x > gabs.y ? gabs.x : gabs.y;
            gmax_t = g2 > gmax_t ? g2 : gmax_t;   // (a NaN residual is reported through `nonfinite`)
            p_r2 = pk::fma(rhs, rhs, p_r2);
        }
        const T l_plane = p_l.x + p_l.y;
        num += (double)(p_num.x + p_num.y); den += (double)(p_den.x + p_den.y); lsum += (double)l_plane; rhs2 += (double)(p_r2.x + p_r2.y);
        vnum += (double)(p_vn.x + p_vn.y); vden += (double)(p_vd.x + p_vd.y);
        wnum += (double)(p_wn.x + p_wn.y); wden += (double)(p_wd.x + p_wd.y);
        // Non-finite values.  Every one of the ten stored values feeds the Lagrangian (NaN or Inf in, NaN or Inf out), so a
        // finite plane sum clears all of them at once; otherwise the stored values themselves are examined (a finite value
        // whose square overflows the storage type is not an error: include/ahs.h "nonfinite").
        if (!finite_t(l_plane)) {
            bool bad = false;
#pragma unroll
            for (int v = 0; v < V; ++v)
                bad = bad || !finite_t(pr.v[v]) || !finite_t(pi.v[v]) || !finite_t(Pr.v[v]) || !finite_t(Pi.v[v]) || !finite_t(t0.v[v]) ||
                      !finite_t(t1.v[v]) || !finite_t(t2.v[v]) || !finite_t(E0.v[v]) || !finite_t(E1.v[v]) || !finite_t(E2.v[v]);
            // (the forward neighbours that also feed this plane's sum are the own sites of other threads)
            nonfinite += bad ? 1u : 0u;
        }
        E2m = E2;
        // This warp is done with stage `ring` (plane it).  The LAST of the CTA's warps to say so re-fills it with plane it + NS: nobody
        // ever waits for a stage to become free.  (An earlier version let a rotating warp spin on an `empty` mbarrier before issuing:
        // its elected lane and its 31 siblings then ran the rest of the plane as two groups, every instruction issued twice, and a
        // __syncwarp() there made the whole warp wait instead -- profiles/r4_diag1024_f32_full.md.)  The acq_rel counter orders all
        // warps' reads of the stage before the last one's fence.proxy.async and copy.
        __syncwarp();
        if (lane == 0) {
            unsigned before;
            asm volatile("atom.acq_rel.cta.shared::cta.add.u32 %0, [%1], 1;" : "=r"(before) : "r"(smem_u32(&released[ring])) : "memory");
            if (before == C::NWARPS - 1) {
                released[ring] = 0u;
                if (it + NS <= zlen) {
                    fence_proxy_async();
                    issue_plane(ring, it + NS);
                }
            }
        }
        sc = sn;
        ring = ring_n;
        g += plane_stride;
    }

    const unsigned long long n_fast = (unsigned long long)pierced_f;
    DiagPartial acc = { n_fast, n_fast, num, den, lsum, (double)gmax_t, rhs2, (unsigned long long)nonfinite, vnum, vden, wnum, wden };
    block_reduce_store(acc, partials + blockIdx.x);
}

// z-chunks per tile, measured (profiles/r4_chunks.md; see pick_chunks of the step march): 32 up to 512^3, 16 beyond and for
// fp64 lattices; halved until the partial records fit and the count divides N.
template <typename T>
int pick_chunks(int N, int nz, long tiles, int max_partials)
{
    int c = (sizeof(T) == 4 && N <= 512) ? 32 : 16;
    while (c > 1 && (N % c != 0 || N / c < 4 || tiles * c + 2 > max_partials)) c /= 2;
    const int zlen = N / c;                 // planes per chunk, read off the whole lattice; a slab of nz planes gets nz / zlen chunks
    return nz >= zlen ? nz / zlen : 1;
}

}  // namespace

template <typename T>
int launch_diag_march(const DiagPtrs<T>& f, int N, const ZRange& zr, const DiagCoef& c, DiagPartial* partials, int max_partials, DiagPartial* result,
                      void* list, size_t list_bytes, const DiagMaps* tmap, const MarchOptions& opt, cudaStream_t st)
{
    using C = DiagCfg<T>;
    if (!march_supported<T>(N) || zr.nz < 1) return AHS_ERR_INVALID_ARG;
    // a doubt-list entry keeps the LOCAL plane index in its top 11 bits: the last own plane must be <= 2047 (a whole 2048^3 lattice
    // is; a single slab of 2048 planes with its ghost plane below is not -- ahs_group_create refuses it)
    if (zr.zbase + zr.nz > 2048) return AHS_ERR_INVALID_ARG;
    // fp64 lattices always take the polynomials (the hardware unit is an fp32 one)
    const bool hw = sizeof(T) == 4 && opt.diag_trig == AHS_TRIG_HARDWARE;
    auto kern = hw ? diag_march_kernel<T, sizeof(T) == 4 ? AHS_TRIG_HARDWARE : AHS_TRIG_POLYNOMIAL> : diag_march_kernel<T, AHS_TRIG_POLYNOMIAL>;
    static SmemAttribute attr[2];   // per device and instantiation
    if (!attr[hw].ensure(kern, C::SMEM)) return AHS_ERR_CUDA;
    const long tiles = (long)(N / C::TX) * (N / C::TY);
    int nchunks = pick_chunks<T>(N, zr.nz, tiles, max_partials);
    if (opt.diag_chunks > 0 && opt.diag_chunks <= zr.nz && tiles * opt.diag_chunks + 2 <= max_partials) nchunks = opt.diag_chunks;
    const long blocks = tiles * nchunks;
    // partials[blocks] collects the second pass, partials[blocks + 1].n_pierced is the length of the doubt list
    if (blocks + 2 > max_partials || list_bytes < sizeof(unsigned) * ((size_t)N * N * zr.nz / C::V)) return AHS_ERR_INVALID_ARG;
    DiagPartial* extra = partials + blocks;
    unsigned long long* count = &partials[blocks + 1].n_pierced;
    if (cudaMemsetAsync(extra, 0, 2 * sizeof(DiagPartial), st) != cudaSuccess) return AHS_ERR_CUDA;
    DiagMaps none;
    memset(&none, 0, sizeof(none));
    const bool use_tma = tmap && opt.staging == AHS_STAGING_TENSOR;
    const DiagMaps& mp = use_tma ? *tmap : none;
    kern<<<(unsigned)blocks, C::NTHREADS, C::SMEM, st>>>(f, N, zr, nchunks, c, partials, (unsigned*)list, count, mp.tile, mp.wrap, mp.eps1, use_tma ? 1 : 0);
    if (cudaGetLastError() != cudaSuccess) return AHS_ERR_CUDA;
    diag_resolve_kernel<T><<<148 * 8, 128, 0, st>>>(f, N, zr.periodic, (const unsigned*)list, count, extra);
    if (cudaGetLastError() != cudaSuccess) return AHS_ERR_CUDA;
    const int r = launch_diag_finish(partials, (int)blocks + 1, result, st);
    return r < 0 ? r : 3;
}

// the tensor maps of one (phi, theta) buffer for the tile shape above: box (TX + V, TY + 1, 1, 5), and of eps_1: box (TX, TY + 1, 1, 1)
template <typename T>
bool make_diag_march_map(DiagMaps* out, const void* phi_re_base, const void* eps1_base, int N, int nz_alloc, size_t array_bytes)
{
    using G = typename DiagCfg<T>::G;
    if (!march_supported<T>(N)) return false;
    return make_tile_map<T>(&out->tile, phi_re_base, N, nz_alloc, array_bytes, 5, G::PITCH, G::ROWS, 5) &&
           make_tile_map<T>(&out->wrap, phi_re_base, N, nz_alloc, array_bytes, 5, G::V, G::ROWS, 5) &&
           make_tile_map<T>(&out->eps1, eps1_base, N, nz_alloc, array_bytes, 1, G::TX, G::TY + 1, 1);
}
template bool make_diag_march_map<float>(DiagMaps*, const void*, const void*, int, int, size_t);
template bool make_diag_march_map<double>(DiagMaps*, const void*, const void*, int, int, size_t);

template int launch_diag_march<float>(const DiagPtrs<float>&, int, const ZRange&, const DiagCoef&, DiagPartial*, int, DiagPartial*, void*, size_t, const DiagMaps*, const MarchOptions&, cudaStream_t);
template int launch_diag_march<double>(const DiagPtrs<double>&, int, const ZRange&, const DiagCoef&, DiagPartial*, int, DiagPartial*, void*, size_t, const DiagMaps*, const MarchOptions&, cudaStream_t);

}  // namespace ahs
