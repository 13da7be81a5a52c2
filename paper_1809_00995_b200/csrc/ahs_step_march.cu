// ahs_step_march.cu -- the fused leapfrog step (Eqs. 4-7) as a 2.5D z-march for sm_100a.
//
// One CTA owns a tile of TX x TY sites in (x, y) (TX = 32 lanes x one 16-byte vector, TY rows = TY warps) and
// marches over `zlen` planes.  The level-n fields of the planes ahead are streamed into rings of halo'd shared-memory
// tiles that complete on mbarriers while planes k, k+1 are in use: phi_re, phi_im, theta_0, theta_1 in an NS-stage ring
// (float 3, double 4), theta_2 in a ring of its own (StepShape::T2_RING).  A tile that does not touch the periodic
// boundary in y is fetched by tensor-map TMA (cp.async.bulk.tensor, UTMALDG: one copy for the four-array stage, one for
// theta_2, plus a V-wide copy of the wrapped halo column for x-edge tiles); tiles on the y boundary, lattices one tile
// wide and AHS_STAGING_ROWS use one bulk copy per tile row (cp.async.bulk, UBLKCP; ahs_stage.cuh).  The issuing warp
// rotates.  Pi and eps (no halo) are read with streaming 16-byte loads and all ten outputs leave as 16-byte stores.
//
// Compute-once form.  Each site owner computes, from raw phi, theta of the site and of its FORWARD neighbours only,
//   U_j = exp(-i theta_j)                         3 sincos       (link phases, Eq. 3 / L46-51, q = +1)
//   f_j = U_j phi^{x+k_j}, b_j = conj(U_j) phi^x, J_j = Im[conj(phi^x) f_j]
//   S_01, S_02, S_12 = sin Xi_ij^x                3 sin          (plaquettes based at x, Eq. 3)
// and receives the six products owned by its BACKWARD neighbours:
//   -x : b_0, S_01, S_02   from the thread's previous vector element, else from lane-1 by warp shuffle, else
//                          (lane 0) from the halo column x0-1 through shared memory
//   -y : b_1, S_01, S_12   through a shared-memory exchange row (row -1 = halo row)
//   -z : b_2, S_02, S_12   in the thread's own registers from the previous plane of the march.
// The products of the halo row y0-1 and of the halo column x0-1 are recomputed inside the CTA, one site per lane,
// by warps that take the job in rotation (same function, same inputs => bit-identical link phases on both sides of a tile edge, which is what keeps the Gauss
// law at roundoff: it needs the same U in Eq. 4 and Eq. 5, R4).  Then
//   Lap    = sum_j (f_j + b_j^{x-k_j}) - 6 phi                                              (Eq. 4)
//   curl_0 = (S01 - S01^{-y}) + (S02 - S02^{-z}),  curl_1 = (S01^{-x} - S01) + (S12 - S12^{-z}),
//   curl_2 = (S02^{-x} - S02) + (S12^{-y} - S12)                                            (Eq. 5)
// followed by the kicks and the drift into the other (phi, theta) buffer (Eqs. 6-7).
//
// One exchange point per plane, and it is an mbarrier (`xch`, one phase per plane, every thread arrives), not a
// __syncthreads: a thread ARRIVES as soon as its exchange-row / halo-column stores and its stage reads have been issued and
// WAITS only where it needs the other warps' products, so the trigonometry of the in-plane links sits between the two.
// Phase 1 (before the wait) does all the trigonometry and folds every term that the thread owns -- including the -x terms
// obtained by shuffle and the -z terms carried in registers -- into partial results (q = Pi' without the -y / halo hops,
// phi + dt q, eps' and theta + dt eps' without the -y / halo sines).  Phase 2 (after the wait) adds the few terms that
// crossed a warp boundary and stores.  The exchange rows are double-buffered by plane parity so that the phase of plane
// k+1 also orders "everyone has read plane k's exchange" before it is overwritten at plane k+2; the same phase tells the
// issuing warp that a stage slot has been read by all and may be re-filled.
// The paper's kernels stage raw fields per kernel and recompute every phase (L107-109); this is a different design.
#include <cstring>

#include "ahs_internal.cuh"
#include "ahs_math.cuh"
#include "ahs_stage.cuh"
#include "ahs_tma.cuh"
#include "ahs_trig.cuh"

namespace ahs {

namespace {

template <typename T> struct StepCoefT { T c1, c2, c3, d1, d2, d3, dt, sigma2; };

// Launch shape per storage type: rows per tile (= warps per CTA), CTAs per SM the register budget is cut for, ring depth.
//   float : 4 rows, 3 CTAs/SM (register budget 65536 / (3 x 128) = 170, i.e. at most 168; ptxas uses 160 in the build that ships,
//           profiles/r6_sass_histogram.md), 3 stages -- measured fastest (profiles/r6_step1024_f32_full.md)
//   double: 4 rows, 2 CTAs/SM (255 registers: at 168 the kernel spills ~100 B per thread and plane and waits on the reloads,
//           profiles/r4_step512_f64_full.md), 4 stages (two CTAs leave room for a deeper ring)
template <typename T> struct StepShape;
//   LATE_WAIT: wait for the next plane's stage behind the in-plane trigonometry (float: -2 % under the power cap; double: no gain)
//   T2_RING  : slots of the theta_2 ring.  NS - 1 (theta_2 is never read one plane ahead) with a barrier of its own keeps the float kernel at
//              63.9 KB per CTA, inside the SM's 196 KB shared-memory configuration (profiles/r6_step1024_f32_full.md); the double kernel, two CTAs
//              per SM, has room for NS slots, theta_2 then rides on its plane's stage barrier one plane earlier (4.69 -> 4.62 ms at 512^3)
template <> struct StepShape<float> { static constexpr int TY = 4, MINB = 3, NS = 3, T2_RING = 2; static constexpr bool LATE_WAIT = true; };
template <> struct StepShape<double> { static constexpr int TY = 4, MINB = 2, NS = 4, T2_RING = 4; static constexpr bool LATE_WAIT = false; };

template <typename T, int TY_, int NS_>
struct MarchCfg {
    static constexpr int V = 16 / sizeof(T);
    static constexpr int TY = TY_;
    static constexpr int NSTAGE = NS_;                       // plane it + NSTAGE - 1 is in flight while planes it, it + 1 are read
    using G = TileGeom<T, V, TY, 4, NSTAGE>;                // a stage: phi_re, phi_im, theta_0, theta_1 of one plane
    static constexpr int T2_SLOTS = StepShape<T>::T2_RING;   // NSTAGE - 1 (own barriers) or NSTAGE (theta_2 rides on its plane's stage barrier)
    static constexpr bool T2_OWN = T2_SLOTS < NSTAGE;
    static_assert(T2_SLOTS == NSTAGE || T2_SLOTS == NSTAGE - 1, "theta_2 ring");
    static constexpr int TX = G::TX;
    static constexpr int NTHREADS = TY * 32;
    static constexpr int YEX_ELEMS = 4 * TY * TX;         // b1.re, b1.im, S01, S12 of rows -1 .. TY-2 (one parity)
    static constexpr int XEX_ELEMS = 4 * TY;              // b0.re, b0.im, S01, S02 of the halo column (one parity)
    static constexpr int T2_STRIDE = (int)(((G::ARR_BYTES + 127u) & ~127u) / sizeof(T));   // tensor copies land 128-byte aligned
    static_assert(G::STAGE_BYTES % 128 == 0, "stages stay 128-byte aligned");
    // x-edge tiles under TMA: the wrapped halo column (V wide) of a plane lands in a side buffer, one tensor copy each
    static constexpr int WRAP_ELEMS = (int)(((4 * G::ROWS * V * sizeof(T) + 127) & ~(size_t)127) / sizeof(T));   // phi_re, phi_im, theta_0, theta_1
    static constexpr int WRAP2_STRIDE = (int)(((G::ROWS * V * sizeof(T) + 127) & ~(size_t)127) / sizeof(T));   // theta_2
    static constexpr size_t SMEM = 128 + sizeof(T) * (size_t)(NSTAGE * G::STAGE_ELEMS + T2_SLOTS * T2_STRIDE + NSTAGE * WRAP_ELEMS +
                                                              T2_SLOTS * WRAP2_STRIDE + 2 * YEX_ELEMS + 2 * XEX_ELEMS);
};

template <typename T, int TY, int MINB, int NSTG>
__global__ void __launch_bounds__(MarchCfg<T, TY, NSTG>::NTHREADS, MINB)
step_march_kernel(FieldPtrs<T> f, GhostPtrs<T> gh, int N, ZRange zr, int nchunks, StepCoefT<T> k, const __grid_constant__ CUtensorMap map_stage,
                  const __grid_constant__ CUtensorMap map_th2, const __grid_constant__ CUtensorMap map_wstage,
                  const __grid_constant__ CUtensorMap map_wth2, int use_tma)
{
    using C = MarchCfg<T, TY, NSTG>;
    using G = typename C::G;
    using VecT = Vec<T, C::V>;
    constexpr int V = C::V, TX = C::TX, NS = C::NSTAGE, SE = G::STAGE_ELEMS, T2S = C::T2_SLOTS;
    // rotation of the side jobs over the warps at plane `it` (by (w + it) % ...): the halo row takes TX/32 = V warps
    constexpr int HSTRIDE = TY / V, COLUMN = 1 % TY, ISSUER = 3 % TY;
    static_assert(TY % V == 0, "the halo row is shared out over V warps");

    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem);
    uint64_t* xch = full + NS;   // exchange barrier: one phase per plane, every thread arrives
    uint64_t* t2full = xch + 1;  // t2full[slot]: theta_2 of a plane has landed in its ring slot (its own barriers: theta_2 of the CURRENT plane
                                 // is needed at the top of the plane, the stage of the NEXT plane only half-way through it)
    T* stages = reinterpret_cast<T*>(smem + 128);
    T* th2ring = stages + NS * SE;
    T* wrapS = th2ring + C::T2_SLOTS * C::T2_STRIDE;      // side buffers of the wrapped halo column (x-edge tiles under TMA)
    T* wrapT = wrapS + NS * C::WRAP_ELEMS;
    T* yex = wrapT + C::T2_SLOTS * C::WRAP2_STRIDE;
    T* xex = yex + 2 * C::YEX_ELEMS;

    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int tiles_x = N / TX, tiles_y = N / TY;
    int bid = blockIdx.x;
    const int tx = bid % tiles_x;
    bid /= tiles_x;
    const int ty = bid % tiles_y, zc = bid / tiles_y;
    // z-chunk zc of nchunks: own planes [zc nz / nchunks, (zc + 1) nz / nchunks) -- the chunks need not be of equal length
    const int x0 = tx * TX, y0 = ty * TY, z0 = (int)((long long)zc * zr.nz / nchunks);
    const int zlen = (int)((long long)(zc + 1) * zr.nz / nchunks) - z0;
    const int xi = V * lane;

    const T* const src[4] = { f.phi_re, f.phi_im, f.th[0], f.th[1] };
    const T* const src2[1] = { f.th[2] };

    if (threadIdx.x == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
#pragma unroll
        for (int s = 0; s < C::T2_SLOTS; ++s) mbar_init(&t2full[s], 1);
        mbar_init(xch, C::NTHREADS);
        mbar_fence_init();
    }
    __syncthreads();
    // Programmatic dependent launch (AHS_OPT_STEP_PDL): everything above -- the CTA's index arithmetic and barrier initialisation -- may
    // run while the previous kernel of the stream is still draining its last wave.  From here on the kernel touches global memory
    // (the previous step's output is this step's input, and this step overwrites the previous step's input): wait until that kernel
    // has completed and its stores are visible.  The trigger lets the NEXT launch's CTAs take the SM slots this grid no longer needs
    // once every CTA of this grid has started; they stop at this same wait.  Both are no-ops in a launch without the attribute.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");

    // plane index i of this CTA's march = own plane z0 - 1 + i: periodic inside a whole lattice, running into the ghost planes of a slab
    auto plane_of = [&](int i) {
        int z = z0 - 1 + i;
        if (zr.periodic) z = z < 0 ? z + N : (z >= N ? z - N : z);
        return z + zr.zbase;
    };
    // Tiles that do not touch the periodic boundary fetch a plane with two tensor copies (UTMALDG: the four-array stage
    // and theta_2) instead of 30 row copies; the others keep the row copies (TMA zero-fills out of bounds, it does not wrap).
    // x-edge tiles: the main box runs out of bounds on one side (zero-filled) and the wrapped halo column (x = N-V.. for the
    // left edge, x = 0.. for the right edge) arrives by a second, V-wide tensor copy in a side buffer, which the few readers of
    // that column use instead.  y-edge tiles (2 of N/TY tile rows) and lattices one tile wide keep the row copies.
    const bool left_edge = x0 == 0, right_edge = x0 + TX == N;
    const bool tma_tile = use_tma && y0 > 0 && y0 + TY < N && !(left_edge && right_edge);
    const bool wrapL = tma_tile && left_edge, wrapR = tma_tile && right_edge;
    const int xw = left_edge ? N - V : 0;
    const uint32_t wrap_tx = (wrapL || wrapR) ? (uint32_t)(4 * G::ROWS * V * sizeof(T)) : 0u, wrap2_tx = (wrapL || wrapR) ? (uint32_t)(G::ROWS * V * sizeof(T)) : 0u;
    auto issue_stage = [&](int s, int p) {   // phi_re, phi_im, theta_0, theta_1 of march plane p -> stage s
        if (tma_tile) {
            tma_load_4d(stages + s * SE, &map_stage, x0 - V, y0 - 1, plane_of(p), 0, &full[s]);
            if (wrapL || wrapR) tma_load_4d(wrapS + s * C::WRAP_ELEMS, &map_wstage, xw, y0 - 1, plane_of(p), 0, &full[s]);
        } else {
            issue_rows<G, 4>(stages + s * SE, &full[s], src, N, x0, y0, plane_of(p));
        }
    };
    // theta_2 of march plane p -> ring slot p % T2S; completion on t2full[slot], or (T2S = NS: same slot index as the stage) on full[slot]
    auto issue_th2 = [&](int slot, int p) {
        uint64_t* bar = C::T2_OWN ? &t2full[slot] : &full[slot];
        if (C::T2_OWN) mbar_arrive_expect_tx(bar, G::ARR_BYTES + wrap2_tx);
        if (tma_tile) {
            tma_load_4d(th2ring + slot * C::T2_STRIDE, &map_th2, x0 - V, y0 - 1, plane_of(p), 4, bar);
            if (wrapL || wrapR) tma_load_4d(wrapT + slot * C::WRAP2_STRIDE, &map_wth2, xw, y0 - 1, plane_of(p), 4, bar);
        } else {
            issue_rows<G, 1>(th2ring + slot * C::T2_STRIDE, bar, src2, N, x0, y0, plane_of(p));
        }
    };
    const uint32_t stage_tx = G::STAGE_BYTES + wrap_tx + (C::T2_OWN ? 0u : G::ARR_BYTES + wrap2_tx);
    // column x0-1 (array a, row r) of a staged plane / of a theta_2 slot, and the element right of this thread's vector
    auto colL = [&](const T* st, const T* side, int a, int r) -> T {
        return wrapL ? side[(a * G::ROWS + r + 1) * V + V - 1] : st[G::idx(a, r, -1)];
    };
    auto edgeR = [&](const T* st, const T* side, int a, int r, int c) -> T {   // c = column index of the element, <= TX
        return (wrapR && c == TX) ? side[(a * G::ROWS + r + 1) * V] : st[G::idx(a, r, c)];
    };
    if (w == 0) {
#pragma unroll
        for (int i = 0; i < NS; ++i) {
            if (i <= zlen + 1 && elect_one()) {   // (planes 0 .. zlen+1 are all this chunk reads; nothing may be in flight at exit)
                mbar_arrive_expect_tx(&full[i], stage_tx);
                issue_stage(i, i);
                if (!C::T2_OWN || (i < T2S && i <= zlen)) issue_th2(i, i);   // (own ring: theta_2 is read of planes 0 .. zlen only)
            }
        }
    }

    // products of the previous plane, carried in registers: b_2 = conj(U_2) phi, S_02, S_12
    T cb2r[V], cb2i[V], cS02[V], cS12[V];

    // ---- prologue: z-products of plane z0-1 (needs planes z0-1 and z0) ---------------------------------------------
    mbar_wait(&full[0], 0);
    mbar_wait(&full[1], 0);
    if (C::T2_OWN) mbar_wait(&t2full[0], 0);
    {
        const T* sc = stages;
        const T* sn = stages + SE;
        const T* t2c = th2ring;
        const VecT pr = lds_vec<T, V>(sc + G::idx(0, w, xi)), pi = lds_vec<T, V>(sc + G::idx(1, w, xi));
        const VecT t0 = lds_vec<T, V>(sc + G::idx(2, w, xi)), t1 = lds_vec<T, V>(sc + G::idx(3, w, xi)), t2 = lds_vec<T, V>(t2c + G::idx(0, w, xi));
        const VecT t2y = lds_vec<T, V>(t2c + G::idx(0, w + 1, xi));
        const VecT t0z = lds_vec<T, V>(sn + G::idx(2, w, xi)), t1z = lds_vec<T, V>(sn + G::idx(3, w, xi));
        const T t2x_edge = edgeR(t2c, wrapT, 0, w, xi + V);
        T s2[V], c2[V], X02[V], X12[V];
        sincos_vec<V>(t2.v, s2, c2);
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const Cx<T> b = mulUc<T>(c2[v], s2[v], { pr.v[v], pi.v[v] });
            cb2r[v] = b.re;
            cb2i[v] = b.im;
            X02[v] = t0.v[v] + next_x<T, V>(t2, v, t2x_edge) - t0z.v[v] - t2.v[v];
            X12[v] = t1.v[v] + t2y.v[v] - t1z.v[v] - t2.v[v];
        }
        sin_vec<V>(X02, cS02);
        sin_vec<V>(X12, cS12);
    }
    // Hand stage 0 and theta_2 slot 0 over to the copy engine with the protocol the march uses: every thread signals the
    // exchange barrier once its prologue reads have been issued (the arrive travels down the same shared-memory pipe
    // behind them, release semantics) and waits for the phase to complete, so the thread that re-fills the stage at plane 1
    // has synchronised with every reader before its fence.proxy.async.  (A __syncthreads() here was not enough on sm_100:
    // profiles/HISTORY.md, "r2 race".)  Phase 0 of `xch` = prologue, phase it = plane it.
    mbar_arrive(xch);
    mbar_wait(xch, 0);

    const T dtc2 = k.dt * k.c2, dtd3 = k.dt * k.d3;

    // The momenta (no halo) are streamed with 16-byte loads, software-pipelined by one plane: those of plane it+1 are
    // requested right after the barrier of plane it, where register pressure is lowest, and consumed at the end of phase 1
    // of plane it+1 (profiles/HISTORY.md r1: requested at the top of their own plane they cost 15 % of the issue slots in stalls).
    const size_t plane_stride = (size_t)N * N;
    size_t gnext = ((size_t)(zr.zbase + z0) * N + (size_t)(y0 + w)) * N + (size_t)(x0 + xi);
    const size_t in_plane = (size_t)(y0 + w) * N + (size_t)(x0 + xi);   // offset inside a plane: for the neighbours' ghost planes
    VecT nPr = ldg_vec<T, V>(f.pi_re + gnext), nPi = ldg_vec<T, V>(f.pi_im + gnext);
    VecT nE0 = ldg_vec<T, V>(f.eps[0] + gnext), nE1 = ldg_vec<T, V>(f.eps[1] + gnext), nE2 = ldg_vec<T, V>(f.eps[2] + gnext);

    // ---- the march -----------------------------------------------------------------------------------------------------
    for (int it = 1; it <= zlen; ++it) {
        const T* sc = stages + (it % NS) * SE;
        const T* sn = stages + ((it + 1) % NS) * SE;
        const T* t2c = th2ring + (it % T2S) * C::T2_STRIDE;
        const T* wsc = wrapS + (it % NS) * C::WRAP_ELEMS;
        const T* wsn = wrapS + ((it + 1) % NS) * C::WRAP_ELEMS;
        const T* wtc = wrapT + (it % T2S) * C::WRAP2_STRIDE;
        T* yexp = yex + (it & 1) * C::YEX_ELEMS;
        T* xexp = xex + (it & 1) * C::XEX_ELEMS;

        // ---- plane it+NS-1 -> the stage that held plane it-1 (its last readers passed the barrier of iteration it-1) ----
        if (((w + it) % TY) == ISSUER && it + NS - 1 <= zlen + 1 && elect_one()) {
            const int s = (it + NS - 1) % NS;   // with it: theta_2 of plane it+NS-2 -> the slot that held plane it-1
            fence_proxy_async();   // (this thread waited on the exchange barrier of plane it-1 / of the prologue: all reads of that stage are done)
            mbar_arrive_expect_tx(&full[s], stage_tx);
            issue_stage(s, it + NS - 1);
            if (C::T2_OWN) issue_th2((it + NS - 2) % T2S, it + NS - 2);   // (read at iteration it+NS-2, after the wait on its own barrier)
            else issue_th2(s, it + NS - 1);
        }

        const size_t g = gnext;                                         // plane z0 + it - 1
        const VecT Pr = nPr, Pi = nPi, E0 = nE0, E1 = nE1, E2 = nE2;   // requested one plane ago

        if (C::T2_OWN) mbar_wait(&t2full[it % T2S], (it / T2S) & 1);   // theta_2 of this plane (requested NS-2 planes ago)
        // The stage of the NEXT plane is needed for the +z neighbours only.  fp32: wait for it after the trigonometry of the in-plane links (a
        // third of the plane's work later: the copy has that much longer to land; 15.3 -> 15.05 ms at 1024^3 on a 1.49 GHz board); fp64: here
        // (measured: no gain from waiting later, profiles/HISTORY.md r5)
        if constexpr (!StepShape<T>::LATE_WAIT) mbar_wait(&full[(it + 1) % NS], ((it + 1) / NS) & 1);

        // ---- halo products, shared out over the warps (no dedicated producer warp).  Row y0-1: one site per lane, every
        //      HSTRIDE-th warp in rotation; column x0-1: one warp per plane.  Called before the exchange barrier is signalled.
        auto halo_jobs = [&]() {
            if (((w + it) % HSTRIDE) == 0) {
                const int x = 32 * (w / HSTRIDE) + lane;   // halo row y0-1: b_1, S_01, S_12 -> exchange row 0
                const T pr = sc[G::idx(0, -1, x)], pi = sc[G::idx(1, -1, x)];
                const T t0 = sc[G::idx(2, -1, x)], t1 = sc[G::idx(3, -1, x)], t2 = t2c[G::idx(0, -1, x)];
                const T t1x = edgeR(sc, wsc, 3, -1, x + 1), t0y = sc[G::idx(2, 0, x)], t2y = t2c[G::idx(0, 0, x)], t1z = sn[G::idx(3, -1, x)];
                T s, c;
                sincos_fast(t1, s, c);
                const Cx<T> b = mulUc<T>(c, s, { pr, pi });
                yexp[(0 * TY + 0) * TX + x] = b.re;
                yexp[(1 * TY + 0) * TX + x] = b.im;
                yexp[(2 * TY + 0) * TX + x] = sin_fast(t0 + t1x - t0y - t1);
                yexp[(3 * TY + 0) * TX + x] = sin_fast(t1 + t2y - t1z - t2);
            }
            if (((w + it) % TY) == COLUMN && lane < TY) {   // halo column x0-1, row r = lane: b_0, S_01, S_02
                const int r = lane;
                const T pr = colL(sc, wsc, 0, r), pi = colL(sc, wsc, 1, r);
                const T t0 = colL(sc, wsc, 2, r), t1 = colL(sc, wsc, 3, r), t2 = colL(t2c, wtc, 0, r);
                const T t1x = sc[G::idx(3, r, 0)], t2x = t2c[G::idx(0, r, 0)];
                const T t0y = colL(sc, wsc, 2, r + 1), t0z = colL(sn, wsn, 2, r);
                T s, c;
                sincos_fast(t0, s, c);
                const Cx<T> b = mulUc<T>(c, s, { pr, pi });
                xexp[0 * TY + r] = b.re;
                xexp[1 * TY + r] = b.im;
                xexp[2 * TY + r] = sin_fast(t0 + t1x - t0y - t1);
                xexp[3 * TY + r] = sin_fast(t0 + t2x - t0z - t2);
            }
        };

        // partial results that cross the barrier (phase 1 -> phase 2)
        T qr[V], qi[V], fr[V], fi[V], e0[V], e1[V], e2[V], g0[V], g1[V], g2[V];
        {
            // ---- phase 1: products and everything this thread owns -----------------------------------------------------
            const VecT pr = lds_vec<T, V>(sc + G::idx(0, w, xi)), pi = lds_vec<T, V>(sc + G::idx(1, w, xi));
            const VecT t0 = lds_vec<T, V>(sc + G::idx(2, w, xi)), t1 = lds_vec<T, V>(sc + G::idx(3, w, xi)), t2 = lds_vec<T, V>(t2c + G::idx(0, w, xi));
            const VecT pry = lds_vec<T, V>(sc + G::idx(0, w + 1, xi)), piy = lds_vec<T, V>(sc + G::idx(1, w + 1, xi));
            const VecT t0y = lds_vec<T, V>(sc + G::idx(2, w + 1, xi)), t2y = lds_vec<T, V>(t2c + G::idx(0, w + 1, xi));
            const T prx_e = edgeR(sc, wsc, 0, w, xi + V), pix_e = edgeR(sc, wsc, 1, w, xi + V);
            const T t1x_e = edgeR(sc, wsc, 3, w, xi + V), t2x_e = edgeR(t2c, wtc, 0, w, xi + V);
            T lfr[V], lfi[V], J0[V], J1[V], J2[V], b0r[V], b0i[V], S01[V], S02[V], S12[V], b2r[V], b2i[V];
            VecT yb1r, yb1i, yS01, yS12;
            // the six transcendental evaluations per site, V sites at once (fp32: packed two-lane arithmetic, ahs_trig.cuh)
            T s0[V], c0[V], s1[V], c1[V], s2[V], c2[V];
            sincos_vec<V>(t0.v, s0, c0);
            sincos_vec<V>(t1.v, s1, c1);
            sincos_vec<V>(t2.v, s2, c2);
            {
                // Xi_ij^x = th_i^x + th_j^{x+k_i} - th_i^{x+k_j} - th_j^x  (Eq. 3): the plaquette inside the plane first
                T X01[V];
#pragma unroll
                for (int v = 0; v < V; ++v) X01[v] = t0.v[v] + next_x<T, V>(t1, v, t1x_e) - t0y.v[v] - t1.v[v];
                sin_vec<V>(X01, S01);
            }
            if constexpr (StepShape<T>::LATE_WAIT) mbar_wait(&full[(it + 1) % NS], ((it + 1) / NS) & 1);
            const VecT prz = lds_vec<T, V>(sn + G::idx(0, w, xi)), piz = lds_vec<T, V>(sn + G::idx(1, w, xi));
            const VecT t0z = lds_vec<T, V>(sn + G::idx(2, w, xi)), t1z = lds_vec<T, V>(sn + G::idx(3, w, xi));
            {
                T X02[V], X12[V];
#pragma unroll
                for (int v = 0; v < V; ++v) {
                    X02[v] = t0.v[v] + next_x<T, V>(t2, v, t2x_e) - t0z.v[v] - t2.v[v];
                    X12[v] = t1.v[v] + t2y.v[v] - t1z.v[v] - t2.v[v];
                }
                sin_vec<V>(X02, S02);
                sin_vec<V>(X12, S12);
            }
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const Cx<T> ph = { pr.v[v], pi.v[v] };
                const Cx<T> f0 = mulU<T>(c0[v], s0[v], { next_x<T, V>(pr, v, prx_e), next_x<T, V>(pi, v, pix_e) });
                const Cx<T> b0 = mulUc<T>(c0[v], s0[v], ph);
                const Cx<T> f1 = mulU<T>(c1[v], s1[v], { pry.v[v], piy.v[v] });
                const Cx<T> b1 = mulUc<T>(c1[v], s1[v], ph);
                const Cx<T> f2 = mulU<T>(c2[v], s2[v], { prz.v[v], piz.v[v] });
                const Cx<T> b2 = mulUc<T>(c2[v], s2[v], ph);
                lfr[v] = (f0.re + f1.re) + f2.re;
                lfi[v] = (f0.im + f1.im) + f2.im;
                // J_j = Im[conj(phi^x) U_j phi^{x+k_j}]  (Eq. 5, 2nd term)
                J0[v] = ph.re * f0.im - ph.im * f0.re;
                J1[v] = ph.re * f1.im - ph.im * f1.re;
                J2[v] = ph.re * f2.im - ph.im * f2.re;
                b0r[v] = b0.re; b0i[v] = b0.im;
                yb1r.v[v] = b1.re; yb1i.v[v] = b1.im;
                b2r[v] = b2.re; b2i[v] = b2.im;
                yS01.v[v] = S01[v];
                yS12.v[v] = S12[v];
            }
            if (w + 1 < TY) {   // (the last row's -y products belong to the tile above, which recomputes them)
            sts_vec<T, V>(yexp + (0 * TY + w + 1) * TX + xi, yb1r);
            sts_vec<T, V>(yexp + (1 * TY + w + 1) * TX + xi, yb1i);
            sts_vec<T, V>(yexp + (2 * TY + w + 1) * TX + xi, yS01);
            sts_vec<T, V>(yexp + (3 * TY + w + 1) * TX + xi, yS12);
            }
            halo_jobs();
            // Everything other warps need from this one is in shared memory and this warp has finished reading the staged
            // planes: signal the exchange barrier now and fold the owned terms (no shared memory involved) while the other
            // warps catch up; the wait comes just before phase 2.
            mbar_arrive(xch);
            // -x products of the lane to the left (lane 0 gets its halo-column values in phase 2)
            T lb0r = __shfl_up_sync(0xffffffffu, b0r[V - 1], 1), lb0i = __shfl_up_sync(0xffffffffu, b0i[V - 1], 1);
            T lS01 = __shfl_up_sync(0xffffffffu, S01[V - 1], 1), lS02 = __shfl_up_sync(0xffffffffu, S02[V - 1], 1);
            if (lane == 0) { lb0r = T(0); lb0i = T(0); lS01 = T(0); lS02 = T(0); }
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const int vp = v > 0 ? v - 1 : 0;
                const T mb0r = v > 0 ? b0r[vp] : lb0r, mb0i = v > 0 ? b0i[vp] : lb0i;
                const T mS01 = v > 0 ? S01[vp] : lS01, mS02 = v > 0 ? S02[vp] : lS02;
                const T lap_re = (lfr[v] - T(6) * pr.v[v]) + (mb0r + cb2r[v]);   // without b_1^{-y} (and the halo b_0)
                const T lap_im = (lfi[v] - T(6) * pi.v[v]) + (mb0i + cb2i[v]);
                const T higgs = k.c3 * (pr.v[v] * pr.v[v] + pi.v[v] * pi.v[v] - k.sigma2);
                qr[v] = k.c1 * Pr.v[v] - higgs * pr.v[v] + k.c2 * lap_re;       // Eq. 4, owned part
                qi[v] = k.c1 * Pi.v[v] - higgs * pi.v[v] + k.c2 * lap_im;
                fr[v] = pr.v[v] + k.dt * qr[v];                                  // Eq. 6, owned part
                fi[v] = pi.v[v] + k.dt * qi[v];
                // Eq. 5, owned part of the curl: everything except S01^{-y}, S12^{-y} (and the halo S01^{-x}, S02^{-x})
                e0[v] = k.d1 * E0.v[v] + k.d2 * J0[v] - k.d3 * ((S01[v] + S02[v]) - cS02[v]);
                e1[v] = k.d1 * E1.v[v] + k.d2 * J1[v] - k.d3 * ((S12[v] - S01[v]) + (mS01 - cS12[v]));
                e2[v] = k.d1 * E2.v[v] + k.d2 * J2[v] - k.d3 * (mS02 - (S02[v] + S12[v]));
                g0[v] = t0.v[v] + k.dt * e0[v];                                  // Eq. 7, owned part
                g1[v] = t1.v[v] + k.dt * e1[v];
                g2[v] = t2.v[v] + k.dt * e2[v];
                cb2r[v] = b2r[v]; cb2i[v] = b2i[v]; cS02[v] = S02[v]; cS12[v] = S12[v];
            }
        }
        gnext = g + plane_stride;
        if (it < zlen) {
            nPr = ldg_vec<T, V>(f.pi_re + gnext); nPi = ldg_vec<T, V>(f.pi_im + gnext);
            nE0 = ldg_vec<T, V>(f.eps[0] + gnext); nE1 = ldg_vec<T, V>(f.eps[1] + gnext); nE2 = ldg_vec<T, V>(f.eps[2] + gnext);
        }
        mbar_wait(xch, it & 1);   // all 128 threads have signalled plane `it`: exchange rows complete, stages no longer read
        {
            // ---- phase 2: the terms that crossed a warp or tile boundary, then the stores ----------------------------
            const VecT yb1r = lds_vec<T, V>(yexp + (0 * TY + w) * TX + xi), yb1i = lds_vec<T, V>(yexp + (1 * TY + w) * TX + xi);
            const VecT yS01 = lds_vec<T, V>(yexp + (2 * TY + w) * TX + xi), yS12 = lds_vec<T, V>(yexp + (3 * TY + w) * TX + xi);
            T hb0r = xexp[0 * TY + w], hb0i = xexp[1 * TY + w], hS01 = xexp[2 * TY + w], hS02 = xexp[3 * TY + w];
            if (lane != 0) { hb0r = T(0); hb0i = T(0); hS01 = T(0); hS02 = T(0); }
            VecT oPr, oPi, oE0, oE1, oE2, oFr, oFi, oT0, oT1, oT2;
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const T nr = v == 0 ? yb1r.v[v] + hb0r : yb1r.v[v];
                const T ni = v == 0 ? yb1i.v[v] + hb0i : yb1i.v[v];
                const T c1x = v == 0 ? hS01 : T(0);                 // S01^{-x} of the halo column
                const T c2x = v == 0 ? yS12.v[v] + hS02 : yS12.v[v];   // S12^{-y} + S02^{-x}(halo)
                oPr.v[v] = qr[v] + k.c2 * nr;
                oPi.v[v] = qi[v] + k.c2 * ni;
                oFr.v[v] = fr[v] + dtc2 * nr;
                oFi.v[v] = fi[v] + dtc2 * ni;
                oE0.v[v] = e0[v] + k.d3 * yS01.v[v];
                oT0.v[v] = g0[v] + dtd3 * yS01.v[v];
                oE1.v[v] = v == 0 ? e1[v] - k.d3 * c1x : e1[v];
                oT1.v[v] = v == 0 ? g1[v] - dtd3 * c1x : g1[v];
                oE2.v[v] = e2[v] - k.d3 * c2x;
                oT2.v[v] = g2[v] - dtd3 * c2x;
            }
            stg_vec<T, V>(f.pi_re + g, oPr); stg_vec<T, V>(f.pi_im + g, oPi);
            stg_vec<T, V>(f.eps[0] + g, oE0); stg_vec<T, V>(f.eps[1] + g, oE1); stg_vec<T, V>(f.eps[2] + g, oE2);
            stg_vec<T, V>(f.phi_re_out + g, oFr); stg_vec<T, V>(f.phi_im_out + g, oFi);
            stg_vec<T, V>(f.th_out[0] + g, oT0); stg_vec<T, V>(f.th_out[1] + g, oT1); stg_vec<T, V>(f.th_out[2] + g, oT2);
            // z-slabs: the new (phi, theta) of the bottom / top own plane also go into the neighbouring slabs' ghost planes (peer
            // memory when they live on another GPU: the exchange of DESIGN.md 10 is these stores), eps_2 of the top plane as well
            const int zown = z0 + it - 1;
            if (zown == 0 && gh.lo[0] != nullptr) {
                stg_vec<T, V>(gh.lo[0] + in_plane, oFr); stg_vec<T, V>(gh.lo[1] + in_plane, oFi);
                stg_vec<T, V>(gh.lo[2] + in_plane, oT0); stg_vec<T, V>(gh.lo[3] + in_plane, oT1); stg_vec<T, V>(gh.lo[4] + in_plane, oT2);
            }
            if (zown == zr.nz - 1 && gh.hi[0] != nullptr) {
                stg_vec<T, V>(gh.hi[0] + in_plane, oFr); stg_vec<T, V>(gh.hi[1] + in_plane, oFi);
                stg_vec<T, V>(gh.hi[2] + in_plane, oT0); stg_vec<T, V>(gh.hi[3] + in_plane, oT1); stg_vec<T, V>(gh.hi[4] + in_plane, oT2);
                stg_vec<T, V>(gh.eps2_hi + in_plane, oE2);
            }
        }
    }
}

// Number of z-chunks per tile.  A chunk start costs one extra staged plane and the trigonometry of its -z products, so long
// marches look attractive -- but measured (profiles/r4_chunks.md) shorter ones win: CTAs that start together drift apart
// along z, their halo rows then miss L2, and every chunk boundary re-aligns them.  32 chunks (fp32) / 16 (fp64, twice the
// tiles per plane) were fastest at 256^3, 512^3 and 1024^3 alike; chunk counts that do not divide N lose 3-6 % at small N.
template <typename T>
int pick_chunks(int N, int nz)
{
    int c = sizeof(T) == 4 ? 32 : 16;
    while (c > 1 && (N % c != 0 || N / c < 4)) c /= 2;
    const int zlen = N / c;                 // planes per chunk, read off the whole lattice; a slab of nz planes gets nz / zlen chunks
    return nz >= zlen ? nz / zlen : 1;
}

template <typename T, int TY, int MINB, int NSTG>
int launch_cfg(const FieldPtrs<T>& f, int N, const ZRange& zr, const GhostPtrs<T>* ghosts, const StepCoef& c, const StepMaps* maps,
               const MarchOptions& opt, cudaStream_t st)
{
    using C = MarchCfg<T, TY, NSTG>;
    auto kern = step_march_kernel<T, TY, MINB, NSTG>;
    static SmemAttribute attr;   // per device: the kernel needs more than the default 48 KB of dynamic shared memory
    if (!attr.ensure(kern, C::SMEM)) return AHS_ERR_CUDA;
    const int nchunks = (opt.step_chunks > 0 && opt.step_chunks <= zr.nz) ? opt.step_chunks : pick_chunks<T>(N, zr.nz);
    const long blocks = (long)(N / C::TX) * (N / TY) * nchunks;
    GhostPtrs<T> gh;
    memset(&gh, 0, sizeof(gh));
    if (ghosts) gh = *ghosts;
    StepCoefT<T> k = { (T)c.c1, (T)c.c2, (T)c.c3, (T)c.d1, (T)c.d2, (T)c.d3, (T)c.dt, (T)c.sigma2 };
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3((unsigned)blocks);
    cfg.blockDim = dim3(C::NTHREADS);
    cfg.dynamicSmemBytes = C::SMEM;
    cfg.stream = st;
    cudaLaunchAttribute pdl[1];
    pdl[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // this launch may begin before the stream's previous kernel has drained
    pdl[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = pdl;
    cfg.numAttrs = opt.step_pdl ? 1 : 0;
    StepMaps none;
    memset(&none, 0, sizeof(none));
    const bool tma = maps && opt.staging == AHS_STAGING_TENSOR;
    const StepMaps& mp = tma ? *maps : none;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, kern, f, gh, N, zr, nchunks, k, mp.stage, mp.th2, mp.wstage, mp.wth2, tma ? 1 : 0);
    return (e == cudaSuccess && cudaGetLastError() == cudaSuccess) ? 1 : AHS_ERR_CUDA;
}

}  // namespace

template <typename T>
bool march_supported(int N)
{
    using C = MarchCfg<T, StepShape<T>::TY, StepShape<T>::NS>;
    return N >= C::TX && N % C::TX == 0 && N % C::TY == 0;
}

template <typename T>
int launch_step_march(const FieldPtrs<T>& f, int N, const ZRange& zr, const GhostPtrs<T>* ghosts, const StepCoef& c, const StepMaps* maps,
                      const MarchOptions& opt, cudaStream_t st)
{
    if (!march_supported<T>(N) || zr.nz < 1) return AHS_ERR_INVALID_ARG;
    return launch_cfg<T, StepShape<T>::TY, StepShape<T>::MINB, StepShape<T>::NS>(f, N, zr, ghosts, c, maps, opt, st);
}

// the marching diagnostics kernel lives in ahs_diag_march.cu
template bool march_supported<float>(int);
template bool march_supported<double>(int);
template int launch_step_march<float>(const FieldPtrs<float>&, int, const ZRange&, const GhostPtrs<float>*, const StepCoef&, const StepMaps*, const MarchOptions&, cudaStream_t);
template int launch_step_march<double>(const FieldPtrs<double>&, int, const ZRange&, const GhostPtrs<double>*, const StepCoef&, const StepMaps*, const MarchOptions&, cudaStream_t);

// tensor maps of one (phi, theta) buffer for the tile shape above
template <typename T>
bool make_step_march_maps(StepMaps* out, const void* phi_re_base, int N, int nz_alloc, size_t array_bytes)
{
    using C = MarchCfg<T, StepShape<T>::TY, StepShape<T>::NS>;
    using G = typename C::G;
    if (!march_supported<T>(N)) return false;
    return make_tile_map<T>(&out->stage, phi_re_base, N, nz_alloc, array_bytes, 5, G::PITCH, G::ROWS, 4) &&
           make_tile_map<T>(&out->th2, phi_re_base, N, nz_alloc, array_bytes, 5, G::PITCH, G::ROWS, 1) &&
           make_tile_map<T>(&out->wstage, phi_re_base, N, nz_alloc, array_bytes, 5, C::V, G::ROWS, 4) &&
           make_tile_map<T>(&out->wth2, phi_re_base, N, nz_alloc, array_bytes, 5, C::V, G::ROWS, 1);
}
template bool make_step_march_maps<float>(StepMaps*, const void*, int, int, size_t);
template bool make_step_march_maps<double>(StepMaps*, const void*, int, int, size_t);

}  // namespace ahs
