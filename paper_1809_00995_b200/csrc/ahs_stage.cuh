// ahs_stage.cuh -- shared-memory staging of halo'd xy tiles of the level-n fields, one z-plane per stage,
// filled by the bulk asynchronous copy engine (cp.async.bulk, SASS UBLKCP) and tracked by mbarriers.
//
// A CTA owns a tile of TX x TY sites in (x, y) and marches along z.  A stage holds, for each staged array,
// rows y0-1 .. y0+TY of the plane and, in each row, the sites x0-V .. x0+TX+V-1 (V = 16 bytes worth of
// elements, so that every row segment is a 16-byte aligned contiguous run in global memory; periodic wrap
// is resolved per row segment by the issuing lane).  No tensor map is needed: a row segment of an x-fastest
// SoA array IS contiguous.  The paper stages tiles with per-thread loads and explicit halo threads
// (Fig. 1); here one thread issues the row copies of a plane and nobody touches the data until
// the mbarrier flips.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

namespace ahs {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
// Order this thread's earlier generic-proxy accesses to shared memory (and those it has synchronised with) before its
// later async-proxy operations: to be executed by the copy-issuing thread before it re-fills a stage that was read
// with ordinary loads.
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)   // release semantics at CTA scope (the PTX default)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    const uint32_t a = smem_u32(bar);
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(a), "r"(parity)
            : "memory");
    } while (!done);
}
// one lane of the (converged) warp: elect.sync tells the compiler that exactly one thread runs the guarded code, so
// the uniform-register operands of cp.async.bulk need no per-lane serialisation loop
__device__ __forceinline__ bool elect_one()
{
    uint32_t pred;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(pred));
    return pred != 0;
}
// global -> shared bulk copy of `bytes` (multiple of 16; both addresses 16-byte aligned), completion on `bar`
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// 16-byte vector of V elements of T
template <typename T, int V>
struct alignas(sizeof(T) * V) Vec {
    T v[V];
};

// ---- vector access helpers shared by the marching kernels -------------------------------------------------------
template <typename T> struct NativeVec;
template <> struct NativeVec<float> { using type = float4; };
template <> struct NativeVec<double> { using type = double2; };

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
    *reinterpret_cast<NV*>(p) = n;   // (st.global.cs measured: no difference, profiles/HISTORY.md r3)
}

// element v+1 of a vector, or the scalar `edge` (the first element of the next vector) for the last one
template <typename T, int V>
__device__ __forceinline__ T next_x(const Vec<T, V>& a, int v, T edge) { return v + 1 < V ? a.v[v + 1 < V ? v + 1 : v] : edge; }


// Geometry of a staged tile.  NA = number of staged arrays; LH = halo columns left of the tile (V or 0), BH = halo rows
// below it (1 or 0).  The forward halo (V columns right, one row above) is always there.
template <typename T, int V_, int TY_, int NA_, int NSTAGE_, int LH_ = V_, int BH_ = 1>
struct TileGeom {
    static constexpr int V = V_;
    static constexpr int TY = TY_;
    static constexpr int NA = NA_;
    static constexpr int NSTAGE = NSTAGE_;
    static constexpr int LH = LH_;
    static constexpr int BH = BH_;
    static constexpr int TX = 32 * V;              // one warp spans the tile in x
    static constexpr int PITCH = TX + LH + V;      // x0-LH .. x0+TX+V-1
    static constexpr int ROWS = TY + BH + 1;       // y0-BH .. y0+TY
    static constexpr int ARR_ELEMS = ROWS * PITCH;
    static constexpr int STAGE_ELEMS = NA * ARR_ELEMS;
    static constexpr uint32_t STAGE_BYTES = STAGE_ELEMS * sizeof(T);
    static constexpr uint32_t ARR_BYTES = ARR_ELEMS * sizeof(T);
    static_assert(sizeof(T) * V == 16, "a vector is 16 bytes");
    static_assert(LH == 0 || LH == V, "the left halo is one vector or nothing");

    // element (array a, row r in [-BH, TY], column xi in [-LH, TX+V)) of a stage
    __device__ __forceinline__ static int idx(int a, int r, int xi) { return (a * ROWS + (r + BH)) * PITCH + (xi + LH); }
};

// Issue the copies of one z-plane of NA arrays into NA consecutive array slots at `dst`.  Called by ONE thread, after
// it has posted the expected byte count on `bar` (mbar_arrive_expect_tx).  cp.async.bulk takes its operands from
// uniform registers, so copies issued by several lanes of a warp are serialised by a per-lane loop of ~15
// instructions each (profiles/HISTORY.md r1: 15 % of all instructions executed); a single thread walking the rows with
// running pointers costs a third of that.
//   src[a]  : global base pointers of the arrays
//   z       : plane (already wrapped into [0, N))
template <typename G, int NA, typename T>
__device__ __forceinline__ void issue_rows(T* dst_base, uint64_t* bar, const T* const (&src)[NA], int N, int x0, int y0, int z)
{
    const bool x_interior = (G::LH == 0 || x0 > 0) && (x0 + G::TX < N);
    const bool y_interior = (G::BH == 0 || y0 > 0) && (y0 + G::TY < N);
    const size_t plane = (size_t)z * N * N;
    if (x_interior && y_interior) {
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            const T* row = src[a] + plane + (size_t)(y0 - G::BH) * N + (x0 - G::LH);
            T* dst = dst_base + a * G::ARR_ELEMS;
#pragma unroll
            for (int rr = 0; rr < G::ROWS; ++rr) bulk_g2s(dst + rr * G::PITCH, row + (size_t)rr * N, G::PITCH * sizeof(T), bar);
        }
        return;
    }
    const int xl = x0 == 0 ? N - G::V : x0 - G::V;
    const int xr = x0 + G::TX == N ? 0 : x0 + G::TX;
#pragma unroll
    for (int a = 0; a < NA; ++a) {
        T* dst = dst_base + a * G::ARR_ELEMS;
#pragma unroll 1
        for (int rr = 0; rr < G::ROWS; ++rr) {
            int y = y0 + rr - G::BH;
            y = y < 0 ? y + N : (y >= N ? y - N : y);
            const T* row = src[a] + plane + (size_t)y * N;
            if (x_interior) {
                bulk_g2s(dst + rr * G::PITCH, row + x0 - G::LH, G::PITCH * sizeof(T), bar);
            } else {
                if (G::LH > 0) bulk_g2s(dst + rr * G::PITCH, row + xl, 16, bar);
                bulk_g2s(dst + rr * G::PITCH + G::LH, row + x0, G::TX * sizeof(T), bar);
                bulk_g2s(dst + rr * G::PITCH + G::LH + G::TX, row + xr, 16, bar);
            }
        }
    }
}

}  // namespace ahs
