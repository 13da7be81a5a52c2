// ahs_stage.cuh -- shared-memory staging of halo'd xy tiles of the level-n fields, one z-plane per stage,
// filled by the bulk asynchronous copy engine (cp.async.bulk, SASS UBLKCP) and tracked by mbarriers.
//
// A CTA owns a tile of TX x TY sites in (x, y) and marches along z.  A stage holds, for each staged array,
// rows y0-1 .. y0+TY of the plane and, in each row, the sites x0-V .. x0+TX+V-1 (V = 16 bytes worth of
// elements, so that every row segment is a 16-byte aligned contiguous run in global memory; periodic wrap
// is resolved per row segment by the issuing lane).  No tensor map is needed: a row segment of an x-fastest
// SoA array IS contiguous.  The paper stages tiles with per-thread loads and explicit halo threads
// (Fig. 1); here one warp issues ~50 row copies per plane and nobody touches the data until
// the mbarrier flips.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

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
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
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

// Geometry of a staged tile.  NA = number of staged arrays.
template <typename T, int V_, int TY_, int NA_, int NSTAGE_>
struct TileGeom {
    static constexpr int V = V_;
    static constexpr int TY = TY_;
    static constexpr int NA = NA_;
    static constexpr int NSTAGE = NSTAGE_;
    static constexpr int TX = 32 * V;              // one warp spans the tile in x
    static constexpr int PITCH = TX + 2 * V;       // x0-V .. x0+TX+V-1
    static constexpr int ROWS = TY + 2;            // y0-1 .. y0+TY
    static constexpr int ARR_ELEMS = ROWS * PITCH;
    static constexpr int STAGE_ELEMS = NA * ARR_ELEMS;
    static constexpr uint32_t STAGE_BYTES = STAGE_ELEMS * sizeof(T);
    static_assert(sizeof(T) * V == 16, "a vector is 16 bytes");

    // element (array a, row r in [-1, TY], column xi in [-V, TX+V)) of a stage
    __device__ __forceinline__ static int idx(int a, int r, int xi) { return (a * ROWS + (r + 1)) * PITCH + (xi + V); }
};

// Issue the copies of one z-plane into one stage.  Called by all 32 lanes of the producer warp.
//   src[a]  : global base pointers of the NA staged arrays
//   z       : plane (already wrapped into [0, N))
template <typename G, typename T>
__device__ __forceinline__ void issue_plane(T* stage, uint64_t* bar, const T* const (&src)[G::NA], int N, int x0, int y0, int z, int lane)
{
    if (lane == 0) mbar_arrive_expect_tx(bar, G::STAGE_BYTES);
    __syncwarp();
    const bool interior = (x0 > 0) && (x0 + G::TX < N);   // warp-uniform
    for (int i = lane; i < G::NA * G::ROWS; i += 32) {
        const int a = i / G::ROWS, rr = i - a * G::ROWS;
        int y = y0 + rr - 1;
        y = y < 0 ? y + N : (y >= N ? y - N : y);
        // (a select chain, not src[a]: a dynamically indexed pointer array would live in local memory)
        const T* base = src[0];
#pragma unroll
        for (int j = 1; j < G::NA; ++j) base = (a == j) ? src[j] : base;
        const T* row = base + ((size_t)z * N + y) * N;
        T* dst = stage + (a * G::ROWS + rr) * G::PITCH;
        if (interior) {
            bulk_g2s(dst, row + x0 - G::V, G::PITCH * sizeof(T), bar);
        } else {
            const int xl = x0 == 0 ? N - G::V : x0 - G::V;
            const int xr = x0 + G::TX == N ? 0 : x0 + G::TX;
            bulk_g2s(dst, row + xl, 16, bar);
            bulk_g2s(dst + G::V, row + x0, G::TX * sizeof(T), bar);
            bulk_g2s(dst + G::V + G::TX, row + xr, 16, bar);
        }
    }
}

}  // namespace ahs
