// ahs_tma.cuh -- tensor-map (TMA) loads of a whole halo'd tile of several SoA arrays with ONE instruction.
//
// The level-n fields of one (phi, theta) buffer are five equally spaced N^3 arrays, i.e. a rank-4 tensor
// (x, y, z, array) with byte strides (sizeof T, N sizeof T, N^2 sizeof T, array_bytes).  A box of
// (PITCH, ROWS, 1, NA) elements of it is exactly the shared-memory layout of TileGeom (array-major, then rows of
// PITCH elements), so cp.async.bulk.tensor.4d (SASS UTMALDG) fills a stage that took 25-30 row copies (UBLKCP) before.
// Measured reason (profiles/HISTORY.md r2): the copy engine serves ~35 bulk requests per microsecond and SM; with 3 CTAs x 25-90
// row copies per plane the marching kernels waited for their stages 30 % of the time.
// TMA fills out-of-bounds elements with zeros, it does not wrap: tiles that touch the periodic boundary keep the
// row-copy path of ahs_stage.cuh (1/8 of the tiles at 1024^3).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace ahs {

#ifdef __CUDACC__
// global -> shared tensor copy of one box; completion (box bytes, zero-filled parts included) on `bar`
__device__ __forceinline__ void tma_load_4d(void* dst_smem, const CUtensorMap* map, int c0, int c1, int c2, int c3, uint64_t* bar)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(
            (uint32_t)__cvta_generic_to_shared(dst_smem)),
        "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"((uint32_t)__cvta_generic_to_shared(bar))
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_descriptor(const CUtensorMap* map)
{
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(map)) : "memory");
}
#endif

// Host: encode the rank-4 map of `narrays` arrays of N^3 elements starting at `base` (DEVICE pointer, 16-byte aligned),
// spaced by array_bytes, with a box of (box_x, box_y, 1, box_a) elements.  Returns false if the driver entry point is
// missing or the encode fails (the callers then keep the row-copy path).
template <typename T>
inline bool make_tile_map(CUtensorMap* out, const void* base, int N, int nz_alloc, size_t array_bytes, int narrays, int box_x, int box_y, int box_a)
{
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                 const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static EncodeFn encode = [] {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) fn = nullptr;
        return reinterpret_cast<EncodeFn>(fn);
    }();
    if (!encode) { cudaGetLastError(); return false; }
    const cuuint64_t gdim[4] = { (cuuint64_t)N, (cuuint64_t)N, (cuuint64_t)nz_alloc, (cuuint64_t)narrays };
    const cuuint64_t gstride[3] = { (cuuint64_t)N * sizeof(T), (cuuint64_t)N * N * sizeof(T), (cuuint64_t)array_bytes };
    const cuuint32_t box[4] = { (cuuint32_t)box_x, (cuuint32_t)box_y, 1u, (cuuint32_t)box_a };
    const cuuint32_t estr[4] = { 1u, 1u, 1u, 1u };
    const CUtensorMapDataType dt = sizeof(T) == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
    const CUresult r = encode(out, dt, 4, const_cast<void*>(base), gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

}  // namespace ahs
