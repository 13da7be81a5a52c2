// ahs_reduce.cuh -- warp-shuffle and block reductions of the diagnostics record (PAPER.md L140 uses CUB block
// sums and a host-side final sum; here: shuffle tree -> shared memory -> one partial per block -> one finishing block).
#pragma once
#include "ahs_internal.cuh"

namespace ahs {

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ unsigned long long warp_sum(unsigned long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// Block-level reduction of a per-thread record; thread 0 of the block writes the block's partial.
// The order is fixed by (warp lane tree, then warp index), so a given launch shape is deterministic.
// Every thread of the block must call it (it contains a __syncthreads).
__device__ __forceinline__ void block_reduce_store(DiagPartial v, DiagPartial* out)
{
    __shared__ DiagPartial sh[32];
    v.n_pierced = warp_sum(v.n_pierced);
    v.sum_abs_w = warp_sum(v.sum_abs_w);
    v.num = warp_sum(v.num);
    v.den = warp_sum(v.den);
    v.lsum = warp_sum(v.lsum);
    v.gmax = warp_max(v.gmax);
    v.rhs2 = warp_sum(v.rhs2);
    v.nonfinite = warp_sum(v.nonfinite);
    v.vnum = warp_sum(v.vnum);
    v.vden = warp_sum(v.vden);
    v.wnum = warp_sum(v.wnum);
    v.wden = warp_sum(v.wden);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        DiagPartial t = sh[0];
        for (int w = 1; w < nwarp; ++w) {
            t.n_pierced += sh[w].n_pierced; t.sum_abs_w += sh[w].sum_abs_w;
            t.num += sh[w].num; t.den += sh[w].den; t.lsum += sh[w].lsum;
            t.gmax = fmax(t.gmax, sh[w].gmax); t.rhs2 += sh[w].rhs2; t.nonfinite += sh[w].nonfinite;
            t.vnum += sh[w].vnum; t.vden += sh[w].vden; t.wnum += sh[w].wnum; t.wden += sh[w].wden;
        }
        *out = t;
    }
}

}  // namespace ahs
