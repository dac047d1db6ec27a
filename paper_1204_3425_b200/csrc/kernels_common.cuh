// Device helpers shared by all kernels of libhubbard_b200: deterministic block
// and grid reductions (warp shuffles -> shared memory -> per-block partial ->
// the last block to arrive sums the partials in index order).
#pragma once
#include <cuda_runtime.h>

#include "model.h"

namespace hub {

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum over the block; result valid in thread 0.  `red` has >= 32 doubles.
__device__ __forceinline__ double block_sum(double v, double *red)
{
    v = warp_sum(v);
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();  // protect `red` from a previous use
    if (lane == 0) red[w] = v;
    __syncthreads();
    if (w == 0) {
        int nw = (blockDim.x + 31) >> 5;
        v = (lane < nw) ? red[lane] : 0.0;
        v = warp_sum(v);
    }
    return v;
}

// Called by every thread of every block after block_sum: thread 0 publishes the
// block's partial at `slot`; returns true (block-uniformly) in the block that
// arrives last, after which that block may read all `n_slots` partials.
__device__ __forceinline__ bool publish_and_check_last(double partial, double *partials, int64_t slot,
                                                       unsigned n_blocks, unsigned *ticket, int *flag_smem)
{
    if (threadIdx.x == 0) {
        partials[slot] = partial;
        __threadfence();
        unsigned prev = atomicAdd(ticket, 1u);
        *flag_smem = (prev == n_blocks - 1);
    }
    __syncthreads();
    bool last = (*flag_smem != 0);
    if (last) __threadfence();
    return last;
}

// Fixed-order sum of partials[0..n) by one block; result valid in thread 0.
__device__ __forceinline__ double sum_partials(const double *partials, int64_t n, double *red)
{
    double s = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += blockDim.x) s += __ldcg(partials + i);
    return block_sum(s, red);
}

// +-v chosen by the low bit of a hop entry (1: +, 0: -)
template <typename T>
__device__ __forceinline__ T signed_by(uint32_t e, T v)
{
    return (e & 1u) ? v : -v;
}

}  // namespace hub
