// Deterministic two-stage reductions: warp shuffles -> one value per block -> the LAST block to finish
// (atomic ticket) adds the per-block partials in a fixed order.  The grid of every kernel using this is
// fixed for a given problem, so results are bit-reproducible run to run (reading R14).
#pragma once
#include "semb_internal.h"

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// sum over the block; result valid in every thread.  red: shared scratch of >= 32 doubles.
__device__ __forceinline__ double block_sum(double v, double* red)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    v = warp_sum(v);
    __syncthreads();                       // red may still be read from a previous call
    if (lane == 0) red[wid] = v;
    __syncthreads();
    double t = (lane < nw) ? red[lane] : 0.0;
    t = warp_sum(t);
    return t;
}

// K simultaneous grid-wide sums.  Every block calls this with its block sums v[K] (valid in thread 0 at
// least).  Returns true in ALL threads of the last block to arrive, with tot[K] = the grid totals (valid in
// every thread of that block).  partials: [K][SEMB_MAX_BLOCKS]; *ticket must be 0 on entry and is reset.
template <int K>
__device__ __forceinline__ bool grid_sum(const double (&v)[K], double* __restrict__ partials,
                                         unsigned int* ticket, double (&tot)[K], double* red)
{
    __shared__ int s_last;
    const unsigned nb = gridDim.x * gridDim.y;
    const unsigned bid = blockIdx.y * gridDim.x + blockIdx.x;
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < K; ++k) partials[k * SEMB_MAX_BLOCKS + bid] = v[k];
        __threadfence();
        const unsigned t = atomicAdd(ticket, 1u);
        s_last = (t == nb - 1);
    }
    __syncthreads();
    if (!s_last) return false;
    __threadfence();
#pragma unroll
    for (int k = 0; k < K; ++k) {
        double a = 0.0;
        for (unsigned b = threadIdx.x; b < nb; b += blockDim.x) a += __ldcg(&partials[k * SEMB_MAX_BLOCKS + b]);
        tot[k] = block_sum(a, red);
    }
    if (threadIdx.x == 0) *ticket = 0u;
    return true;
}
