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

// Sum over the `live` lowest lanes of a warp whose other lanes were never launched (the last warp of a block whose
// size is not a multiple of 32: blockDim = n1^2 * EPB of k_axhelm_line).  The shuffle names only the live lanes and a
// partner's value is added only when that partner exists, so no value of an inactive lane is ever read.  The total
// is valid in lane 0 (the xor butterfly is not closed over a ragged set of lanes); with live == 32 it is warp_sum.
__device__ __forceinline__ double warp_sum_live(double v, int lane, int live)
{
    if (live >= 32) return warp_sum(v);
    const unsigned mask = (1u << live) - 1u;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const int src = lane ^ o;
        const double t = __shfl_sync(mask, v, src < live ? src : lane);
        if (src < live) v += t;
    }
    return v;
}

// sum over the block; result valid in every thread.  red: shared scratch of >= 32 doubles.  Any blockDim.x <= 1024:
// the ragged last warp goes through warp_sum_live, and the per-warp sums are added in ascending warp order by every
// thread (fixed order, no shuffle across warps that may not exist).
__device__ __forceinline__ double block_sum(double v, double* red)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    const int live = min(32, (int)blockDim.x - (wid << 5));
    v = warp_sum_live(v, lane, live);
    __syncthreads();                       // red may still be read from a previous call
    if (lane == 0) red[wid] = v;
    __syncthreads();
    double t = 0.0;
    for (int w = 0; w < nw; ++w) t += red[w];
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
