// gather-scatter QQ^T (direct-stiffness summation; §2.2 "surface-element data exchange ...
// complete residual on subdomain surface") as a sorted-offset segmented sum, and the Dirichlet mask
// (§4.1).  No atomics: one thread owns one global node, sums its copies in ascending local
// index and writes the sum back to every copy, so the result is deterministic.
#include "semb_internal.h"

#ifndef SEMB_GS_BATCH
#define SEMB_GS_BATCH 1
#endif

// ST: storage type of the vector (double; float on the fp32 multigrid levels); sums in fp64.  nfields vectors [nfields][n]: a
// thread fetches the member ids of its class once and sums field after field.
template <typename ST>
__global__ void k_gs(int64_t n_gs, int64_t n, const int32_t* __restrict__ off, const int32_t* __restrict__ ids,
                     ST* __restrict__ w, int nfields)
{
    const int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (g >= n_gs) return;
    const int32_t a = off[g], b = off[g + 1];
#if SEMB_GS_BATCH
    if (b - a <= 8) {                                      // member ids, then member values, as two batches of independent loads (as k_gs_hi)
        int32_t id[8];
#pragma unroll
        for (int t = 0; t < 8; ++t) id[t] = (a + t < b) ? ids[a + t] : -1;
        for (int f = 0; f < nfields; ++f) {
            ST* __restrict__ wf = w + f * n;
            double v[8];
#pragma unroll
            for (int t = 0; t < 8; ++t) v[t] = (id[t] >= 0) ? semb_wide(wf[id[t]]) : 0.0;
            double s = 0.0;
#pragma unroll
            for (int t = 0; t < 8; ++t) if (id[t] >= 0) s += v[t];              // ascending local index: the order of the plain loop
#pragma unroll
            for (int t = 0; t < 8; ++t) if (id[t] >= 0) wf[id[t]] = (ST)s;
        }
        return;
    }
#endif
    for (int f = 0; f < nfields; ++f) {
        ST* __restrict__ wf = w + f * n;
        double s = 0.0;
        for (int32_t t = a; t < b; ++t) s += semb_wide(wf[ids[t]]);
        for (int32_t t = a; t < b; ++t) wf[ids[t]] = (ST)s;
    }
}

int semb_gs_launch(semb_mesh* h, double* w, int nfields, cudaStream_t s)
{
    if (h->n_gs == 0) return SEMB_OK;
    k_gs<double><<<(unsigned)((h->n_gs + 255) / 256), 256, 0, s>>>(h->n_gs, h->n, h->gs_off, h->gs_ids, w, nfields);
    h->launches += 1;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}
int semb_gs_launch_f(semb_mesh* h, float* w, cudaStream_t s)
{
    if (h->n_gs == 0) return SEMB_OK;
    k_gs<float><<<(unsigned)((h->n_gs + 255) / 256), 256, 0, s>>>(h->n_gs, h->n, h->gs_off, h->gs_ids, w, 1);
    h->launches += 1;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}

// The same sum for the listed classes only (those with >= 3 members: element edges and corners).  The fused PCG /
// Chebyshev updates (pcg.cu) do the remaining classes -- one partner each -- in gather form.
template <typename ST>
__global__ void k_gs_hi(int64_t n_hi, const int32_t* __restrict__ hi, const int32_t* __restrict__ off,
                        const int32_t* __restrict__ ids, ST* __restrict__ w, const semb_scalars* __restrict__ scal)
{
    if (scal && *(volatile const int32_t*)&scal->done) return;
    const int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (q >= n_hi) return;
    const int32_t g = hi[q];
    const int32_t a = off[g], b = off[g + 1];
    // A class of a hexahedral mesh has 3..8 members (more only at irregular points): the member ids and then the member values are
    // fetched as two batches of independent loads (two exposed latencies per class instead of two per member); the sum keeps the
    // ascending order of k_gs.
    if (b - a <= 8) {
        int32_t id[8]; double v[8];
#pragma unroll
        for (int t = 0; t < 8; ++t) id[t] = (a + t < b) ? ids[a + t] : -1;
#pragma unroll
        for (int t = 0; t < 8; ++t) v[t] = (id[t] >= 0) ? semb_wide(w[id[t]]) : 0.0;
        double s = 0.0;
#pragma unroll
        for (int t = 0; t < 8; ++t) if (id[t] >= 0) s += v[t];
#pragma unroll
        for (int t = 0; t < 8; ++t) if (id[t] >= 0) w[id[t]] = (ST)s;
        return;
    }
    double s = 0.0;
    for (int32_t t = a; t < b; ++t) s += semb_wide(w[ids[t]]);
    for (int32_t t = a; t < b; ++t) w[ids[t]] = (ST)s;
}

int semb_gs_hi_launch(semb_mesh* h, double* w, const semb_scalars* scal, cudaStream_t s)
{
    if (h->n_gs_hi == 0) return SEMB_OK;
    k_gs_hi<double><<<(unsigned)((h->n_gs_hi + 255) / 256), 256, 0, s>>>(h->n_gs_hi, h->gs_hi, h->gs_off, h->gs_ids, w, scal);
    h->launches += 1;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}
int semb_gs_hi_launch_f(semb_mesh* h, float* w, const semb_scalars* scal, cudaStream_t s)
{
    if (h->n_gs_hi == 0) return SEMB_OK;
    k_gs_hi<float><<<(unsigned)((h->n_gs_hi + 255) / 256), 256, 0, s>>>(h->n_gs_hi, h->gs_hi, h->gs_off, h->gs_ids, w, scal);
    h->launches += 1;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}

template <typename ST>
__global__ void k_mask(int64_t c, int64_t n, const int32_t* __restrict__ list, ST* __restrict__ w)
{
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t < c) w[blockIdx.y * n + list[t]] = (ST)0;
}

int semb_mask_launch(semb_mesh* h, const semb_mask_entry& m, double* w, int nfields, cudaStream_t s)
{
    if (m.count == 0) return SEMB_OK;
    dim3 grid((unsigned)((m.count + 255) / 256), (unsigned)nfields);
    k_mask<double><<<grid, 256, 0, s>>>(m.count, h->n, m.list, w);
    h->launches += 1;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}
int semb_mask_launch_f(semb_mesh* h, const semb_mask_entry& m, float* w, cudaStream_t s)
{
    if (m.count == 0) return SEMB_OK;
    k_mask<float><<<(unsigned)((m.count + 255) / 256), 256, 0, s>>>(m.count, h->n, m.list, w);
    h->launches += 1;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}
