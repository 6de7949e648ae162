// In-situ hand-off (§2.3 zero-copy; L138-159 §3.1 Listing 2: device pointers registered once,
// state/cycle + state/time + publish per analysis step) and the in-device consumer north_star names:
// min / max / histogram of a field, plus the derived field velocity_magnitude.
#include <math.h>

#include "semb_internal.h"

// values per thread and pass, all loads issued before the first use (scalar field / three components); blocks per SM of the grids
#ifndef MH_BPS
#define MH_BPS 8
#endif
#ifndef MH_U1
#define MH_U1 8
#endif
#ifndef MH_U3
#define MH_U3 4
#endif

// |v| = sqrt(fma(vz, vz, fma(vy, vy, vx*vx)))  (reading R11: the fma form is part of the definition)
__global__ void k_vmag(int64_t n, const double* __restrict__ vx, const double* __restrict__ vy,
                       const double* __restrict__ vz, double* __restrict__ out)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const double a = vx[l], b = vy[l], c = vz[l];
        out[l] = sqrt(fma(c, c, fma(b, b, __dmul_rn(a, a))));
    }
}

int semb_vmag_launch(const double* vx, const double* vy, const double* vz, double* out, int64_t n, cudaStream_t s)
{
    int64_t b = (n + 1023) / 1024; if (b > semb_sm_count() * 8) b = semb_sm_count() * 8; if (b < 1) b = 1;
    k_vmag<<<(unsigned)b, 256, 0, s>>>(n, vx, vy, vz, out);
    return cudaGetLastError() == cudaSuccess ? SEMB_OK : SEMB_ECUDA;
}

__device__ __forceinline__ unsigned long long enc(double v)
{
    unsigned long long u = (unsigned long long)__double_as_longlong(v);
    return (u & 0x8000000000000000ull) ? ~u : (u | 0x8000000000000000ull);
}
__device__ __forceinline__ double dec(unsigned long long o)
{
    unsigned long long u = (o & 0x8000000000000000ull) ? (o & 0x7fffffffffffffffull) : ~o;
    return __longlong_as_double((long long)u);
}

__global__ void k_mm_init(unsigned long long* mm) { mm[0] = ~0ull; mm[1] = 0ull; }
__global__ void k_mm_decode(unsigned long long* mm)
{
    const double a = dec(mm[0]), b = dec(mm[1]);
    ((double*)mm)[0] = a; ((double*)mm)[1] = b;
}

__global__ void __launch_bounds__(256)
k_minmax(int64_t n, int64_t stride, const double* __restrict__ v, unsigned long long* __restrict__ mm)
{
    double mn = INFINITY, mx = -INFINITY;
    for (int64_t c0 = blockIdx.x * (int64_t)(256 * MH_U1); c0 < n; c0 += (int64_t)gridDim.x * (256 * MH_U1)) {       // batched loads, as k_minmax_hist
        double a[MH_U1];
#pragma unroll
        for (int u = 0; u < MH_U1; ++u) { const int64_t l = c0 + u * 256 + threadIdx.x; a[u] = (l < n) ? v[l * stride] : NAN; }
#pragma unroll
        for (int u = 0; u < MH_U1; ++u) if (c0 + u * 256 + threadIdx.x < n) { mn = fmin(mn, a[u]); mx = fmax(mx, a[u]); }
    }
    for (int o = 16; o > 0; o >>= 1) {
        mn = fmin(mn, __shfl_xor_sync(0xffffffffu, mn, o));
        mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    __shared__ double smn[8], smx[8];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { smn[wid] = mn; smx[wid] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { mn = fmin(mn, smn[w]); mx = fmax(mx, smx[w]); }
        atomicMin(&mm[0], enc(mn)); atomicMax(&mm[1], enc(mx));
    }
}

// bin = min(nbins-1, floor((v - lo) * scale)), scale = nbins / (hi - lo); v < lo -> bin 0.
// The subtraction and the multiplication are rounded separately (no fused multiply-add).
template <int NV>
__global__ void __launch_bounds__(256)
k_hist(int64_t n, int64_t stride, const double* __restrict__ v, const double* __restrict__ v1, const double* __restrict__ v2, int nbins,
       double lo, double hi, const double* __restrict__ range_dev, unsigned long long* __restrict__ hist)
{
    extern __shared__ unsigned int sh[];
    for (int b = threadIdx.x; b < nbins; b += blockDim.x) sh[b] = 0u;
    if (range_dev) { lo = range_dev[0]; hi = range_dev[1]; }
    const double scale = __ddiv_rn((double)nbins, __dsub_rn(hi, lo));
    __syncthreads();
    constexpr int U = (NV == 3) ? MH_U3 : MH_U1;
    for (int64_t c0 = blockIdx.x * (int64_t)(256 * U); c0 < n; c0 += (int64_t)gridDim.x * (256 * U)) {
        double a[U], b3[NV == 3 ? U : 1], c3[NV == 3 ? U : 1];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t l = c0 + u * 256 + threadIdx.x; const bool ok = l < n;
            a[u] = ok ? v[l * stride] : 0.0;
            if (NV == 3) { b3[u] = ok ? v1[l * stride] : 0.0; c3[u] = ok ? v2[l * stride] : 0.0; }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) if (c0 + u * 256 + threadIdx.x < n) {
            double x = a[u];
            if (NV == 3) x = sqrt(fma(c3[NV == 3 ? u : 0], c3[NV == 3 ? u : 0], fma(b3[NV == 3 ? u : 0], b3[NV == 3 ? u : 0], __dmul_rn(x, x))));
            const double sc = __dmul_rn(__dsub_rn(x, lo), scale);
            long long b = (sc < 0.0) ? 0ll : (long long)floor(sc);
            if (b > nbins - 1) b = nbins - 1;
            atomicAdd(&sh[b], 1u);
        }
    }
    __syncthreads();
    for (int b = threadIdx.x; b < nbins; b += blockDim.x) if (sh[b]) atomicAdd(&hist[b], (unsigned long long)sh[b]);
}

// One pass over the data when the range is known: min, max and the histogram together.  NV = 1: a scalar field; NV = 3: the
// magnitude of a vector field computed on the fly, sqrt(fma(vz, vz, fma(vy, vy, vx vx))) (reading R11), never written to memory.
template <int NV>
__global__ void __launch_bounds__(256)
k_minmax_hist(int64_t n, int64_t stride, const double* __restrict__ v0, const double* __restrict__ v1, const double* __restrict__ v2,
              int nbins, double lo, double hi, unsigned long long* __restrict__ mm, unsigned long long* __restrict__ hist)
{
    extern __shared__ unsigned int sh[];
    for (int b = threadIdx.x; b < nbins; b += blockDim.x) sh[b] = 0u;
    const double scale = __ddiv_rn((double)nbins, __dsub_rn(hi, lo));
    __syncthreads();
    double mn = INFINITY, mx = -INFINITY;
    // MH_U values per thread and pass, all loads issued before the first use: with one 64-bit load in flight per thread the kernel
    // was latency bound at 60 % of the DRAM peak (profiles/r2_consumers_flow.md)
    constexpr int U = (NV == 3) ? MH_U3 : MH_U1;
    for (int64_t c0 = blockIdx.x * (int64_t)(256 * U); c0 < n; c0 += (int64_t)gridDim.x * (256 * U)) {
        double a[U], b3[NV == 3 ? U : 1], c3[NV == 3 ? U : 1];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t l = c0 + u * 256 + threadIdx.x;
            const bool ok = l < n;
            a[u] = ok ? v0[l * stride] : 0.0;
            if (NV == 3) { b3[u] = ok ? v1[l * stride] : 0.0; c3[u] = ok ? v2[l * stride] : 0.0; }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (c0 + u * 256 + threadIdx.x < n) {
                double x = a[u];
                if (NV == 3) x = sqrt(fma(c3[NV == 3 ? u : 0], c3[NV == 3 ? u : 0], fma(b3[NV == 3 ? u : 0], b3[NV == 3 ? u : 0], __dmul_rn(x, x))));
                mn = fmin(mn, x); mx = fmax(mx, x);
                const double sc = __dmul_rn(__dsub_rn(x, lo), scale);
                long long b = (sc < 0.0) ? 0ll : (long long)floor(sc);
                if (b > nbins - 1) b = nbins - 1;
                atomicAdd(&sh[b], 1u);
            }
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        mn = fmin(mn, __shfl_xor_sync(0xffffffffu, mn, o));
        mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    __shared__ double smn[8], smx[8];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { smn[wid] = mn; smx[wid] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { mn = fmin(mn, smn[w]); mx = fmax(mx, smx[w]); }
        atomicMin(&mm[0], enc(mn)); atomicMax(&mm[1], enc(mx));
    }
    for (int b = threadIdx.x; b < nbins; b += blockDim.x) if (sh[b]) atomicAdd(&hist[b], (unsigned long long)sh[b]);
}

// min / max of |v| alone (first pass when the histogram range is to be found on the device)
__global__ void __launch_bounds__(256)
k_minmax_vmag(int64_t n, int64_t stride, const double* __restrict__ v0, const double* __restrict__ v1, const double* __restrict__ v2,
              unsigned long long* __restrict__ mm)
{
    double mn = INFINITY, mx = -INFINITY;
    for (int64_t c0 = blockIdx.x * (int64_t)(256 * MH_U3); c0 < n; c0 += (int64_t)gridDim.x * (256 * MH_U3)) {
        double a0[MH_U3], b[MH_U3], c[MH_U3];
#pragma unroll
        for (int u = 0; u < MH_U3; ++u) {
            const int64_t l = c0 + u * 256 + threadIdx.x; const bool ok = l < n;
            a0[u] = ok ? v0[l * stride] : 0.0; b[u] = ok ? v1[l * stride] : 0.0; c[u] = ok ? v2[l * stride] : 0.0;
        }
#pragma unroll
        for (int u = 0; u < MH_U3; ++u) if (c0 + u * 256 + threadIdx.x < n) {
            const double a = sqrt(fma(c[u], c[u], fma(b[u], b[u], __dmul_rn(a0[u], a0[u]))));
            mn = fmin(mn, a); mx = fmax(mx, a);
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        mn = fmin(mn, __shfl_xor_sync(0xffffffffu, mn, o));
        mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    __shared__ double smn[8], smx[8];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { smn[wid] = mn; smx[wid] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { mn = fmin(mn, smn[w]); mx = fmax(mx, smx[w]); }
        atomicMin(&mm[0], enc(mn)); atomicMax(&mm[1], enc(mx));
    }
}

// v1 == NULL: scalar field v0; else the magnitude of (v0, v1, v2) computed on the fly
int semb_minmax_hist_launch(const double* v, const double* v1, const double* v2, int64_t n, int64_t stride, int nbins, double lo, double hi,
                            double* minmax_dev, uint64_t* hist_dev, cudaStream_t s)
{
    if (nbins < 1 || nbins > 8192 || n < 1 || stride < 1) return SEMB_EINVAL;
    // each block's shared counters are 32-bit: keep every block's share of the input below 2^32
    int64_t blocks = (n + 2047) / 2048; if (blocks > semb_sm_count() * MH_BPS) blocks = semb_sm_count() * MH_BPS; if (blocks < 1) blocks = 1;
    unsigned long long* mm = (unsigned long long*)minmax_dev;
    unsigned long long* hist = (unsigned long long*)hist_dev;
    k_mm_init<<<1, 1, 0, s>>>(mm);
    if (cudaMemsetAsync(hist_dev, 0, sizeof(uint64_t) * nbins, s) != cudaSuccess) return SEMB_ECUDA;
    const size_t smem = sizeof(unsigned int) * nbins;
    if (lo < hi) {                       // range given: ONE pass (8 B/node for a scalar, 24 B/node for a magnitude)
        if (v1) k_minmax_hist<3><<<(unsigned)blocks, 256, smem, s>>>(n, stride, v, v1, v2, nbins, lo, hi, mm, hist);
        else    k_minmax_hist<1><<<(unsigned)blocks, 256, smem, s>>>(n, stride, v, nullptr, nullptr, nbins, lo, hi, mm, hist);
        k_mm_decode<<<1, 1, 0, s>>>(mm);
    } else {                             // range = [min, max] found by a first pass
        if (v1) k_minmax_vmag<<<(unsigned)blocks, 256, 0, s>>>(n, stride, v, v1, v2, mm);
        else    k_minmax<<<(unsigned)blocks, 256, 0, s>>>(n, stride, v, mm);
        k_mm_decode<<<1, 1, 0, s>>>(mm);
        if (v1) k_hist<3><<<(unsigned)blocks, 256, smem, s>>>(n, stride, v, v1, v2, nbins, lo, hi, minmax_dev, hist);
        else    k_hist<1><<<(unsigned)blocks, 256, smem, s>>>(n, stride, v, nullptr, nullptr, nbins, lo, hi, minmax_dev, hist);
    }
    return cudaGetLastError() == cudaSuccess ? SEMB_OK : SEMB_ECUDA;
}
