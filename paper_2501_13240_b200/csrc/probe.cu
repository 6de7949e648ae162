// Measurement aid (SURVEY.md §8d "measured read-heavy stream ceiling", H1): a pure streaming kernel with the read : write
// mix of axhelm -- dst[l] = sum_{c < nread} src[c * n + l] -- so that bench.py can state what HBM delivers for a 7 : 1
// stream on this very device next to the 1 : 1 copy figure of MEASURED_PEAKS.json (which the axhelm kernels exceed).
// No method arithmetic; not on the hot path.
#include "semb_internal.h"

// One block per tile of 2048 doubles per stream (the axhelm kernels' shape: one block per element, every load issued
// before the first use), and the same bulk L2 prefetch of the tile `pf` blocks ahead (cp.async.bulk.prefetch.L2, issued by one
// thread) that keeps DRAM busy while the resident blocks wait on their loads.
#define PROBE_TILE 1024        // double2 per stream and block
template <int NR>
__global__ void __launch_bounds__(256)
k_stream_probe(int64_t n2, const double2* __restrict__ src, double2* __restrict__ dst, int pf)
{
    const int64_t t0 = blockIdx.x * (int64_t)PROBE_TILE;
    if (pf > 0 && threadIdx.x == 0) {
        const int64_t tp = t0 + (int64_t)pf * PROBE_TILE;
        if (tp + PROBE_TILE <= n2) {
#pragma unroll
            for (int c = 0; c < NR; ++c)
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(src + c * n2 + tp), "r"((unsigned)(PROBE_TILE * sizeof(double2))) : "memory");
        }
    }
    double2 v[NR][PROBE_TILE / 256];
#pragma unroll
    for (int q = 0; q < PROBE_TILE / 256; ++q) {
        const int64_t l = t0 + q * 256 + threadIdx.x;
#pragma unroll
        for (int c = 0; c < NR; ++c) v[c][q] = (l < n2) ? __ldg(src + c * n2 + l) : make_double2(0.0, 0.0);
    }
#pragma unroll
    for (int q = 0; q < PROBE_TILE / 256; ++q) {
        const int64_t l = t0 + q * 256 + threadIdx.x;
        double2 s = v[0][q];
#pragma unroll
        for (int c = 1; c < NR; ++c) { s.x += v[c][q].x; s.y += v[c][q].y; }
        if (l < n2) dst[l] = s;
    }
}

extern "C" int semb_stream_probe(const double* src, double* dst, int64_t n, int nread, void* stream)
{
    if (!src || !dst || n < 2 || (n & 1) || nread < 1 || nread > 8) return SEMB_EINVAL;
    if (((uintptr_t)src | (uintptr_t)dst) & 15) return SEMB_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t n2 = n / 2;
    const int64_t blocks = (n2 + PROBE_TILE - 1) / PROBE_TILE;
    const int pf = (int)(((int64_t)8 << 20) / ((int64_t)(nread + 1) * PROBE_TILE * 16));      // ~8 MB of traffic ahead, as in axhelm
    const double2* a = (const double2*)src; double2* b = (double2*)dst;
#define PROBE(NR) case NR: k_stream_probe<NR><<<(unsigned)blocks, 256, 0, s>>>(n2, a, b, pf); break;
    switch (nread) { PROBE(1) PROBE(2) PROBE(3) PROBE(4) PROBE(5) PROBE(6) PROBE(7) PROBE(8) }
#undef PROBE
    return cudaGetLastError() == cudaSuccess ? SEMB_OK : SEMB_ECUDA;
}
