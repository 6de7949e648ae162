// semb_field_minmax_hist_noalloc: the min / max / histogram consumer (PAPER.md:L171-177 zero-copy hand-off to an
// in-situ consumer) for callers that must not allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc.  The call allocates nothing -- no cudaMalloc, cudaFree, cudaMemset or allocating library routine -- and never touches
// the caller's outputs until the final values are known.
//
// The kernels of the existing path (export.cu) accumulate in the caller's buffers: the order-encoded min / max words live in
// minmax_dev and the 64-bit bin counters in hist_dev, which a memset has to clear first (4 launches + a memset).  The variant here
// keeps those accumulators, and the completion ticket of the last-block hand-off, in ONE file-scope device array of a fixed size
// (g_na_scratch below: 32 832 bytes, held by every GPU that loads the library until the process exits); the last block to finish
// copies the counts and the decoded min / max to the outputs.  Arithmetic is the existing path's, operation for operation (same
// roundings), and all accumulation is on integers or by min / max, so the results are identical bit for bit.
//
// In HOST code the array's name is a host-side stand-in, not a device address; the device address is fetched once per device with
// cudaGetSymbolAddress (na_scratch, below) and passed to the kernels.
//
// Every call shares the array, which keeps the last call's contents: each call clears what must start at zero with a launch of its
// own first.  Calls that OVERLAP on the GPU (two streams, two host threads without an ordering between their launches) race on it.
#include <mutex>
#include <string>

#include "semb_internal.h"

#define NA_HEADER 8                                                   // words before the bins: [0] min, [1] max, [2] ticket
static __device__ __align__(256) unsigned long long g_na_scratch[NA_HEADER + SEMB_NOALLOC_MAX_BINS];

static thread_local std::string g_na_error;
static int na_fail(int code, const std::string& msg) { g_na_error = msg; return code; }
extern "C" SEMB_API const char* semb_noalloc_last_error(void) { return g_na_error.c_str(); }

// device address of g_na_scratch on the CURRENT device; looked up once per device
static int na_scratch(unsigned long long** out)
{
    static std::mutex mtx;
    static unsigned long long* ptr[64] = {nullptr};
    int dev = 0;
    cudaError_t rc = cudaGetDevice(&dev);
    if (rc != cudaSuccess) return na_fail(SEMB_ECUDA, std::string("noalloc: cudaGetDevice: ") + cudaGetErrorString(rc));
    if (dev < 0 || dev >= 64) return na_fail(SEMB_EINVAL, "noalloc: device ordinal above 63");
    std::lock_guard<std::mutex> lock(mtx);
    if (!ptr[dev]) {
        unsigned long long* p = nullptr;
        rc = cudaGetSymbolAddress((void**)&p, g_na_scratch);
        if (rc != cudaSuccess || !p)
            return na_fail(SEMB_ECUDA, std::string("noalloc: cudaGetSymbolAddress(g_na_scratch): ") + cudaGetErrorString(rc));
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return SEMB_OK;
}

// order-preserving map double -> uint64 (so that min / max of doubles are atomicMin / atomicMax of words) and back
__device__ __forceinline__ unsigned long long na_enc(double v)
{
    unsigned long long u = (unsigned long long)__double_as_longlong(v);
    return (u & 0x8000000000000000ull) ? ~u : (u | 0x8000000000000000ull);
}
__device__ __forceinline__ double na_dec(unsigned long long o)
{
    unsigned long long u = (o & 0x8000000000000000ull) ? (o & 0x7fffffffffffffffull) : ~o;
    return __longlong_as_double((long long)u);
}

// what must start at zero: the ticket and the bins; min / max start at their neutral words
static __global__ void k_na_clear(unsigned long long* __restrict__ sc, int nbins)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t == 0) { sc[0] = ~0ull; sc[1] = 0ull; sc[2] = 0ull; }
    if (t < nbins) sc[NA_HEADER + t] = 0ull;
}

// pass 1 of the range-from-data mode: min and max of the field into sc[0], sc[1]
static __global__ void __launch_bounds__(256)
k_na_minmax(int64_t n, int64_t stride, const double* __restrict__ v, unsigned long long* __restrict__ sc)
{
    double mn = INFINITY, mx = -INFINITY;
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const double a = v[l * stride];
        mn = fmin(mn, a); mx = fmax(mx, a);
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
        atomicMin(&sc[0], na_enc(mn)); atomicMax(&sc[1], na_enc(mx));
    }
}

// bin = min(nbins-1, floor((v - lo) * scale)), scale = nbins / (hi - lo); v < lo -> bin 0; subtraction and multiplication rounded
// separately (export.cu: k_minmax_hist, k_hist).  FROM_DATA: [lo, hi] = the [min, max] that k_na_minmax left in sc[0], sc[1];
// otherwise min and max are found in this pass as well.  The last block to finish writes the outputs.
template <bool FROM_DATA>
static __global__ void __launch_bounds__(256)
k_na_hist(int64_t n, int64_t stride, const double* __restrict__ v, int nbins, double lo, double hi, unsigned long long* sc,
          double* __restrict__ minmax_out, unsigned long long* __restrict__ hist_out)
{
    extern __shared__ unsigned int sh[];
    __shared__ double smn[8], smx[8];
    __shared__ unsigned long long ticket;
    for (int b = threadIdx.x; b < nbins; b += blockDim.x) sh[b] = 0u;
    if (FROM_DATA) { lo = na_dec(__ldcg(&sc[0])); hi = na_dec(__ldcg(&sc[1])); }
    const double scale = __ddiv_rn((double)nbins, __dsub_rn(hi, lo));
    __syncthreads();
    double mn = INFINITY, mx = -INFINITY;
    constexpr int U = 8;                                   // values per thread and pass, all loads issued before the first use (export.cu)
    for (int64_t c0 = blockIdx.x * (int64_t)(256 * U); c0 < n; c0 += (int64_t)gridDim.x * (256 * U)) {
        double a[U];
#pragma unroll
        for (int u = 0; u < U; ++u) { const int64_t l = c0 + u * 256 + threadIdx.x; a[u] = (l < n) ? v[l * stride] : 0.0; }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            if (c0 + u * 256 + threadIdx.x < n) {
                if (!FROM_DATA) { mn = fmin(mn, a[u]); mx = fmax(mx, a[u]); }
                const double s = __dmul_rn(__dsub_rn(a[u], lo), scale);
                long long b = (s < 0.0) ? 0ll : (long long)floor(s);
                if (b > nbins - 1) b = nbins - 1;
                atomicAdd(&sh[b], 1u);
            }
        }
    }
    if (!FROM_DATA) {
        for (int o = 16; o > 0; o >>= 1) {
            mn = fmin(mn, __shfl_xor_sync(0xffffffffu, mn, o));
            mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        }
        const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
        if (lane == 0) { smn[wid] = mn; smx[wid] = mx; }
    }
    __syncthreads();
    if (!FROM_DATA && threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { mn = fmin(mn, smn[w]); mx = fmax(mx, smx[w]); }
        atomicMin(&sc[0], na_enc(mn)); atomicMax(&sc[1], na_enc(mx));
    }
    for (int b = threadIdx.x; b < nbins; b += blockDim.x) if (sh[b]) atomicAdd(&sc[NA_HEADER + b], (unsigned long long)sh[b]);
    // hand-off: every thread's updates are visible device-wide before this block takes its ticket
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) ticket = atomicAdd(&sc[2], 1ull);
    __syncthreads();
    if (ticket != (unsigned long long)gridDim.x - 1ull) return;
    __threadfence();
    for (int b = threadIdx.x; b < nbins; b += blockDim.x) hist_out[b] = __ldcg(&sc[NA_HEADER + b]);
    if (threadIdx.x == 0) { minmax_out[0] = na_dec(__ldcg(&sc[0])); minmax_out[1] = na_dec(__ldcg(&sc[1])); }
}

extern "C" SEMB_API int semb_field_minmax_hist_noalloc(const semb_field_desc* f, int nbins, double lo, double hi, double* minmax_dev,
                                                       uint64_t* hist_dev, void* stream)
{
    if (!f || !f->ptr || !minmax_dev || !hist_dev) return na_fail(SEMB_EINVAL, "minmax_hist_noalloc: null argument");
    if (f->memspace != SEMB_MEM_DEVICE || f->dtype != SEMB_F64) return na_fail(SEMB_EINVAL, "minmax_hist_noalloc: the field must be fp64 in device memory");
    if (nbins < 1 || f->count < 1 || f->stride < 1) return na_fail(SEMB_EINVAL, "minmax_hist_noalloc: nbins, count and stride must be >= 1");
    if (nbins > SEMB_NOALLOC_MAX_BINS)
        return na_fail(SEMB_EINVAL, "minmax_hist_noalloc: nbins = " + std::to_string(nbins) + " exceeds the static scratch (SEMB_NOALLOC_MAX_BINS = " +
                                    std::to_string(SEMB_NOALLOC_MAX_BINS) + "); use semb_field_minmax_hist");
    unsigned long long* sc = nullptr;
    int rc = na_scratch(&sc); if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t n = f->count;
    // each block's shared counters are 32-bit: keep every block's share of the input below 2^32
    int64_t blocks = (n + 2047) / 2048; if (blocks > semb_sm_count() * 8) blocks = semb_sm_count() * 8; if (blocks < 1) blocks = 1;
    const size_t smem = sizeof(unsigned int) * (size_t)nbins;
    const double* v = (const double*)f->ptr;
    unsigned long long* hist = (unsigned long long*)hist_dev;
    k_na_clear<<<(nbins + 255) / 256, 256, 0, s>>>(sc, nbins);
    if (lo < hi) {
        k_na_hist<false><<<(unsigned)blocks, 256, smem, s>>>(n, f->stride, v, nbins, lo, hi, sc, minmax_dev, hist);
    } else {
        k_na_minmax<<<(unsigned)blocks, 256, 0, s>>>(n, f->stride, v, sc);
        k_na_hist<true><<<(unsigned)blocks, 256, smem, s>>>(n, f->stride, v, nbins, lo, hi, sc, minmax_dev, hist);
    }
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail(SEMB_ECUDA, std::string("minmax_hist_noalloc: launch: ") + cudaGetErrorString(e));
    return SEMB_OK;
}
