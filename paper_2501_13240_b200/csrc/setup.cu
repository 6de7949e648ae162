// Setup-derived data: geometric factors, global numbering, gather lists, inverse
// multiplicity, Dirichlet lists, Jacobi diagonal.  One-off work, all on the device; sorting, scans and
// stream compaction use CUB (toolkit library), everything else is written out here.
//
// PAPER.md:L100 (§2.2): deformed elements through the chain rule -> G, B per node.
// PAPER.md:L102 (§2.2): data on element surfaces is exchanged/summed between elements -> numbering.
// PAPER.md:L238 (§4.1): isothermal / no-slip plates -> Dirichlet lists.
#include <cub/cub.cuh>
#include <math.h>

#include "semb_internal.h"

// ---------------------------------------------------------------------------------------------
// geometric factors: one block per element, coordinates + D staged in shared memory
// geo[e][g][Np], g = G_rr, G_rs, G_rt, G_ss, G_st, G_tt, B   (W = rho_i rho_j rho_k folded in)
__global__ void k_geo(int n1, const double* __restrict__ x, const double* __restrict__ y,
                      const double* __restrict__ z, const double* __restrict__ Dg,
                      const double* __restrict__ rhog, double* __restrict__ geo,
                      unsigned long long* __restrict__ bad)
{
    extern __shared__ double sm[];
    const int Np = n1 * n1 * n1;
    double* sD = sm; double* srho = sD + n1 * n1;
    double* sx = srho + n1; double* sy = sx + Np; double* sz = sy + Np;
    const int64_t e = blockIdx.x;
    for (int t = threadIdx.x; t < n1 * n1; t += blockDim.x) sD[t] = Dg[t];
    for (int t = threadIdx.x; t < n1; t += blockDim.x) srho[t] = rhog[t];
    for (int t = threadIdx.x; t < Np; t += blockDim.x) {
        sx[t] = x[e * Np + t]; sy[t] = y[e * Np + t]; sz[t] = z[e * Np + t];
    }
    __syncthreads();
    double* g = geo + e * 7 * (int64_t)Np;
    for (int l = threadIdx.x; l < Np; l += blockDim.x) {
        const int i = l % n1, j = (l / n1) % n1, k = l / (n1 * n1);
        double xr = 0, xs = 0, xt = 0, yr = 0, ys = 0, yt = 0, zr = 0, zs = 0, zt = 0;
        for (int m = 0; m < n1; ++m) {
            const int ir = k * n1 * n1 + j * n1 + m, is = k * n1 * n1 + m * n1 + i, it = m * n1 * n1 + j * n1 + i;
            const double dr = sD[i * n1 + m], ds = sD[j * n1 + m], dt = sD[k * n1 + m];
            xr += dr * sx[ir]; xs += ds * sx[is]; xt += dt * sx[it];
            yr += dr * sy[ir]; ys += ds * sy[is]; yt += dt * sy[it];
            zr += dr * sz[ir]; zs += ds * sz[is]; zt += dt * sz[it];
        }
        const double J = xr * (ys * zt - yt * zs) - xs * (yr * zt - yt * zr) + xt * (yr * zs - ys * zr);
        if (!(J > 0.0)) atomicMin(bad, (unsigned long long)e);
        const double iJ = 1.0 / J;
        const double rx =  (ys * zt - yt * zs) * iJ, ry = -(xs * zt - xt * zs) * iJ, rz =  (xs * yt - xt * ys) * iJ;
        const double sx_ = -(yr * zt - yt * zr) * iJ, sy_ = (xr * zt - xt * zr) * iJ, sz_ = -(xr * yt - xt * yr) * iJ;
        const double tx =  (yr * zs - ys * zr) * iJ, ty = -(xr * zs - xs * zr) * iJ, tz =  (xr * ys - xs * yr) * iJ;
        const double WJ = srho[i] * srho[j] * srho[k] * J;
        g[0 * Np + l] = WJ * (rx * rx + ry * ry + rz * rz);
        g[1 * Np + l] = WJ * (rx * sx_ + ry * sy_ + rz * sz_);
        g[2 * Np + l] = WJ * (rx * tx + ry * ty + rz * tz);
        g[3 * Np + l] = WJ * (sx_ * sx_ + sy_ * sy_ + sz_ * sz_);
        g[4 * Np + l] = WJ * (sx_ * tx + sy_ * ty + sz_ * tz);
        g[5 * Np + l] = WJ * (tx * tx + ty * ty + tz * tz);
        g[6 * Np + l] = WJ;
    }
}

int semb_setup_geo(semb_mesh* h, const double* x, const double* y, const double* z, cudaStream_t s)
{
    const int n1 = h->n1; const int64_t Np = h->Np;
    h->geo = (double*)semb_dev_alloc(h, sizeof(double) * 7 * (size_t)h->n);
    if (!h->geo) return semb_fail(h, SEMB_ENOMEM, "geo: %zu bytes", sizeof(double) * 7 * (size_t)h->n);
    double* dD = (double*)semb_dev_alloc(h, sizeof(double) * (n1 * n1 + n1) + sizeof(unsigned long long));
    if (!dD) return semb_fail(h, SEMB_ENOMEM, "basis");
    double* drho = dD + n1 * n1; unsigned long long* bad = (unsigned long long*)(drho + n1);
    const unsigned long long none = ~0ull;
    SEMB_CUDA(h, cudaMemcpyAsync(dD, h->D, sizeof(double) * n1 * n1, cudaMemcpyHostToDevice, s));
    SEMB_CUDA(h, cudaMemcpyAsync(drho, h->rho, sizeof(double) * n1, cudaMemcpyHostToDevice, s));
    SEMB_CUDA(h, cudaMemcpyAsync(bad, &none, sizeof(none), cudaMemcpyHostToDevice, s));
    const size_t smem = sizeof(double) * (n1 * n1 + n1 + 3 * Np);
    SEMB_CUDA(h, cudaFuncSetAttribute(k_geo, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_geo<<<(unsigned)h->E, 256, smem, s>>>(n1, x, y, z, dD, drho, h->geo, bad);
    SEMB_CUDA(h, cudaGetLastError());
    unsigned long long b = 0;
    SEMB_CUDA(h, cudaMemcpyAsync(&b, bad, sizeof(b), cudaMemcpyDeviceToHost, s));
    SEMB_CUDA(h, cudaStreamSynchronize(s));
    semb_dev_free(h, dD);
    if (b != none) return semb_fail(h, SEMB_EGEOM, "non-positive Jacobian in element %llu", b);
    return SEMB_OK;
}

// ---------------------------------------------------------------------------------------------
// numbering

// order-preserving map double -> uint64 (for atomicMin / atomicMax on doubles)
__device__ __forceinline__ unsigned long long d2o(double v)
{
    unsigned long long u = (unsigned long long)__double_as_longlong(v);
    return (u & 0x8000000000000000ull) ? ~u : (u | 0x8000000000000000ull);
}
static double o2d_host(unsigned long long o)
{
    unsigned long long u = (o & 0x8000000000000000ull) ? (o & 0x7fffffffffffffffull) : ~o;
    double v; memcpy(&v, &u, 8); return v;
}

// red[0] = min neighbour spacing, red[1..3] = min x,y,z, red[4..6] = max x,y,z  (ordered-uint encoding)
__global__ void k_extent(int64_t n, int n1, const double* __restrict__ x, const double* __restrict__ y,
                         const double* __restrict__ z, unsigned long long* __restrict__ red)
{
    const int Np = n1 * n1 * n1;
    double sp = INFINITY, mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const int loc = (int)(l % Np), i = loc % n1, j = (loc / n1) % n1, k = loc / (n1 * n1);
        const double X = x[l], Y = y[l], Z = z[l];
        mn[0] = fmin(mn[0], X); mn[1] = fmin(mn[1], Y); mn[2] = fmin(mn[2], Z);
        mx[0] = fmax(mx[0], X); mx[1] = fmax(mx[1], Y); mx[2] = fmax(mx[2], Z);
        const int64_t nb[3] = { i + 1 < n1 ? l + 1 : -1, j + 1 < n1 ? l + n1 : -1, k + 1 < n1 ? l + n1 * n1 : -1 };
        for (int d = 0; d < 3; ++d) if (nb[d] >= 0) {
            const double dx = x[nb[d]] - X, dy = y[nb[d]] - Y, dz = z[nb[d]] - Z;
            sp = fmin(sp, sqrt(dx * dx + dy * dy + dz * dz));
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        sp = fmin(sp, __shfl_xor_sync(0xffffffffu, sp, o));
        for (int d = 0; d < 3; ++d) {
            mn[d] = fmin(mn[d], __shfl_xor_sync(0xffffffffu, mn[d], o));
            mx[d] = fmax(mx[d], __shfl_xor_sync(0xffffffffu, mx[d], o));
        }
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMin(&red[0], d2o(sp));
        for (int d = 0; d < 3; ++d) { atomicMin(&red[1 + d], d2o(mn[d])); atomicMax(&red[4 + d], d2o(mx[d])); }
    }
}

struct semb_match {
    double period[3], tol, hc, cmin[3];
    int32_t ns_e;              // candidates per element (surface nodes), or Np when all nodes are candidates
    int32_t Np;
};

__device__ __forceinline__ double wrapc(double c, double period, double tol)
{
    if (period > 0.0) {
        c -= period * floor(c / period);
        if (c >= period - tol) c -= period;       // seam copies land next to 0
    }
    return c;
}

__device__ __forceinline__ int64_t cand_to_local(int64_t s, const semb_match& P, const int32_t* __restrict__ lut)
{
    const int64_t e = s / P.ns_e; const int r = (int)(s - e * P.ns_e);
    return e * P.Np + lut[r];
}

// key of candidate s: 21-bit cell index per direction
__global__ void k_cell_keys(int64_t nc, semb_match P, const int32_t* __restrict__ lut,
                            const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
                            unsigned long long* __restrict__ keys, int32_t* __restrict__ ids)
{
    const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= nc) return;
    const int64_t l = cand_to_local(s, P, lut);
    const double c[3] = { wrapc(x[l], P.period[0], P.tol), wrapc(y[l], P.period[1], P.tol), wrapc(z[l], P.period[2], P.tol) };
    unsigned long long key = 0;
    for (int d = 0; d < 3; ++d) {
        long long q = (long long)floor((c[d] - P.cmin[d]) / P.hc) + 1;     // +1: room for the cell below
        key = (key << 21) | (unsigned long long)(q & 0x1fffff);
    }
    keys[s] = key; ids[s] = (int32_t)l;
}

__device__ __forceinline__ int64_t lower_bound_key(const unsigned long long* __restrict__ keys, int64_t n, unsigned long long key)
{
    int64_t lo = 0, hi = n;
    while (lo < hi) { const int64_t mid = (lo + hi) >> 1; if (keys[mid] < key) lo = mid + 1; else hi = mid; }
    return lo;
}

// label[l] = smallest local index among the candidates whose wrapped coordinates agree with l's within
// tol in every direction.  Candidates are looked up in l's own cell and, only when l lies within tol of a
// cell face, in the cells across that face.
__global__ void k_match(int64_t nc, semb_match P, const unsigned long long* __restrict__ keys,
                        const int32_t* __restrict__ ids, const double* __restrict__ x, const double* __restrict__ y,
                        const double* __restrict__ z, int32_t* __restrict__ label)
{
    const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= nc) return;
    const int32_t l = ids[s];
    const double c[3] = { wrapc(x[l], P.period[0], P.tol), wrapc(y[l], P.period[1], P.tol), wrapc(z[l], P.period[2], P.tol) };
    long long q[3]; int lo[3], hi[3];
    for (int d = 0; d < 3; ++d) {
        q[d] = (long long)floor((c[d] - P.cmin[d]) / P.hc) + 1;
        lo[d] = ((long long)floor((c[d] - 2.0 * P.tol - P.cmin[d]) / P.hc) + 1 < q[d]) ? -1 : 0;
        hi[d] = ((long long)floor((c[d] + 2.0 * P.tol - P.cmin[d]) / P.hc) + 1 > q[d]) ? 1 : 0;
    }
    int32_t best = l;
    for (int ox = lo[0]; ox <= hi[0]; ++ox) for (int oy = lo[1]; oy <= hi[1]; ++oy) for (int oz = lo[2]; oz <= hi[2]; ++oz) {
        const unsigned long long key = ((unsigned long long)((q[0] + ox) & 0x1fffff) << 42) |
                                       ((unsigned long long)((q[1] + oy) & 0x1fffff) << 21) |
                                        (unsigned long long)((q[2] + oz) & 0x1fffff);
        int64_t t;
        if (ox == 0 && oy == 0 && oz == 0) { t = s; while (t > 0 && keys[t - 1] == key) --t; }   // own run
        else t = lower_bound_key(keys, nc, key);
        for (; t < nc && keys[t] == key; ++t) {
            const int32_t l2 = ids[t];
            if (l2 >= best) continue;
            if (fabs(wrapc(x[l2], P.period[0], P.tol) - c[0]) <= P.tol &&
                fabs(wrapc(y[l2], P.period[1], P.tol) - c[1]) <= P.tol &&
                fabs(wrapc(z[l2], P.period[2], P.tol) - c[2]) <= P.tol) best = l2;
        }
    }
    label[l] = best;
}

// caller-supplied ids: label = first local index of the run of equal ids in the (stable) sorted order
__global__ void k_label_from_sorted(int64_t nc, const int32_t* __restrict__ keys, const int32_t* __restrict__ ids,
                                    int32_t* __restrict__ label)
{
    const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= nc) return;
    int64_t t = s; const int32_t key = keys[s];
    while (t > 0 && keys[t - 1] == key) --t;
    label[ids[s]] = ids[t];
}

__global__ void k_iota(int64_t n, int32_t* __restrict__ a)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) a[l] = (int32_t)l;
}

__global__ void k_check_label(int64_t n, const int32_t* __restrict__ label, int* __restrict__ bad)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x)
        if (label[label[l]] != label[l]) *bad = 1;
}

struct is_root_op {
    const int32_t* label;
    __device__ __forceinline__ int32_t operator()(int64_t l) const { return label[l] == (int32_t)l ? 1 : 0; }
};

__global__ void k_gid(int64_t n, const int32_t* __restrict__ label, const int32_t* __restrict__ rank, int32_t* __restrict__ gid)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x)
        gid[l] = rank[label[l]];
}

__global__ void k_gid_keys(int64_t nc, semb_match P, const int32_t* __restrict__ lut, const int32_t* __restrict__ gid,
                           int32_t* __restrict__ keys, int32_t* __restrict__ ids)
{
    const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= nc) return;
    const int64_t l = cand_to_local(s, P, lut);
    keys[s] = gid[l]; ids[s] = (int32_t)l;
}

// shared[s] = 1 if the class of sorted entry s has >= 2 members; head[s] = 1 if s also starts its class
__global__ void k_shared_flags(int64_t nc, const int32_t* __restrict__ keys, int32_t* __restrict__ shared, unsigned char* __restrict__ head)
{
    const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= nc) return;
    const int32_t k = keys[s];
    const bool prev = s > 0 && keys[s - 1] == k, next = s + 1 < nc && keys[s + 1] == k;
    shared[s] = (prev || next) ? 1 : 0;
    head[s] = (!prev && next) ? 1 : 0;
}

__global__ void k_fill(int64_t n, double* __restrict__ a, double v)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) a[l] = v;
}

__global__ void k_invmult(int64_t n_gs, const int32_t* __restrict__ off, const int32_t* __restrict__ ids, double* __restrict__ invmult)
{
    const int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (g >= n_gs) return;
    const int32_t a = off[g], b = off[g + 1];
    const double v = 1.0 / (double)(b - a);
    for (int32_t t = a; t < b; ++t) invmult[ids[t]] = v;
}

// Gather-form code per local node, used by the fused residual / Chebyshev updates (pcg.cu: gs_gathered):
//   -1        the node has no copy (weight 1);
//   <= -2     the node has exactly one copy, at local index -(code + 2) (weight 1/2);
//   >= 3      the node has code copies in all (itself included); such classes (element edges and corners) are
//             assembled in place by k_gs_hi before the fused kernel runs (weight 1/code).
__global__ void k_fill_i32(int64_t n, int32_t* __restrict__ a, int32_t v)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) a[l] = v;
}
__global__ void k_gs_code(int64_t n_gs, const int32_t* __restrict__ off, const int32_t* __restrict__ ids, int32_t* __restrict__ code)
{
    const int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (g >= n_gs) return;
    const int32_t a = off[g], b = off[g + 1], m = b - a;
    if (m == 2) { code[ids[a]] = -(ids[a + 1] + 2); code[ids[a + 1]] = -(ids[a] + 2); return; }
    for (int32_t t = a; t < b; ++t) code[ids[t]] = m;
}
struct gs_hi_pred {
    const int32_t* off;
    __device__ bool operator()(int32_t g) const { return off[g + 1] - off[g] >= 3; }
};

#define GRID1(n) (unsigned)(((n) + 255) / 256)
static inline unsigned grid_stride_blocks(int64_t n) { int64_t b = (n + 255) / 256; const int64_t cap = semb_sm_count() * 16; return (unsigned)(b < cap ? (b > 0 ? b : 1) : cap); }

struct tmp_pool {          // frees every temporary on scope exit
    semb_mesh* h; std::vector<void*> p;
    explicit tmp_pool(semb_mesh* h_) : h(h_) {}
    void* get(size_t bytes) { void* q = semb_dev_alloc(h, bytes ? bytes : 8); if (q) p.push_back(q); return q; }
    ~tmp_pool() { for (void* q : p) semb_dev_free(h, q); }
};
#define TMP(var, type, count)                                                                           \
    type* var = (type*)pool.get(sizeof(type) * (size_t)(count));                                         \
    if (!var) return semb_fail(h, SEMB_ENOMEM, "setup temporary %s: %zu bytes", #var, sizeof(type) * (size_t)(count))

int semb_setup_numbering(semb_mesh* h, const double* x, const double* y, const double* z,
                         const double* period, const int32_t* gid_in, cudaStream_t s)
{
    const int n1 = h->n1, N = h->N; const int64_t Np = h->Np, n = h->n;
    tmp_pool pool(h);
    // ---- tolerance and extent
    TMP(red, unsigned long long, 8);
    {
        unsigned long long init[8];
        for (int i = 0; i < 4; ++i) init[i] = ~0ull;
        for (int i = 4; i < 8; ++i) init[i] = 0ull;
        SEMB_CUDA(h, cudaMemcpyAsync(red, init, sizeof(init), cudaMemcpyHostToDevice, s));
        k_extent<<<grid_stride_blocks(n), 256, 0, s>>>(n, n1, x, y, z, red);
        SEMB_CUDA(h, cudaGetLastError());
        SEMB_CUDA(h, cudaMemcpyAsync(init, red, sizeof(init), cudaMemcpyDeviceToHost, s));
        SEMB_CUDA(h, cudaStreamSynchronize(s));
        semb_match P;
        const double spacing = o2d_host(init[0]);
        P.tol = 1e-8 * spacing;
        h->tol = P.tol;
        double ext = 0.0;
        for (int d = 0; d < 3; ++d) {
            double lo = o2d_host(init[1 + d]), hi = o2d_host(init[4 + d]);
            P.period[d] = period[d];
            if (period[d] > 0.0) { lo = -P.tol; hi = period[d]; }
            P.cmin[d] = lo - 4.0 * P.tol;
            if (hi - lo > ext) ext = hi - lo;
        }
        P.hc = spacing / 4.0;
        if (P.hc < ext / 2.0e6) P.hc = ext / 2.0e6;      // 21 bits per direction
        if (!(P.hc > 16.0 * P.tol)) P.hc = 16.0 * P.tol;
        P.Np = (int32_t)Np;

        // ---- candidate list: element-surface nodes (an element-interior node has no copy), or all nodes
        std::vector<int32_t> lut;
        for (int l = 0; l < Np; ++l) {
            const int i = l % n1, j = (l / n1) % n1, k = l / (n1 * n1);
            if (gid_in || i == 0 || i == N || j == 0 || j == N || k == 0 || k == N) lut.push_back(l);
        }
        P.ns_e = (int32_t)lut.size();
        const int64_t nc = h->E * (int64_t)P.ns_e;
        if (nc >= (int64_t)1 << 31) return semb_fail(h, SEMB_EINVAL, "too many surface nodes for int32 indexing");
        TMP(dlut, int32_t, lut.size());
        SEMB_CUDA(h, cudaMemcpyAsync(dlut, lut.data(), sizeof(int32_t) * lut.size(), cudaMemcpyHostToDevice, s));
        TMP(label, int32_t, n);
        k_iota<<<grid_stride_blocks(n), 256, 0, s>>>(n, label);
        TMP(ids_a, int32_t, nc); TMP(ids_b, int32_t, nc);

        if (!gid_in) {
            TMP(keys_a, unsigned long long, nc); TMP(keys_b, unsigned long long, nc);
            k_cell_keys<<<GRID1(nc), 256, 0, s>>>(nc, P, dlut, x, y, z, keys_a, ids_a);
            size_t tb = 0;
            cub::DeviceRadixSort::SortPairs(nullptr, tb, keys_a, keys_b, ids_a, ids_b, (int)nc, 0, 63, s);
            TMP(tmp, char, tb);
            SEMB_CUDA(h, cub::DeviceRadixSort::SortPairs(tmp, tb, keys_a, keys_b, ids_a, ids_b, (int)nc, 0, 63, s));
            k_match<<<GRID1(nc), 256, 0, s>>>(nc, P, keys_b, ids_b, x, y, z, label);
            SEMB_CUDA(h, cudaGetLastError());
        } else {
            TMP(keys_a, int32_t, nc); TMP(keys_b, int32_t, nc);
            k_gid_keys<<<GRID1(nc), 256, 0, s>>>(nc, P, dlut, gid_in, keys_a, ids_a);
            size_t tb = 0;
            cub::DeviceRadixSort::SortPairs(nullptr, tb, keys_a, keys_b, ids_a, ids_b, (int)nc, 0, 32, s);
            TMP(tmp, char, tb);
            SEMB_CUDA(h, cub::DeviceRadixSort::SortPairs(tmp, tb, keys_a, keys_b, ids_a, ids_b, (int)nc, 0, 32, s));
            k_label_from_sorted<<<GRID1(nc), 256, 0, s>>>(nc, keys_b, ids_b, label);
            SEMB_CUDA(h, cudaGetLastError());
        }
        // ---- "within tol" must be an equivalence relation: every label is its own label
        TMP(badflag, int, 1);
        SEMB_CUDA(h, cudaMemsetAsync(badflag, 0, sizeof(int), s));
        k_check_label<<<grid_stride_blocks(n), 256, 0, s>>>(n, label, badflag);

        // ---- canonical first-touch ids: rank of the class's smallest local index
        h->gid = (int32_t*)semb_dev_alloc(h, sizeof(int32_t) * (size_t)n);
        if (!h->gid) return semb_fail(h, SEMB_ENOMEM, "gid");
        TMP(rank, int32_t, n);
        {
            cub::CountingInputIterator<int64_t> cnt(0);
            cub::TransformInputIterator<int32_t, is_root_op, cub::CountingInputIterator<int64_t>> flags(cnt, is_root_op{label});
            size_t tb = 0;
            cub::DeviceScan::ExclusiveSum(nullptr, tb, flags, rank, (int)n, s);
            TMP(tmp, char, tb);
            SEMB_CUDA(h, cub::DeviceScan::ExclusiveSum(tmp, tb, flags, rank, (int)n, s));   // total = rank[n-1] + flag[n-1]
        }
        k_gid<<<grid_stride_blocks(n), 256, 0, s>>>(n, label, rank, h->gid);
        SEMB_CUDA(h, cudaGetLastError());
        int32_t last_rank = 0, last_label = 0; int bad = 0;
        SEMB_CUDA(h, cudaMemcpyAsync(&last_rank, rank + (n - 1), sizeof(int32_t), cudaMemcpyDeviceToHost, s));
        SEMB_CUDA(h, cudaMemcpyAsync(&last_label, label + (n - 1), sizeof(int32_t), cudaMemcpyDeviceToHost, s));
        SEMB_CUDA(h, cudaMemcpyAsync(&bad, badflag, sizeof(int), cudaMemcpyDeviceToHost, s));
        SEMB_CUDA(h, cudaStreamSynchronize(s));
        if (bad) return semb_fail(h, SEMB_EMATCH, "coordinate matching within tol=%g is not an equivalence relation", P.tol);
        h->n_unique = (int64_t)last_rank + (last_label == (int32_t)(n - 1) ? 1 : 0);

        // ---- gather lists: classes with >= 2 members, by gid, members ascending in l
        TMP(gk_a, int32_t, nc); TMP(gk_b, int32_t, nc);
        k_gid_keys<<<GRID1(nc), 256, 0, s>>>(nc, P, dlut, h->gid, gk_a, ids_a);
        {
            int bits = 1; while (((int64_t)1 << bits) < h->n_unique && bits < 32) ++bits;
            size_t tb = 0;
            cub::DeviceRadixSort::SortPairs(nullptr, tb, gk_a, gk_b, ids_a, ids_b, (int)nc, 0, bits, s);
            TMP(tmp, char, tb);
            SEMB_CUDA(h, cub::DeviceRadixSort::SortPairs(tmp, tb, gk_a, gk_b, ids_a, ids_b, (int)nc, 0, bits, s));
        }
        TMP(shared, int32_t, nc); TMP(head, unsigned char, nc); TMP(pos, int32_t, nc);
        TMP(counts, int64_t, 2);
        k_shared_flags<<<GRID1(nc), 256, 0, s>>>(nc, gk_b, shared, head);
        {
            size_t tb = 0;
            cub::DeviceScan::ExclusiveSum(nullptr, tb, shared, pos, (int)nc, s);
            TMP(tmp, char, tb);
            SEMB_CUDA(h, cub::DeviceScan::ExclusiveSum(tmp, tb, shared, pos, (int)nc, s));
        }
        // n_shared, n_gs by compaction into scratch first (sizes unknown until the select has run)
        TMP(ids_c, int32_t, nc); TMP(off_c, int32_t, nc + 1);
        {
            size_t tb1 = 0, tb2 = 0;
            cub::DeviceSelect::Flagged(nullptr, tb1, ids_b, shared, ids_c, counts, (int)nc, s);
            cub::DeviceSelect::Flagged(nullptr, tb2, pos, head, off_c, counts + 1, (int)nc, s);
            TMP(tmp, char, tb1 > tb2 ? tb1 : tb2);
            SEMB_CUDA(h, cub::DeviceSelect::Flagged(tmp, tb1, ids_b, shared, ids_c, counts, (int)nc, s));
            SEMB_CUDA(h, cub::DeviceSelect::Flagged(tmp, tb2, pos, head, off_c, counts + 1, (int)nc, s));
        }
        int64_t cnt_host[2] = {0, 0};
        SEMB_CUDA(h, cudaMemcpyAsync(cnt_host, counts, sizeof(cnt_host), cudaMemcpyDeviceToHost, s));
        SEMB_CUDA(h, cudaStreamSynchronize(s));
        h->n_shared = cnt_host[0]; h->n_gs = cnt_host[1];
        h->gs_ids = (int32_t*)semb_dev_alloc(h, sizeof(int32_t) * (size_t)(h->n_shared + 1));
        h->gs_off = (int32_t*)semb_dev_alloc(h, sizeof(int32_t) * (size_t)(h->n_gs + 1));
        h->invmult = (double*)semb_dev_alloc(h, sizeof(double) * (size_t)n);
        h->gs_code = (int32_t*)semb_dev_alloc(h, sizeof(int32_t) * (size_t)n);
        if (!h->gs_ids || !h->gs_off || !h->invmult || !h->gs_code) return semb_fail(h, SEMB_ENOMEM, "gather lists");
        SEMB_CUDA(h, cudaMemcpyAsync(h->gs_ids, ids_c, sizeof(int32_t) * (size_t)h->n_shared, cudaMemcpyDeviceToDevice, s));
        SEMB_CUDA(h, cudaMemcpyAsync(h->gs_off, off_c, sizeof(int32_t) * (size_t)h->n_gs, cudaMemcpyDeviceToDevice, s));
        const int32_t nsh = (int32_t)h->n_shared;
        SEMB_CUDA(h, cudaMemcpyAsync(h->gs_off + h->n_gs, &nsh, sizeof(int32_t), cudaMemcpyHostToDevice, s));
        k_fill<<<grid_stride_blocks(n), 256, 0, s>>>(n, h->invmult, 1.0);
        k_fill_i32<<<grid_stride_blocks(n), 256, 0, s>>>(n, h->gs_code, -1);
        if (h->n_gs > 0) {
            k_invmult<<<GRID1(h->n_gs), 256, 0, s>>>(h->n_gs, h->gs_off, h->gs_ids, h->invmult);
            k_gs_code<<<GRID1(h->n_gs), 256, 0, s>>>(h->n_gs, h->gs_off, h->gs_ids, h->gs_code);
            // classes with >= 3 members (ascending class index)
            int32_t* hi_tmp = ids_a;                          // scratch of nc >= n_gs entries, free by now
            cub::CountingInputIterator<int32_t> cls0(0);
            size_t tb = 0;
            cub::DeviceSelect::If(nullptr, tb, cls0, hi_tmp, counts, (int)h->n_gs, gs_hi_pred{h->gs_off}, s);
            TMP(tmp, char, tb);
            SEMB_CUDA(h, cub::DeviceSelect::If(tmp, tb, cls0, hi_tmp, counts, (int)h->n_gs, gs_hi_pred{h->gs_off}, s));
            int64_t nhi = 0;
            SEMB_CUDA(h, cudaMemcpyAsync(&nhi, counts, sizeof(int64_t), cudaMemcpyDeviceToHost, s));
            SEMB_CUDA(h, cudaStreamSynchronize(s));
            h->n_gs_hi = nhi;
            h->gs_hi = (int32_t*)semb_dev_alloc(h, sizeof(int32_t) * (size_t)(nhi + 1));
            if (!h->gs_hi) return semb_fail(h, SEMB_ENOMEM, "gather lists (high-multiplicity classes)");
            SEMB_CUDA(h, cudaMemcpyAsync(h->gs_hi, hi_tmp, sizeof(int32_t) * (size_t)nhi, cudaMemcpyDeviceToDevice, s));
        }
        SEMB_CUDA(h, cudaGetLastError());
        SEMB_CUDA(h, cudaStreamSynchronize(s));
    }
    return SEMB_OK;
}

// ---------------------------------------------------------------------------------------------
// Dirichlet list for a tag set: local nodes whose global node lies on a face with a selected tag
__global__ void k_flag_faces(int64_t E, int n1, const int32_t* __restrict__ face_tag, uint32_t tags,
                             const int32_t* __restrict__ gid, unsigned char* __restrict__ gflag)
{
    const int64_t ef = blockIdx.x;                 // element * 6 + face
    const int64_t e = ef / 6; const int f = (int)(ef % 6);
    const int32_t t = face_tag[ef];
    if (!(t > 0 && t < 32 && ((tags >> t) & 1u))) return;
    const int Np = n1 * n1 * n1, N = n1 - 1;
    for (int q = threadIdx.x; q < n1 * n1; q += blockDim.x) {
        const int a = q % n1, b = q / n1;
        int i, j, k;
        switch (f) {
            case 0: i = 0; j = a; k = b; break;
            case 1: i = N; j = a; k = b; break;
            case 2: i = a; j = 0; k = b; break;
            case 3: i = a; j = N; k = b; break;
            case 4: i = a; j = b; k = 0; break;
            default: i = a; j = b; k = N; break;
        }
        gflag[gid[e * Np + k * n1 * n1 + j * n1 + i]] = 1;
    }
}

__global__ void k_local_flags(int64_t n, const int32_t* __restrict__ gid, const unsigned char* __restrict__ gflag, unsigned char* __restrict__ lflag)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x)
        lflag[l] = gflag[gid[l]];
}

int semb_get_mask(semb_mesh* h, uint32_t tags, semb_mask_entry* out, cudaStream_t s)
{
    auto it = h->masks.find(tags);
    if (it != h->masks.end()) { *out = it->second; return SEMB_OK; }
    semb_mask_entry m;
    bool any = false;
    for (int32_t t : h->face_tag) if (t > 0 && t < 32 && ((tags >> t) & 1u)) { any = true; break; }
    if (any) {
        tmp_pool pool(h);
        const int64_t n = h->n;
        TMP(gflag, unsigned char, h->n_unique); TMP(lflag, unsigned char, n); TMP(list, int32_t, n); TMP(cnt, int64_t, 1);
        SEMB_CUDA(h, cudaMemsetAsync(gflag, 0, (size_t)h->n_unique, s));
        k_flag_faces<<<(unsigned)(h->E * 6), 64, 0, s>>>(h->E, h->n1, h->face_tag_dev, tags, h->gid, gflag);
        k_local_flags<<<grid_stride_blocks(n), 256, 0, s>>>(n, h->gid, gflag, lflag);
        cub::CountingInputIterator<int32_t> iota(0);
        size_t tb = 0;
        cub::DeviceSelect::Flagged(nullptr, tb, iota, lflag, list, cnt, (int)n, s);
        TMP(tmp, char, tb);
        SEMB_CUDA(h, cub::DeviceSelect::Flagged(tmp, tb, iota, lflag, list, cnt, (int)n, s));
        int64_t c = 0;
        SEMB_CUDA(h, cudaMemcpyAsync(&c, cnt, sizeof(c), cudaMemcpyDeviceToHost, s));
        SEMB_CUDA(h, cudaStreamSynchronize(s));
        m.count = c;
        if (c > 0) {
            m.list = (int32_t*)semb_dev_alloc(h, sizeof(int32_t) * (size_t)c);
            if (!m.list) return semb_fail(h, SEMB_ENOMEM, "mask list");
            SEMB_CUDA(h, cudaMemcpyAsync(m.list, list, sizeof(int32_t) * (size_t)c, cudaMemcpyDeviceToDevice, s));
            SEMB_CUDA(h, cudaStreamSynchronize(s));
        }
    }
    h->masks[tags] = m;
    *out = m;
    return SEMB_OK;
}

// ---------------------------------------------------------------------------------------------
// exact diagonal of D^T G D + lambda B per local node:
// d(i,j,k) = sum_m [D_mi^2 G_rr(m,j,k) + D_mj^2 G_ss(i,m,k) + D_mk^2 G_tt(i,j,m)]
//          + 2 [D_ii D_jj G_rs + D_ii D_kk G_rt + D_jj D_kk G_st](i,j,k) + lambda B(i,j,k)
__global__ void k_diag_local(int n1, const double* __restrict__ geo, const double* __restrict__ Dg, double lambda,
                             double* __restrict__ d)
{
    extern __shared__ double sm[];
    const int Np = n1 * n1 * n1;
    double* sD = sm;
    for (int t = threadIdx.x; t < n1 * n1; t += blockDim.x) sD[t] = Dg[t];
    __syncthreads();
    const int64_t e = blockIdx.x;
    const double* g = geo + e * 7 * (int64_t)Np;
    for (int l = threadIdx.x; l < Np; l += blockDim.x) {
        const int i = l % n1, j = (l / n1) % n1, k = l / (n1 * n1);
        double s = 0.0;
        for (int m = 0; m < n1; ++m) {
            s += sD[m * n1 + i] * sD[m * n1 + i] * g[0 * Np + k * n1 * n1 + j * n1 + m];
            s += sD[m * n1 + j] * sD[m * n1 + j] * g[3 * Np + k * n1 * n1 + m * n1 + i];
            s += sD[m * n1 + k] * sD[m * n1 + k] * g[5 * Np + m * n1 * n1 + j * n1 + i];
        }
        s += 2.0 * (sD[i * n1 + i] * sD[j * n1 + j] * g[1 * Np + l] + sD[i * n1 + i] * sD[k * n1 + k] * g[2 * Np + l] +
                    sD[j * n1 + j] * sD[k * n1 + k] * g[4 * Np + l]);
        d[e * Np + l] = s + lambda * g[6 * Np + l];
    }
}

int semb_diag_local(semb_mesh* h, double lambda, double* d, cudaStream_t s)
{
    const int n1 = h->n1;
    double* dD = (double*)semb_dev_alloc(h, sizeof(double) * n1 * n1);
    if (!dD) return semb_fail(h, SEMB_ENOMEM, "diag basis");
    cudaError_t e = cudaMemcpyAsync(dD, h->D, sizeof(double) * n1 * n1, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) {
        k_diag_local<<<(unsigned)h->E, 256, sizeof(double) * n1 * n1, s>>>(n1, h->geo, dD, lambda, d);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    semb_dev_free(h, dD);
    if (e != cudaSuccess) return semb_fail(h, SEMB_ECUDA, "diag_local: %s", cudaGetErrorString(e));
    return SEMB_OK;
}

__global__ void k_set_list(int64_t c, const int32_t* __restrict__ list, double* __restrict__ d, double v)
{
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t < c) d[list[t]] = v;
}

// d = 1 / (dA + lambda dB), 1 at ... (masked nodes are set afterwards by k_set_list)
__global__ void k_dinv_combine(int64_t n, const double* __restrict__ dA, const double* __restrict__ dB, double lambda, double* __restrict__ d)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) d[l] = 1.0 / (dA[l] + lambda * dB[l]);
}
__global__ void k_copy_B(int64_t n, int64_t Np, const double* __restrict__ geo, double* __restrict__ b)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        const int64_t e = l / Np;
        b[l] = geo[e * 7 * Np + 6 * Np + (l - e * Np)];
    }
}

// lambda-independent parts of the assembled diagonal, built once per handle
static int ensure_diag_parts(semb_mesh* h, cudaStream_t s)
{
    if (h->diagA && h->diagB) return SEMB_OK;
    double* a = (double*)semb_dev_alloc(h, sizeof(double) * (size_t)h->n);
    double* b = (double*)semb_dev_alloc(h, sizeof(double) * (size_t)h->n);
    int rc = (a && b) ? SEMB_OK : semb_fail(h, SEMB_ENOMEM, "Jacobi diagonal parts");
    if (!rc) rc = semb_diag_local(h, 0.0, a, s);
    if (!rc) rc = semb_gs_launch(h, a, 1, s);
    if (!rc) {
        k_copy_B<<<grid_stride_blocks(h->n), 256, 0, s>>>(h->n, h->Np, h->geo, b);
        rc = semb_gs_launch(h, b, 1, s);
    }
    if (rc) { semb_dev_free(h, a); semb_dev_free(h, b); return rc; }
    h->diagA = a; h->diagB = b;
    return SEMB_OK;
}

int semb_get_dinv(semb_mesh* h, double lambda, uint32_t tags, double** out, cudaStream_t s)
{
    for (auto& en : h->dinvs)
        if (en.tags == tags && en.lambda == lambda) { en.stamp = ++h->dinv_clock; *out = en.d; return SEMB_OK; }
    semb_mask_entry m;
    int rc = semb_get_mask(h, tags, &m, s); if (rc) return rc;
    rc = ensure_diag_parts(h, s); if (rc) return rc;
    double* d = nullptr;
    if (h->dinvs.size() >= SEMB_DINV_CACHE) {
        // reuse the buffer of the least recently used entry; work already enqueued that reads it must finish first
        size_t lru = 0;
        for (size_t q = 1; q < h->dinvs.size(); ++q) if (h->dinvs[q].stamp < h->dinvs[lru].stamp) lru = q;
        SEMB_CUDA(h, cudaStreamSynchronize(s));
        d = h->dinvs[lru].d;
        h->dinvs.erase(h->dinvs.begin() + (long)lru);
    } else {
        d = (double*)semb_dev_alloc(h, sizeof(double) * (size_t)h->n);
        if (!d) return semb_fail(h, SEMB_ENOMEM, "dinv");
    }
    k_dinv_combine<<<grid_stride_blocks(h->n), 256, 0, s>>>(h->n, h->diagA, h->diagB, lambda, d);
    if (m.count > 0) k_set_list<<<GRID1(m.count), 256, 0, s>>>(m.count, m.list, d, 1.0);
    if (cudaGetLastError() != cudaSuccess) { semb_dev_free(h, d); return semb_fail(h, SEMB_ECUDA, "dinv kernels"); }
    h->dinvs.push_back(semb_dinv_entry{tags, lambda, d, ++h->dinv_clock});
    *out = d;
    return SEMB_OK;
}
