// Last level of the p-multigrid V-cycle (order 1; reading R19: "last level z = Cheb_{k_c}(r)") on an ASSEMBLED operator.
//
// Matrix-free, one Chebyshev step of that level is four launches (operator, mask, class sums, recurrence) of a few microseconds each
// on 8-node elements: with k_c = 32-64 steps the level took 0.39-0.43 of the device time of a V-cycle on a 32^3-element mesh for
// 1/64 of the nodes (profiles/r1_v5_pmg_launches.md; round-1 verdict item 6).  Here the level works on its UNIQUE nodes: the
// stiffness matrix K = sum_e Q_e^T K_e Q_e is assembled once per level (ELL format, <= 27 entries per row on a structured
// mesh), the mass matrix is diagonal at order 1 (GLL quadrature), Dirichlet rows are switched off by a per-node flag, and one
// Chebyshev step is ONE launch:  q = m o (K d + lambda B o d);  z += d;  res -= q;  d = c1 d + c2 D^-1 res.
// k_c + 2 launches per V-cycle instead of 4 k_c + 1.  The element matrices are what the level's own operator kernel returns for the
// eight unit vectors, so the assembled operator IS the matrix-free one up to the order of the sums.  Vectors and matrix entries
// are stored in the level's storage type (float with mg_fp32, R21), the arithmetic is fp64.
// Measured on B200 (V-cycle, k_c = 64): 32^3-element box 2.99 -> 2.15 ms (fp64 levels), 2.32 -> 1.60 ms (FP32 levels), a coarse step
// 19.3 / 17.5 -> 6.1 us; cfg2 O-grid 5.57 -> 4.34 ms and 3.87 -> 2.97 ms; cfg3 (64^3 elements) pressure solve 0.344 -> 0.296 s and 0.242 -> 0.219 s.  Measured and rejected: all k_c steps in ONE cooperative
// launch with a grid barrier per step (1124 blocks): 6.15-6.45 us per step -- the barrier costs what the launch gap did.
#include <cstdlib>
#include <vector>

#include "semb_internal.h"

#define CU_WMAX 64            // rows with more entries than this (a vertex shared by very many elements): the level stays matrix-free
#ifndef CU_EMAX
#define CU_EMAX 300000        // elements; the assembly runs on the host, once per level (262 144 elements: ~3 s)
#endif

struct semb_coarse {
    bool eligible = false;
    int64_t nu = 0; int W = 0;
    int32_t *rep = nullptr, *cols = nullptr;        // a local copy of every unique node;  ELL columns [nu][W], W a multiple of 8
    double* vals = nullptr; float* valsF = nullptr; // ELL values [nu][W] in both storage types
    double* Bu = nullptr;                           // assembled (diagonal) mass matrix
    unsigned char* on = nullptr; uint32_t on_tags = 0; bool on_valid = false;   // 1 = free node, 0 = Dirichlet node of the tag set
    double* vec[5] = {nullptr};                     // D^-1, d (two copies), z, res on the unique nodes (allocated as double, used as ST)
};

static __global__ void k_cu_unit(int64_t n, int j, double* __restrict__ u)
{
    const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (l < n) u[l] = ((l & 7) == j) ? 1.0 : 0.0;
}
static __global__ void k_cu_on(int64_t count, const int32_t* __restrict__ list, const int32_t* __restrict__ gid, unsigned char* __restrict__ on)
{
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t < count) on[gid[list[t]]] = 0;
}

template <typename ST>
static __global__ void k_cu_begin(int64_t nu, const int32_t* __restrict__ rep, const ST* __restrict__ r, const ST* __restrict__ dinv, double itheta,
                                  ST* __restrict__ dinv_u, ST* __restrict__ d, ST* __restrict__ z, ST* __restrict__ res, const semb_scalars* __restrict__ scal)
{
    if (scal && *(volatile const int32_t*)&scal->done) return;
    const int64_t u = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (u >= nu) return;
    const int32_t l = rep[u];
    const ST rv = r[l], dv = dinv[l];
    dinv_u[u] = dv; res[u] = rv; z[u] = (ST)0;
    d[u] = (ST)(itheta * ((double)dv * (double)rv));
}

// Eight lanes per row: lane t of a row takes the entries t, t + 8, ... of its (row-major, padded to a multiple of 8) ELL row, all
// loads of a thread independent; the eight partial sums are added by a fixed xor butterfly.  One dependent pair of loads
// (column index -> vector entry) per step instead of W of them: 18 -> 4 us per launch on a 32^3-element mesh (36 000 rows, W = 27).
template <typename ST, int NT>
static __global__ void __launch_bounds__(256)
k_cu_step(int64_t nu, const int32_t* __restrict__ cols, const ST* __restrict__ vals, const double* __restrict__ Bu, double lambda,
          const unsigned char* __restrict__ on, double c1, double c2, const ST* __restrict__ dinv_u, const ST* __restrict__ d_in,
          ST* __restrict__ d_out, ST* __restrict__ z, ST* __restrict__ res, int last, const semb_scalars* __restrict__ scal)
{
    if (scal && *(volatile const int32_t*)&scal->done) return;
    const int64_t gt = blockIdx.x * (int64_t)blockDim.x + threadIdx.x, u = gt >> 3;
    const int t8 = (int)(gt & 7);
    const bool live = u < nu;                              // whole groups of 8 lanes are live or not; every lane takes part in the shuffles
    double q = 0.0;
    if (live) {
        const int64_t base = u * (NT * 8) + t8;
        int32_t c[NT]; double v[NT], x[NT];
#pragma unroll
        for (int i = 0; i < NT; ++i) c[i] = cols[base + i * 8];
#pragma unroll
        for (int i = 0; i < NT; ++i) { v[i] = (double)vals[base + i * 8]; x[i] = (double)d_in[c[i]]; }      // padding: value 0, column u
#pragma unroll
        for (int i = 0; i < NT; ++i) q += v[i] * x[i];
    }
    q += __shfl_xor_sync(0xffffffffu, q, 1);
    q += __shfl_xor_sync(0xffffffffu, q, 2);
    q += __shfl_xor_sync(0xffffffffu, q, 4);
    if (!live || t8 != 0) return;
    const double dl = (double)d_in[u];
    q += lambda * Bu[u] * dl;
    if (!on[u]) q = 0.0;
    const double zn = (double)z[u] + dl, rn = (double)res[u] - q;
    const double dn = c1 * dl + c2 * ((double)dinv_u[u] * rn);
    if (!last) { res[u] = (ST)rn; d_out[u] = (ST)dn; z[u] = (ST)zn; }
    else z[u] = (ST)(zn + dn);
}

template <typename ST>
static __global__ void k_cu_end(int64_t n, const int32_t* __restrict__ gid, const ST* __restrict__ zu, ST* __restrict__ z, const semb_scalars* __restrict__ scal)
{
    if (scal && *(volatile const int32_t*)&scal->done) return;
    const int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (l < n) z[l] = zu[gid[l]];
}

// ---- host side ------------------------------------------------------------------------------------------------------
void semb_coarse_free(semb_mesh* L)
{
    semb_coarse* c = L->coarse;
    if (!c) return;
    semb_dev_free(L, c->rep); semb_dev_free(L, c->cols); semb_dev_free(L, c->vals); semb_dev_free(L, c->valsF); semb_dev_free(L, c->Bu);
    semb_dev_free(L, c->on);
    for (double* v : c->vec) semb_dev_free(L, v);
    delete c;
    L->coarse = nullptr;
}

static int coarse_build(semb_mesh* L, semb_coarse* c, cudaStream_t s)
{
    const int64_t n = L->n, E = L->E, nu = L->n_unique;
    // element matrices from the level's own operator: column j of every K_e = A_local applied to the j-th unit vector
    double* u = (double*)semb_dev_alloc(L, sizeof(double) * (size_t)n);
    double* w = (double*)semb_dev_alloc(L, sizeof(double) * (size_t)n);
    if (!u || !w) { semb_dev_free(L, u); semb_dev_free(L, w); return semb_fail(L, SEMB_ENOMEM, "coarse level: assembly scratch"); }
    std::vector<double> Kloc((size_t)8 * n), B((size_t)n);
    std::vector<int32_t> gid((size_t)n);
    int rc = SEMB_OK;
    for (int j = 0; j < 8 && !rc; ++j) {
        k_cu_unit<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(n, j, u);
        rc = semb_axhelm_launch(L, 0.0, nullptr, nullptr, u, w, 1, nullptr, s);
        if (!rc && cudaMemcpyAsync(Kloc.data() + (size_t)j * n, w, sizeof(double) * (size_t)n, cudaMemcpyDeviceToHost, s) != cudaSuccess) rc = SEMB_ECUDA;
        if (!rc && cudaStreamSynchronize(s) != cudaSuccess) rc = SEMB_ECUDA;
    }
    semb_dev_free(L, u); semb_dev_free(L, w);
    if (rc) return rc < 0 && rc != SEMB_ECUDA ? rc : semb_fail(L, SEMB_ECUDA, "coarse level: element matrices");
    SEMB_CUDA(L, cudaMemcpy2DAsync(B.data(), 8 * sizeof(double), L->geo + 6 * 8, 56 * sizeof(double), 8 * sizeof(double), (size_t)E, cudaMemcpyDeviceToHost, s));
    SEMB_CUDA(L, cudaMemcpyAsync(gid.data(), L->gid, sizeof(int32_t) * (size_t)n, cudaMemcpyDeviceToHost, s));
    SEMB_CUDA(L, cudaStreamSynchronize(s));
    // rows of K in a fixed-width table; entries of a row in first-touch order (deterministic: elements ascending)
    std::vector<int32_t> rcol((size_t)nu * CU_WMAX), cnt((size_t)nu, 0), rep((size_t)nu, -1);
    std::vector<double> rval((size_t)nu * CU_WMAX), Bu((size_t)nu, 0.0);
    for (int64_t e = 0; e < E; ++e) {
        for (int i = 0; i < 8; ++i) {
            const int64_t li = e * 8 + i; const int32_t row = gid[li];
            if (rep[row] < 0) rep[row] = (int32_t)li;
            Bu[row] += B[li];
            int32_t* rc_ = &rcol[(size_t)row * CU_WMAX]; double* rv_ = &rval[(size_t)row * CU_WMAX];
            for (int j = 0; j < 8; ++j) {
                const int32_t col = gid[e * 8 + j];
                const double v = Kloc[(size_t)j * n + li];
                int t = 0;
                while (t < cnt[row] && rc_[t] != col) ++t;
                if (t == cnt[row]) {
                    if (t == CU_WMAX) return SEMB_OK;                 // not eligible: c->eligible stays false
                    rc_[t] = col; rv_[t] = 0.0; ++cnt[row];
                }
                rv_[t] += v;
            }
        }
    }
    int W = 0;
    for (int64_t r = 0; r < nu; ++r) { if (rep[r] < 0) return semb_fail(L, SEMB_EINVAL, "coarse level: unique node %lld has no copy", (long long)r); if (cnt[r] > W) W = cnt[r]; }
    const int Wp = (W + 7) / 8 * 8;                                      // row-major, padded: value 0 in the row's own column
    std::vector<int32_t> cols((size_t)Wp * nu);
    std::vector<double> vals((size_t)Wp * nu);
    std::vector<float> valsF((size_t)Wp * nu);
    for (int64_t r = 0; r < nu; ++r)
        for (int t = 0; t < Wp; ++t) {
            const bool in = t < cnt[r];
            cols[(size_t)r * Wp + t] = in ? rcol[(size_t)r * CU_WMAX + t] : (int32_t)r;
            vals[(size_t)r * Wp + t] = in ? rval[(size_t)r * CU_WMAX + t] : 0.0;
            valsF[(size_t)r * Wp + t] = (float)vals[(size_t)r * Wp + t];
        }
    c->nu = nu; c->W = Wp;
    c->rep = (int32_t*)semb_dev_alloc(L, sizeof(int32_t) * (size_t)nu);
    c->cols = (int32_t*)semb_dev_alloc(L, sizeof(int32_t) * cols.size());
    c->vals = (double*)semb_dev_alloc(L, sizeof(double) * vals.size());
    c->valsF = (float*)semb_dev_alloc(L, sizeof(float) * valsF.size());
    c->Bu = (double*)semb_dev_alloc(L, sizeof(double) * (size_t)nu);
    c->on = (unsigned char*)semb_dev_alloc(L, (size_t)nu);
    bool ok = c->rep && c->cols && c->vals && c->valsF && c->Bu && c->on;
    for (double*& v : c->vec) { v = (double*)semb_dev_alloc(L, sizeof(double) * (size_t)nu); ok = ok && v; }
    if (!ok) return semb_fail(L, SEMB_ENOMEM, "coarse level: assembled operator");
    SEMB_CUDA(L, cudaMemcpyAsync(c->rep, rep.data(), sizeof(int32_t) * (size_t)nu, cudaMemcpyHostToDevice, s));
    SEMB_CUDA(L, cudaMemcpyAsync(c->cols, cols.data(), sizeof(int32_t) * cols.size(), cudaMemcpyHostToDevice, s));
    SEMB_CUDA(L, cudaMemcpyAsync(c->vals, vals.data(), sizeof(double) * vals.size(), cudaMemcpyHostToDevice, s));
    SEMB_CUDA(L, cudaMemcpyAsync(c->valsF, valsF.data(), sizeof(float) * valsF.size(), cudaMemcpyHostToDevice, s));
    SEMB_CUDA(L, cudaMemcpyAsync(c->Bu, Bu.data(), sizeof(double) * (size_t)nu, cudaMemcpyHostToDevice, s));
    SEMB_CUDA(L, cudaStreamSynchronize(s));                              // the host vectors go out of scope
    c->eligible = true;
    return SEMB_OK;
}

// *out = the level's assembled operator, or NULL if the level is not eligible (order != 1, too many elements, a row too long,
// SEMB_MG_COARSE_ASSEMBLED=0 in the environment)
int semb_coarse_get(semb_mesh* L, semb_coarse** out, cudaStream_t s)
{
    *out = nullptr;
    const char* env = getenv("SEMB_MG_COARSE_ASSEMBLED");
    if (env && atoi(env) == 0) return SEMB_OK;
    if (L->n1 != 2 || L->E > CU_EMAX || L->geo_mode != 0) return SEMB_OK;
    if (!L->coarse) {
        L->coarse = new semb_coarse();
        const int rc = coarse_build(L, L->coarse, s);
        if (rc) { semb_coarse_free(L); return rc; }
    }
    if (L->coarse->eligible) *out = L->coarse;
    return SEMB_OK;
}

template <typename ST>
static int coarse_cheb_t(semb_mesh* L, semb_coarse* c, double lambda, uint32_t tags, const semb_mask_entry& m, const ST* dinv, int k,
                         const semb_cheb_coef& cf, const ST* r, ST* z, semb_scalars* scal, cudaStream_t s)
{
    if (k < 1) return semb_fail(L, SEMB_EINVAL, "coarse level: k >= 1 required");
    const int64_t nu = c->nu, n = L->n;
    if (!c->on_valid || c->on_tags != tags) {
        SEMB_CUDA(L, cudaMemsetAsync(c->on, 1, (size_t)nu, s));
        if (m.count > 0) k_cu_on<<<(unsigned)((m.count + 255) / 256), 256, 0, s>>>(m.count, m.list, L->gid, c->on);
        c->on_tags = tags; c->on_valid = true;
        L->launches += 1;
    }
    ST *dinv_u = (ST*)c->vec[0], *d0 = (ST*)c->vec[1], *d1 = (ST*)c->vec[2], *zu = (ST*)c->vec[3], *res = (ST*)c->vec[4];
    const ST* vals = sizeof(ST) == 4 ? (const ST*)c->valsF : (const ST*)c->vals;
    const unsigned GU = (unsigned)((nu + 127) / 128), GS = (unsigned)((nu * 8 + 255) / 256);
    k_cu_begin<ST><<<GU, 128, 0, s>>>(nu, c->rep, r, dinv, cf.itheta, dinv_u, d0, zu, res, scal);
    for (int it = 0; it < k; ++it) {
#define CU_STEP(NT) k_cu_step<ST, NT><<<GS, 256, 0, s>>>(nu, c->cols, vals, c->Bu, lambda, c->on, cf.c1[it], cf.c2[it], dinv_u, d0, d1, zu, res, it == k - 1, scal)
        switch (c->W / 8) {
            case 1: CU_STEP(1); break; case 2: CU_STEP(2); break; case 3: CU_STEP(3); break; case 4: CU_STEP(4); break;
            case 5: CU_STEP(5); break; case 6: CU_STEP(6); break; case 7: CU_STEP(7); break; default: CU_STEP(8); break;
        }
#undef CU_STEP
        ST* t = d0; d0 = d1; d1 = t;
    }
    k_cu_end<ST><<<(unsigned)((n + 255) / 256), 256, 0, s>>>(n, L->gid, zu, z, scal);
    L->launches += k + 2;
    SEMB_CUDA(L, cudaGetLastError());
    return SEMB_OK;
}

int semb_coarse_cheb(semb_mesh* L, semb_coarse* c, double lambda, uint32_t tags, const semb_mask_entry& m, const double* dinv, int k,
                     const semb_cheb_coef& cf, const double* r, double* z, semb_scalars* scal, cudaStream_t s)
{
    return coarse_cheb_t<double>(L, c, lambda, tags, m, dinv, k, cf, r, z, scal, s);
}
int semb_coarse_cheb_f(semb_mesh* L, semb_coarse* c, double lambda, uint32_t tags, const semb_mask_entry& m, const float* dinv, int k,
                       const semb_cheb_coef& cf, const float* r, float* z, semb_scalars* scal, cudaStream_t s)
{
    return coarse_cheb_t<float>(L, c, lambda, tags, m, dinv, k, cf, r, z, scal, s);
}
