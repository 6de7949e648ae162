// p-multigrid V-cycle preconditioner (§2.2: NekRS preconditions the pressure
// Poisson solve with "p-multigrid ... Chebyshev-accelerated ... smoothers"; the paper gives no formulas, DESIGN.md
// reading R19 fixes them).
//
// Level l re-discretises the SAME elements at order N_l (N_0 = N > N_1 > ...): its coordinates are the level-0
// coordinates interpolated to the order-N_l GLL nodes, and everything else -- geometric factors, numbering,
// gather lists, masks, Jacobi diagonal, axhelm kernels -- is an ordinary semb_mesh built from them, so every
// level runs the same hand-written kernels as the fine problem.
//   prolongation  level l+1 -> l : v_f(i,j,k) = sum_abc J_ia J_jb J_kc v_c(a,b,c),  J_ia = l^(l+1)_a(xi^(l)_i)
//   restriction   level l -> l+1 : r_c = M_c QQ^T_c (J^T x J^T x J^T)(invmult_f o r_f)
//   V(l, r):  last level: z = Cheb_{k_coarse}(r);   else
//             z = Cheb_k(r);  res = r - A z;  z += P V(l+1, R res);  res = r - A z;  z += Cheb_k(res)
// which is symmetric positive definite (same symmetric smoother before and after; oracle pin: dense composition).
#include <math.h>

#include <array>
#include <map>

#include "semb_internal.h"

struct semb_mg {
    int nlevels = 0;
    int orders[8] = {0};
    semb_mesh* lev[8] = {nullptr};       // lev[0] = the owner (not owned), lev[l >= 1] owned
    double* J[8] = {nullptr};            // device [n1_l][n1_{l+1}] row-major, transfer between l+1 and l
    double* W[8][6] = {{nullptr}};       // per level: Chebyshev work (res, d, Ad), residual, A z / second smooth, spare
    double* rc[8] = {nullptr};           // level l >= 1: restricted residual
    double* ec[8] = {nullptr};           // level l >= 1: coarse correction
    std::map<std::pair<uint32_t, double>, std::array<double, 8>> lmax_cache;
    // fp32-storage levels (mg_fp32): float copies of the level data and float work vectors, built on first use
    bool f32_ready = false;
    float* geoF[8] = {nullptr};          // [E][7][Np]
    float* invmultF[8] = {nullptr};
    float* WF[8][6] = {{nullptr}};       // Chebyshev work (res, d, Ad), residual, scratch
    float* rF[8] = {nullptr};            // level l: right-hand side (level 0: the converted PCG residual)
    float* zF[8] = {nullptr};            // level l: result
    // float copies of the level diagonals for the MG_DINVF_CACHE most recently used (tags, lambda) pairs, owned
    struct dinvF_entry { uint32_t tags; double lambda; std::array<float*, 8> d; uint64_t stamp; };
    std::vector<dinvF_entry> dinvF; uint64_t dinvF_clock = 0;
    const float* const* dinvF_cur = nullptr;   // the entry mg_f32_prepare selected for the cycle being enqueued
};

// J[(Nto+1) x (Nfrom+1)]: Lagrange basis of the order-Nfrom GLL nodes at the order-Nto GLL nodes (product formula;
// rows at coinciding end nodes are exact unit vectors, so interpolation keeps exact zeros on Dirichlet faces).
static void interp_matrix_host(int Nfrom, int Nto, double* J)
{
    double xf[SEMB_MAXN1], xt[SEMB_MAXN1], w[SEMB_MAXN1], D[SEMB_MAXN1 * SEMB_MAXN1];
    semb_basis_host(Nfrom, xf, w, D);
    semb_basis_host(Nto, xt, w, D);
    for (int i = 0; i <= Nto; ++i)
        for (int a = 0; a <= Nfrom; ++a) {
            long double v = 1.0L;
            for (int m = 0; m <= Nfrom; ++m)
                if (m != a) v *= ((long double)xt[i] - (long double)xf[m]) / ((long double)xf[a] - (long double)xf[m]);
            J[i * (Nfrom + 1) + a] = (double)v;
        }
}

// One block per element: out = (J x J x J) in  (transpose == 0: J is [nout][nin]) or (J^T x J^T x J^T) in
// (transpose != 0: J is [nin][nout]), by three one-dimensional passes through shared memory.
// scale != NULL: the input is multiplied by scale (restriction: invmult);  accumulate: out += result.
#define MG_MAXNP (SEMB_MAXN1 * SEMB_MAXN1 * SEMB_MAXN1)
// NIN, NOUT > 0: compile-time sizes (the pairs the default hierarchies use; index arithmetic and the inner loops
// unroll); NIN = NOUT = 0: run-time sizes nin, nout.
// EPB elements per block, 128 / EPB threads each (the transfers between the N = 3 and N = 1 levels move 8 <-> 64 nodes per
// element: one block per element was 262 144 blocks of almost no work, 285 us per launch on the bench mesh).
template <int NIN, int NOUT, typename ST, int EPB>
__global__ void __launch_bounds__(128)
k_interp3(int64_t E, int nin_rt, int nout_rt, const double* __restrict__ J, int transpose, const ST* __restrict__ in,
          const ST* __restrict__ scale, ST* __restrict__ out, int accumulate, const semb_scalars* __restrict__ scal)
{
    constexpr int SZ = (NIN > 0) ? ((NIN > NOUT ? NIN : NOUT) * (NIN > NOUT ? NIN : NOUT) * (NIN > NOUT ? NIN : NOUT)) : MG_MAXNP;
    constexpr int SJ = (NIN > 0) ? NIN * NOUT : SEMB_MAXN1 * SEMB_MAXN1;
    constexpr int TPE = 128 / EPB;
    typedef ST CT;                                   // float storage => float arithmetic and half the shared-memory traffic
    __shared__ CT As[EPB * SZ], Bs[EPB * SZ], Js[SJ];
    if (scal && *(volatile const int32_t*)&scal->done) return;
    const int nin = (NIN > 0) ? NIN : nin_rt, nout = (NOUT > 0) ? NOUT : nout_rt;
    const int el = threadIdx.x / TPE, tl = threadIdx.x - el * TPE;
    const int64_t e = blockIdx.x * (int64_t)EPB + el;
    const bool valid = e < E;
    CT* __restrict__ A = As + el * SZ; CT* __restrict__ B = Bs + el * SZ;
    const int npi = nin * nin * nin, npo = nout * nout * nout;
    for (int t = threadIdx.x; t < nin * nout; t += blockDim.x) {
        const int o = t / nin, a = t % nin;                       // Js[o][a] = coefficient of input a in output o
        Js[t] = (CT)(transpose ? J[a * nout + o] : J[o * nin + a]);
    }
    if (valid) for (int t = tl; t < npi; t += TPE) {
        const CT v = in[e * npi + t];
        A[t] = scale ? v * scale[e * npi + t] : v;
    }
    __syncthreads();
    // pass 1 (i): B[c][b][i] = sum_a Js[i][a] A[c][b][a]
    if (valid) for (int t = tl; t < nin * nin * nout; t += TPE) {
        const int i = t % nout, cb = t / nout;
        CT s = (CT)0;
#pragma unroll
        for (int a = 0; a < nin; ++a) s += Js[i * nin + a] * A[cb * nin + a];
        B[t] = s;
    }
    __syncthreads();
    // pass 2 (j): A[c][j][i] = sum_b Js[j][b] B[c][b][i]
    if (valid) for (int t = tl; t < nin * nout * nout; t += TPE) {
        const int i = t % nout, j = (t / nout) % nout, c = t / (nout * nout);
        CT s = (CT)0;
#pragma unroll
        for (int b = 0; b < nin; ++b) s += Js[j * nin + b] * B[(c * nin + b) * nout + i];
        A[t] = s;
    }
    __syncthreads();
    // pass 3 (k): out[k][j][i] = sum_c Js[k][c] A[c][j][i]
    if (valid) for (int t = tl; t < npo; t += TPE) {
        const int ji = t % (nout * nout), k = t / (nout * nout);
        CT s = (CT)0;
#pragma unroll
        for (int c = 0; c < nin; ++c) s += Js[k * nin + c] * A[c * nout * nout + ji];
        if (accumulate) out[e * npo + t] += s; else out[e * npo + t] = s;
    }
}

template <typename ST>
static void interp3_launch(int64_t E, int nin, int nout, const double* J, int transpose, const ST* in, const ST* scale,
                           ST* out, int accumulate, const semb_scalars* scal, cudaStream_t s)
{
#define MG_CASE(A_, B_) if (nin == A_ && nout == B_) { constexpr int EPB = ((A_ > B_ ? A_ : B_) <= 4) ? 8 : 1; \
        k_interp3<A_, B_, ST, EPB><<<(unsigned)((E + EPB - 1) / EPB), 128, 0, s>>>(E, nin, nout, J, transpose, in, scale, out, accumulate, scal); return; }
    MG_CASE(8, 4) MG_CASE(4, 8) MG_CASE(4, 2) MG_CASE(2, 4) MG_CASE(10, 6) MG_CASE(6, 10) MG_CASE(6, 4) MG_CASE(4, 6)
    MG_CASE(8, 2) MG_CASE(10, 4) MG_CASE(10, 2) MG_CASE(6, 2) MG_CASE(2, 6) MG_CASE(8, 6) MG_CASE(6, 8)
#undef MG_CASE
    k_interp3<0, 0, ST, 1><<<(unsigned)E, 128, 0, s>>>(E, nin, nout, J, transpose, in, scale, out, accumulate, scal);
}

// u ~ U[-1,1) per local node from the counter-based splitmix64 of the input recipe (R19)
__global__ void k_mg_random(int64_t n, unsigned long long seed, double* __restrict__ a)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) {
        unsigned long long z = seed + ((unsigned long long)l + 1ull) * 0x9E3779B97F4A7C15ull;
        z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
        z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
        z ^= z >> 31;
        a[l] = (double)(z >> 11) * 0x1.0p-53 * 2.0 - 1.0;
    }
}
#define MG_LMAX_SEED (250113240ull + 900ull)
#define MG_DINVF_CACHE 4
#define MG_LMAX_CACHE 256     // (tags, lambda) pairs whose estimated Chebyshev bounds are remembered (64 B each)
static inline unsigned mg_grid(int64_t n) { int64_t b = (n + 1023) / 1024; const int64_t cap = semb_sm_count() * 8; return (unsigned)(b < 1 ? 1 : (b > cap ? cap : b)); }

static void mg_free(semb_mesh* h, semb_mg* g)
{
    for (int l = 0; l < 8; ++l) {
        semb_dev_free(h, g->J[l]); semb_dev_free(h, g->rc[l]); semb_dev_free(h, g->ec[l]);
        for (int w = 0; w < 6; ++w) semb_dev_free(h, g->W[l][w]);
        for (int w = 0; w < 6; ++w) semb_dev_free(h, g->WF[l][w]);
        semb_dev_free(h, g->geoF[l]); semb_dev_free(h, g->invmultF[l]); semb_dev_free(h, g->rF[l]); semb_dev_free(h, g->zF[l]);
        if (l >= 1 && g->lev[l]) semb_destroy(g->lev[l]);        // frees the level's Schwarz data too
    }
    for (auto& en : g->dinvF) for (float* p : en.d) semb_dev_free(h, p);
    delete g;
}
void semb_mg_destroy_all(semb_mesh* h)
{
    for (semb_mg* g : h->mgs) mg_free(h, g);
    h->mgs.clear();
}

// ---- hierarchy ---------------------------------------------------------------------------------------------
static int mg_build(semb_mesh* h, int nlevels, const int* orders, semb_mg** out, cudaStream_t s)
{
    semb_mg* g = new semb_mg();
    g->nlevels = nlevels;
    for (int l = 0; l < nlevels; ++l) g->orders[l] = orders[l];
    g->lev[0] = h;
    int rc = SEMB_OK;
    do {
        // the caller's x, y, z may be gone after setup: the hierarchy is built from the copy semb_setup kept
        if (!h->xyz) { rc = semb_fail(h, SEMB_EINVAL, "multigrid: the handle holds no coordinates"); break; }
        double Jh[SEMB_MAXN1 * SEMB_MAXN1];
        for (int l = 1; l < nlevels && !rc; ++l) {
            const int nc1 = orders[l] + 1; const int64_t npc = (int64_t)nc1 * nc1 * nc1, nl = h->E * npc;
            double* xyz = (double*)semb_dev_alloc(h, sizeof(double) * 3 * (size_t)nl);
            double* Jd = (double*)semb_dev_alloc(h, sizeof(double) * SEMB_MAXN1 * SEMB_MAXN1);
            if (!xyz || !Jd) { semb_dev_free(h, xyz); semb_dev_free(h, Jd); rc = semb_fail(h, SEMB_ENOMEM, "multigrid: level %d coordinates", l); break; }
            interp_matrix_host(h->N, orders[l], Jh);                                  // [nc1][n1]
            if (cudaMemcpyAsync(Jd, Jh, sizeof(double) * nc1 * h->n1, cudaMemcpyHostToDevice, s) != cudaSuccess) rc = semb_fail(h, SEMB_ECUDA, "multigrid: upload");
            for (int c = 0; c < 3 && !rc; ++c)
                interp3_launch<double>(h->E, h->n1, nc1, Jd, 0, h->xyz + c * h->n, nullptr, xyz + c * nl, 0, nullptr, s);
            if (!rc && cudaStreamSynchronize(s) != cudaSuccess) rc = semb_fail(h, SEMB_ECUDA, "multigrid: coordinate interpolation: %s", cudaGetErrorString(cudaGetLastError()));
            if (!rc) {
                rc = semb_setup(h->E, orders[l], xyz, xyz + nl, xyz + 2 * nl, h->face_tag.data(), h->period,
                                nullptr, h->has_alloc ? &h->alloc : nullptr, (void*)s, &g->lev[l]);
                if (rc) semb_fail(h, rc, "multigrid: setup of level %d (order %d) failed: %s", l, orders[l], semb_last_error(nullptr));
            }
            semb_dev_free(h, xyz); semb_dev_free(h, Jd);
        }
        if (rc) break;
        for (int l = 0; l < nlevels; ++l) {
            semb_mesh* L = g->lev[l];
            for (int w = 0; w < 6; ++w) {
                g->W[l][w] = (double*)semb_dev_alloc(h, sizeof(double) * (size_t)L->n);
                if (!g->W[l][w]) rc = semb_fail(h, SEMB_ENOMEM, "multigrid: work vectors of level %d", l);
            }
            if (l >= 1) {
                g->rc[l] = (double*)semb_dev_alloc(h, sizeof(double) * (size_t)L->n);
                g->ec[l] = (double*)semb_dev_alloc(h, sizeof(double) * (size_t)L->n);
                if (!g->rc[l] || !g->ec[l]) rc = semb_fail(h, SEMB_ENOMEM, "multigrid: vectors of level %d", l);
            }
            if (l + 1 < nlevels) {
                const int nf1 = orders[l] + 1, nc1 = orders[l + 1] + 1;
                g->J[l] = (double*)semb_dev_alloc(h, sizeof(double) * nf1 * nc1);
                if (!g->J[l]) { rc = semb_fail(h, SEMB_ENOMEM, "multigrid: transfer matrix"); break; }
                interp_matrix_host(orders[l + 1], orders[l], Jh);                     // [nf1][nc1]
                if (cudaMemcpy(g->J[l], Jh, sizeof(double) * nf1 * nc1, cudaMemcpyHostToDevice) != cudaSuccess) rc = semb_fail(h, SEMB_ECUDA, "multigrid: upload");
            }
            if (rc) break;
        }
    } while (0);
    if (rc) { mg_free(h, g); return rc; }
    h->mgs.push_back(g);
    *out = g;
    return SEMB_OK;
}

// orders of the hierarchy opts describe (defaults filled in), validated against the mesh order; builds nothing
int semb_mg_orders(semb_mesh* h, const semb_pcg_opts* o, int* nlev_out, int* orders)
{
    int nlev = o->mg_nlevels;
    if (nlev == 0) {
        orders[0] = h->N; nlev = 1;
        if (h->N > 7) orders[nlev++] = 5;          // cfg4 (N = 9): 9, 5, 3, 1 needs 64 iterations, 9, 3, 1 needs 94
        if (h->N > 3) orders[nlev++] = 3;
        if (h->N > 1) orders[nlev++] = 1;
    } else {
        if (nlev < 1 || nlev > 8) return semb_fail(h, SEMB_EINVAL, "multigrid: mg_nlevels = %d", nlev);
        for (int l = 0; l < nlev; ++l) orders[l] = o->mg_orders[l];
    }
    if (orders[0] != h->N) return semb_fail(h, SEMB_EINVAL, "multigrid: mg_orders[0] = %d must be the mesh order %d", orders[0], h->N);
    for (int l = 1; l < nlev; ++l)
        if (orders[l] < 1 || orders[l] >= orders[l - 1]) return semb_fail(h, SEMB_EINVAL, "multigrid: orders must decrease strictly and stay >= 1");
    *nlev_out = nlev;
    return SEMB_OK;
}

int semb_mg_prepare(semb_mesh* h, const semb_pcg_opts* o, semb_mg_ctx* ctx, cudaStream_t s)
{
    int nlev = 0, orders[8];
    { const int rc = semb_mg_orders(h, o, &nlev, orders); if (rc) return rc; }
    semb_mg* g = nullptr;
    for (semb_mg* c : h->mgs) {
        bool same = c->nlevels == nlev;
        for (int l = 0; same && l < nlev; ++l) same = c->orders[l] == orders[l];
        if (same) { g = c; break; }
    }
    if (!g) { int rc = mg_build(h, nlev, orders, &g, s); if (rc) return rc; }
    ctx->mg = g; ctx->lambda = o->lambda; ctx->tags = o->dirichlet_tags;
    ctx->k_smooth = o->mg_smooth_degree > 0 ? o->mg_smooth_degree : 1;
    ctx->k_coarse = o->mg_coarse_degree > 0 ? o->mg_coarse_degree : 32;
    ctx->kind = (o->mg_smoother_kind == 4) ? 4 : 1;
    ctx->fp32 = o->mg_fp32 ? 1 : 0;
    if (ctx->k_smooth > SEMB_MAX_CHEB || ctx->k_coarse > SEMB_MAX_CHEB) return semb_fail(h, SEMB_EINVAL, "multigrid: smoother degree > %d", SEMB_MAX_CHEB);
    ctx->coarse_frac = (o->mg_coarse_lmin_frac > 0.0 && o->mg_coarse_lmin_frac < 1.0) ? o->mg_coarse_lmin_frac : 0.01;
    // Chebyshev bounds per level: given, cached, or estimated (10-step Lanczos x 1.1 from M QQ^T B 1)
    const std::pair<uint32_t, double> key(o->dirichlet_tags, o->lambda);
    auto it = g->lmax_cache.find(key);
    std::array<double, 8> est{};
    if (it != g->lmax_cache.end()) est = it->second;
    bool changed = false;
    for (int l = 0; l < nlev; ++l) {
        if (o->mg_lmax[l] > 0.0) { ctx->lmax[l] = o->mg_lmax[l]; continue; }
        if (!(est[l] > 0.0)) {
            semb_mesh* L = g->lev[l];
            // start vector M QQ^T u, u rough (a smooth start vector underestimates lambda_max badly: R19)
            double* v0 = g->W[l][1];
            semb_mask_entry ml;
            k_mg_random<<<mg_grid(L->n), 256, 0, s>>>(L->n, MG_LMAX_SEED + (unsigned long long)l, v0);
            int rc = semb_gs_launch(L, v0, 1, s);
            if (!rc) rc = semb_get_mask(L, o->dirichlet_tags, &ml, s);
            if (!rc) rc = semb_mask_launch(L, ml, v0, 1, s);
            if (!rc) rc = semb_estimate_lmax(L, o->lambda, o->dirichlet_tags, v0, 10, &est[l], (void*)s);
            if (rc) return semb_fail(h, rc, "multigrid: lambda_max estimate on level %d: %s", l, semb_last_error(L));
            changed = true;
        }
        ctx->lmax[l] = est[l];
    }
    if (changed) {
        if (g->lmax_cache.size() >= MG_LMAX_CACHE) g->lmax_cache.clear();
        g->lmax_cache[key] = est;
    }
    // Schwarz smoother (reading R26) on every level of order >= 2 but the last: subdomain data and lambda_max(S A)
    ctx->schwarz = o->mg_schwarz ? 1 : 0;
    for (int l = 0; l < 8; ++l) { ctx->sz[l] = nullptr; ctx->sz_lmax[l] = 0.0; }
    if (ctx->schwarz) {
        for (int l = 0; l + 1 < nlev; ++l) {
            semb_mesh* L = g->lev[l];
            if (L->N < 2) continue;
            semb_mask_entry ml;
            int rc = semb_get_mask(L, o->dirichlet_tags, &ml, s);
            if (!rc) rc = semb_schwarz_get(L, o->dirichlet_tags, o->mg_fp32 != 0, &ctx->sz[l], s);
            if (!rc) {
                double* v0 = g->W[l][5];
                k_mg_random<<<mg_grid(L->n), 256, 0, s>>>(L->n, MG_LMAX_SEED + (unsigned long long)l, v0);
                rc = semb_gs_launch(L, v0, 1, s);
                if (!rc) rc = semb_mask_launch(L, ml, v0, 1, s);
                double* wk[5] = { g->W[l][0], g->W[l][1], g->W[l][2], g->W[l][3], g->W[l][4] };
                if (!rc) rc = semb_schwarz_lmax(L, ctx->sz[l], o->lambda, ml, v0, 10, wk, &ctx->sz_lmax[l], s);
            }
            if (rc) return semb_fail(h, rc, "multigrid: Schwarz smoother of level %d: %s", l, semb_last_error(L));
        }
    }
    // masks and diagonals of every level for this operator (cached in the level handles)
    for (int l = 0; l < nlev; ++l) {
        semb_mask_entry m; double* dinv;
        int rc = semb_get_mask(g->lev[l], ctx->tags, &m, s);
        if (!rc) rc = semb_get_dinv(g->lev[l], ctx->lambda, ctx->tags, &dinv, s);
        if (rc) return semb_fail(h, rc, "multigrid: level %d: %s", l, semb_last_error(g->lev[l]));
    }
    return SEMB_OK;
}

int64_t semb_mg_level_n(const semb_mg_ctx& ctx, int level)
{
    return (level >= 0 && level < ctx.mg->nlevels) ? ctx.mg->lev[level]->n : -1;
}

int semb_mg_transfer_run(semb_mesh* h, const semb_mg_ctx& ctx, int l, int restrict_, const double* in, double* out, cudaStream_t s)
{
    semb_mg* g = ctx.mg;
    if (l < 0 || l + 1 >= g->nlevels) return semb_fail(h, SEMB_EINVAL, "multigrid: transfer level %d", l);
    semb_mesh* F = g->lev[l]; semb_mesh* C = g->lev[l + 1];
    semb_mask_entry m;
    if (!restrict_) {
        interp3_launch<double>(F->E, C->n1, F->n1, g->J[l], 0, in, nullptr, out, 0, nullptr, s);
        int rc = semb_get_mask(F, ctx.tags, &m, s); if (rc) return rc;
        h->launches += 1;
        return semb_mask_launch(F, m, out, 1, s);
    }
    interp3_launch<double>(F->E, F->n1, C->n1, g->J[l], 1, in, (const double*)F->invmult, out, 0, nullptr, s);
    h->launches += 1;
    int rc = semb_gs_launch(C, out, 1, s); if (rc) return rc;
    rc = semb_get_mask(C, ctx.tags, &m, s); if (rc) return rc;
    return semb_mask_launch(C, m, out, 1, s);
}

// z = V(level, r).  scal (may be NULL): the PCG scalars of the fine handle, only read for the early exit.
static int mg_vcycle_f32_top(semb_mesh* h, const semb_mg_ctx& ctx, const double* r, double* z, semb_scalars* scal, cudaStream_t s);
int semb_mg_vcycle_run(semb_mesh* h, const semb_mg_ctx& ctx, int l, const double* r, double* z, semb_scalars* scal, cudaStream_t s)
{
    if (ctx.fp32 && l == 0) return mg_vcycle_f32_top(h, ctx, r, z, scal, s);
    semb_mg* g = ctx.mg;
    semb_mesh* L = g->lev[l];
    const int64_t n = L->n;
    semb_mask_entry m; double* dinv;
    int rc = semb_get_mask(L, ctx.tags, &m, s); if (rc) return rc;
    rc = semb_get_dinv(L, ctx.lambda, ctx.tags, &dinv, s); if (rc) return rc;
    double *cres = g->W[l][0], *cd = g->W[l][1], *cAd = g->W[l][2], *res = g->W[l][3], *t1 = g->W[l][4];
    const int64_t l0 = L->launches;
    if (l == g->nlevels - 1) {
        const semb_cheb_coef cl = semb_cheb_coefficients(ctx.k_coarse, ctx.lmax[l], ctx.kind, ctx.coarse_frac);
        semb_coarse* ca = nullptr;
        rc = semb_coarse_get(L, &ca, s); if (rc) return rc;
        if (ca) rc = semb_coarse_cheb(L, ca, ctx.lambda, ctx.tags, m, dinv, ctx.k_coarse, cl, r, z, scal, s);       // assembled operator: one launch per step
        else rc = semb_cheb_apply(L, ctx.lambda, m, dinv, ctx.k_coarse, cl, r, z, cres, cd, cAd, scal, false, s);
        if (L != h) { h->launches += L->launches - l0; }
        return rc;
    }
    const semb_cheb_coef cc = semb_cheb_coefficients(ctx.k_smooth, ctx.lmax[l], ctx.kind);
    semb_mesh* C = g->lev[l + 1];
    semb_mask_entry mc;
    rc = semb_get_mask(C, ctx.tags, &mc, s); if (rc) return rc;
    double* spare = g->W[l][5];
    if (ctx.sz[l]) rc = semb_schwarz_cheb4(L, ctx.sz[l], ctx.lambda, m, ctx.k_smooth, ctx.sz_lmax[l], r, z, cres, cd, cAd, spare, scal, s, false);
    else rc = semb_cheb_apply(L, ctx.lambda, m, dinv, ctx.k_smooth, cc, r, z, cres, cd, cAd, scal, false, s);                 // z = S r
    if (rc) return rc;
    rc = semb_residual_launch(L, ctx.lambda, m, z, r, res, t1, scal, s); if (rc) return rc;                                  // res = r - A z
    interp3_launch<double>(L->E, L->n1, C->n1, g->J[l], 1, res, (const double*)L->invmult, g->rc[l + 1], 0, scal, s);               // R res
    rc = semb_gs_launch(C, g->rc[l + 1], 1, s); if (rc) return rc;
    rc = semb_mask_launch(C, mc, g->rc[l + 1], 1, s); if (rc) return rc;
    const int64_t lc0 = C->launches;
    rc = semb_mg_vcycle_run(h, ctx, l + 1, g->rc[l + 1], g->ec[l + 1], scal, s); if (rc) return rc;
    (void)lc0;
    interp3_launch<double>(L->E, C->n1, L->n1, g->J[l], 0, (const double*)g->ec[l + 1], (const double*)nullptr, z, 1, scal, s);                    // z += P e
    rc = semb_residual_launch(L, ctx.lambda, m, z, r, res, t1, scal, s); if (rc) return rc;                                  // res = r - A z
    if (ctx.sz[l]) rc = semb_schwarz_cheb4(L, ctx.sz[l], ctx.lambda, m, ctx.k_smooth, ctx.sz_lmax[l], res, z, cres, cd, cAd, spare, scal, s, true);
    else rc = semb_cheb_apply(L, ctx.lambda, m, dinv, ctx.k_smooth, cc, res, z, cres, cd, cAd, scal, false, s, true);         // z += S res
    if (rc) return rc;
    L->launches += 2;
    if (L != h) h->launches += L->launches - l0;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}


// ---- fp32-storage levels (the preconditioner runs in FP32 "to save on memory bandwidth").  Vectors and
// geometric factors of every level live in float and every level kernel computes in float as well (R21; only the class sums of
// the gather-scatter accumulate in fp64).
template <typename TI, typename TO>
__global__ void k_mg_convert(int64_t n, const TI* __restrict__ in, TO* __restrict__ out, const semb_scalars* __restrict__ scal)
{
    if (scal && *(volatile const int32_t*)&scal->done) return;
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x) out[l] = (TO)in[l];
}

static int mg_f32_prepare(semb_mesh* h, const semb_mg_ctx& ctx, cudaStream_t s)
{
    semb_mg* g = ctx.mg;
    if (!g->f32_ready) {
        for (int l = 0; l < g->nlevels; ++l) {
            semb_mesh* L = g->lev[l];
            const int64_t n = L->n, ng = L->E * 7 * L->Np;
            g->geoF[l] = (float*)semb_dev_alloc(h, sizeof(float) * (size_t)ng);
            g->invmultF[l] = (float*)semb_dev_alloc(h, sizeof(float) * (size_t)n);
            g->rF[l] = (float*)semb_dev_alloc(h, sizeof(float) * (size_t)n);
            g->zF[l] = (float*)semb_dev_alloc(h, sizeof(float) * (size_t)n);
            bool ok = g->geoF[l] && g->invmultF[l] && g->rF[l] && g->zF[l];
            for (int w = 0; w < 6; ++w) { g->WF[l][w] = (float*)semb_dev_alloc(h, sizeof(float) * (size_t)n); ok = ok && g->WF[l][w]; }
            if (!ok) return semb_fail(h, SEMB_ENOMEM, "multigrid: fp32 data of level %d", l);
            k_mg_convert<double, float><<<mg_grid(ng), 256, 0, s>>>(ng, L->geo, g->geoF[l], nullptr);
            k_mg_convert<double, float><<<mg_grid(n), 256, 0, s>>>(n, L->invmult, g->invmultF[l], nullptr);
        }
        SEMB_CUDA(h, cudaGetLastError());
        g->f32_ready = true;
    }
    for (auto& en : g->dinvF)
        if (en.tags == ctx.tags && en.lambda == ctx.lambda) { en.stamp = ++g->dinvF_clock; g->dinvF_cur = en.d.data(); return SEMB_OK; }
    std::array<float*, 8> a{};
    if (g->dinvF.size() >= MG_DINVF_CACHE) {       // reuse the buffers of the least recently used operator
        size_t lru = 0;
        for (size_t q = 1; q < g->dinvF.size(); ++q) if (g->dinvF[q].stamp < g->dinvF[lru].stamp) lru = q;
        SEMB_CUDA(h, cudaStreamSynchronize(s));
        a = g->dinvF[lru].d;
        g->dinvF.erase(g->dinvF.begin() + (long)lru);
    } else {
        for (int l = 0; l < g->nlevels; ++l) {
            a[l] = (float*)semb_dev_alloc(h, sizeof(float) * (size_t)g->lev[l]->n);
            if (!a[l]) { for (float* p : a) semb_dev_free(h, p); return semb_fail(h, SEMB_ENOMEM, "multigrid: fp32 diagonal of level %d", l); }
        }
    }
    int rc = SEMB_OK;
    for (int l = 0; l < g->nlevels && !rc; ++l) {
        semb_mesh* L = g->lev[l];
        double* dinv;
        rc = semb_get_dinv(L, ctx.lambda, ctx.tags, &dinv, s);
        if (!rc) k_mg_convert<double, float><<<mg_grid(L->n), 256, 0, s>>>(L->n, dinv, a[l], nullptr);
    }
    if (!rc && cudaGetLastError() != cudaSuccess) rc = semb_fail(h, SEMB_ECUDA, "multigrid: fp32 diagonals");
    if (rc) { for (float* p : a) semb_dev_free(h, p); return rc; }
    g->dinvF.push_back(semb_mg::dinvF_entry{ctx.tags, ctx.lambda, a, ++g->dinvF_clock});
    g->dinvF_cur = g->dinvF.back().d.data();
    return SEMB_OK;
}

static int mg_vcycle_f32(semb_mesh* h, const semb_mg_ctx& ctx, int l, const float* r, float* z, semb_scalars* scal, cudaStream_t s)
{
    semb_mg* g = ctx.mg;
    semb_mesh* L = g->lev[l];
    semb_mask_entry m;
    int rc = semb_get_mask(L, ctx.tags, &m, s); if (rc) return rc;
    const float* dinv = g->dinvF_cur[l];
    const float* geo = g->geoF[l];
    float *cres = g->WF[l][0], *cd = g->WF[l][1], *cAd = g->WF[l][2], *res = g->WF[l][3], *t1 = g->WF[l][4];
    const int64_t l0 = L->launches;
    if (l == g->nlevels - 1) {
        const semb_cheb_coef cl = semb_cheb_coefficients(ctx.k_coarse, ctx.lmax[l], ctx.kind, ctx.coarse_frac);
        semb_coarse* ca = nullptr;
        rc = semb_coarse_get(L, &ca, s); if (rc) return rc;
        if (ca) rc = semb_coarse_cheb_f(L, ca, ctx.lambda, ctx.tags, m, dinv, ctx.k_coarse, cl, r, z, scal, s);
        else rc = semb_cheb_apply_f(L, ctx.lambda, geo, m, dinv, ctx.k_coarse, cl, r, z, cres, cd, cAd, scal, s, false);
        if (L != h) h->launches += L->launches - l0;
        return rc;
    }
    const semb_cheb_coef cc = semb_cheb_coefficients(ctx.k_smooth, ctx.lmax[l], ctx.kind);
    semb_mesh* C = g->lev[l + 1];
    semb_mask_entry mc;
    rc = semb_get_mask(C, ctx.tags, &mc, s); if (rc) return rc;
    float* spare = g->WF[l][5];
    if (ctx.sz[l]) rc = semb_schwarz_cheb4_f(L, ctx.sz[l], ctx.lambda, geo, m, ctx.k_smooth, ctx.sz_lmax[l], r, z, cres, cd, cAd, spare, scal, s, false);
    else rc = semb_cheb_apply_f(L, ctx.lambda, geo, m, dinv, ctx.k_smooth, cc, r, z, cres, cd, cAd, scal, s, false);           // z = S r
    if (rc) return rc;
    rc = semb_residual_launch_f(L, ctx.lambda, geo, m, z, r, res, t1, scal, s); if (rc) return rc;                                  // res = r - A z
    interp3_launch<float>(L->E, L->n1, C->n1, g->J[l], 1, res, g->invmultF[l], g->rF[l + 1], 0, scal, s);                           // R res
    rc = semb_gs_launch_f(C, g->rF[l + 1], s); if (rc) return rc;
    rc = semb_mask_launch_f(C, mc, g->rF[l + 1], s); if (rc) return rc;
    rc = mg_vcycle_f32(h, ctx, l + 1, g->rF[l + 1], g->zF[l + 1], scal, s); if (rc) return rc;
    interp3_launch<float>(L->E, C->n1, L->n1, g->J[l], 0, (const float*)g->zF[l + 1], (const float*)nullptr, z, 1, scal, s);        // z += P e
    rc = semb_residual_launch_f(L, ctx.lambda, geo, m, z, r, res, t1, scal, s); if (rc) return rc;                                  // res = r - A z
    if (ctx.sz[l]) rc = semb_schwarz_cheb4_f(L, ctx.sz[l], ctx.lambda, geo, m, ctx.k_smooth, ctx.sz_lmax[l], res, z, cres, cd, cAd, spare, scal, s, true);
    else rc = semb_cheb_apply_f(L, ctx.lambda, geo, m, dinv, ctx.k_smooth, cc, res, z, cres, cd, cAd, scal, s, true);          // z += S res
    if (rc) return rc;
    L->launches += 2;
    if (L != h) h->launches += L->launches - l0;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}

// double in, double out, fp32 storage inside
static int mg_vcycle_f32_top(semb_mesh* h, const semb_mg_ctx& ctx, const double* r, double* z, semb_scalars* scal, cudaStream_t s)
{
    semb_mg* g = ctx.mg;
    int rc = mg_f32_prepare(h, ctx, s); if (rc) return rc;
    const int64_t n = h->n;
    k_mg_convert<double, float><<<mg_grid(n), 256, 0, s>>>(n, r, g->rF[0], scal);
    rc = mg_vcycle_f32(h, ctx, 0, g->rF[0], g->zF[0], scal, s); if (rc) return rc;
    k_mg_convert<float, double><<<mg_grid(n), 256, 0, s>>>(n, g->zF[0], z, scal);
    h->launches += 2;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}
