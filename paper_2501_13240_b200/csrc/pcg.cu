// Preconditioned conjugate gradients on the assembled, masked operator A = M QQ^T A_L M with Jacobi or
// Chebyshev-Jacobi preconditioning (BASELINE.json:north_star; §2.2: the pressure Poisson
// solve is the stiffest sub-step, Chebyshev-accelerated smoothers).  Vectors live in local (redundant)
// storage and are continuous; <a,b> = sum_l a_l b_l / mult_l.
//
// alpha, beta, the residual norm, the iteration counter and the stop flag stay in device memory
// (semb_scalars).  Every kernel of the loop returns at once when the stop flag is set, so the host can
// enqueue `check_every` iterations between polls and the iteration count is still exact.
#include <math.h>
#include <string.h>

#include <cooperative_groups.h>

#include <cstdlib>
#include "reduce.cuh"
#include "semb_internal.h"

#define VEC_BLOCK 256
static inline unsigned vec_grid(int64_t n)
{
    int64_t b = (n + VEC_BLOCK * 4 - 1) / (VEC_BLOCK * 4);
    if (b < 1) b = 1;
    if (b > semb_sm_count() * 8) b = semb_sm_count() * 8;
    return (unsigned)b;
}
#define GSTRIDE(l, n) for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < (n); l += (int64_t)gridDim.x * blockDim.x)
#define STOPPED(scal) (*(volatile int32_t*)&(scal)->done)

// Gather form of QQ^T for a vector that is consumed once (SURVEY.md §8 a-2 folded into a-6): the value of
// (QQ^T q) at local node l = sum of q over the copies of l's global node.  q itself is not written back, which
// saves most of the read-modify-write pass of the stand-alone gather-scatter.  A node's code (setup.cu:
// k_gs_code) names its single partner directly (faces: 73 % of the shared nodes at N = 7; the two-term sum is
// the same bits on both copies since a + b == b + a); classes with >= 3 members (element edges and corners,
// 16 % of the nodes) have been summed in place by k_gs_hi just before, in ascending local index like k_gs, and
// carry their multiplicity as code.  The remaining chain code -> q[partner] is one dependent load; the codes of
// the NEXT chunk are fetched while the current one is processed, so a chunk exposes a single memory latency
// like a plain streaming kernel (the first version, which followed per-class records inside this kernel, was
// latency-bound: ncu DRAM 25-33 %, long-scoreboard stalls).  wgt = 1 / multiplicity (bitwise = invmult[l]).
#define GS_U 4
struct gs_lists { const int32_t* code; };
__device__ __forceinline__ void gs_codes(const gs_lists& L, int64_t l0, int64_t n, int32_t (&c)[GS_U])
{
#pragma unroll
    for (int u = 0; u < GS_U; ++u) { const int64_t l = l0 + u * VEC_BLOCK; c[u] = (l < n) ? __ldg(L.code + l) : -1; }
}
// own[u] = q at the node itself (already loaded by the caller, coalesced)
// CT: the type the streaming kernels compute in = their storage type (double; float on the fp32 levels, where widening
// every loaded value to fp64 made the kernel conversion-bound: F2F.F64.F32 is a slow-path instruction, the float
// Chebyshev step took 741 us against 568 us for the double one on 134 M nodes)
template <typename ST, typename CT>
__device__ __forceinline__ void gs_partners(const ST* __restrict__ q, const int32_t (&c)[GS_U], CT (&pv)[GS_U])
{
#pragma unroll
    for (int u = 0; u < GS_U; ++u) pv[u] = (c[u] <= -2) ? (CT)q[-(c[u] + 2)] : (CT)0;
}
template <typename CT>
__device__ __forceinline__ void gs_gathered(const int32_t (&c)[GS_U], const CT (&own)[GS_U], const CT (&pv)[GS_U],
                                            CT (&qa)[GS_U], CT (&wgt)[GS_U])
{
#pragma unroll
    for (int u = 0; u < GS_U; ++u) {
        if (c[u] <= -2) { qa[u] = own[u] + pv[u]; wgt[u] = (CT)0.5; }
        else { qa[u] = own[u]; wgt[u] = (c[u] >= 3) ? (CT)1 / (CT)c[u] : (CT)1; }
    }
}
// grid-stride over chunks of GS_U * VEC_BLOCK nodes; thread t of a block handles nodes l0 + u * VEC_BLOCK
#define GS_STEP ((int64_t)gridDim.x * (GS_U * VEC_BLOCK))
#define GS_CHUNKS(l0, n) for (int64_t l0 = blockIdx.x * (int64_t)(GS_U * VEC_BLOCK) + threadIdx.x; l0 - threadIdx.x < (n); l0 += GS_STEP)

// scal->shift = mean of v over the unique nodes (null_mean: reading R20)
__global__ void __launch_bounds__(VEC_BLOCK)
k_mean(int64_t n, const double* __restrict__ v, const double* __restrict__ invmult, double inv_nu,
       semb_scalars* __restrict__ scal, double* __restrict__ partials)
{
    __shared__ double red[32];
    double s = 0.0;
    GSTRIDE(l, n) s += v[l] * invmult[l];
    double vv[1] = { block_sum(s, red) }, tot[1];
    if (grid_sum<1>(vv, partials, &scal->ticket[4], tot, red) && threadIdx.x == 0) scal->shift = tot[0] * inv_nu;
}
__global__ void __launch_bounds__(VEC_BLOCK)
k_shift(int64_t n, double* __restrict__ v, const semb_scalars* __restrict__ scal)
{
    const double sh = scal->shift;
    GSTRIDE(l, n) v[l] -= sh;
}

// r = b (x = 0) or r = b - q (q = A x0);  bb, rr, rz.  use_shift: b is replaced by b - scal->shift (null_mean)
__global__ void __launch_bounds__(VEC_BLOCK)
k_pcg_init(int64_t n, const double* __restrict__ b, const double* __restrict__ q, double* __restrict__ x,
           double* __restrict__ r, const double* __restrict__ invmult, const double* __restrict__ dinv,
           semb_scalars* __restrict__ scal, double* __restrict__ partials, double* __restrict__ hist, int use_shift)
{
    __shared__ double red[32];
    double bb = 0.0, rr = 0.0, rz = 0.0;
    const double sh = use_shift ? scal->shift : 0.0;
    GSTRIDE(l, n) {
        const double bl = b[l] - sh, w = invmult[l];
        double rl = bl;
        if (q) rl -= q[l]; else x[l] = 0.0;
        r[l] = rl;
        bb += bl * bl * w; rr += rl * rl * w;
        rz += (dinv ? dinv[l] : 1.0) * rl * rl * w;
    }
    double v[3] = { block_sum(bb, red), block_sum(rr, red), block_sum(rz, red) }, tot[3];
    if (grid_sum<3>(v, partials, &scal->ticket[1], tot, red) && threadIdx.x == 0) {
        scal->bnorm = sqrt(tot[0]); scal->rr = tot[1]; scal->rnorm = sqrt(tot[1]); scal->r0norm = scal->rnorm;
        scal->target = fmax(scal->rtol * scal->bnorm, scal->atol);
        scal->rho_old = 0.0; scal->rho_new = tot[2]; scal->rz = tot[2]; scal->beta = 0.0; scal->alpha = 0.0;
        scal->iter = 0; scal->status = SEMB_MAXIT;
        scal->done = 0;
        if (hist) hist[0] = scal->rnorm;
        if (scal->rnorm <= scal->target) { scal->done = 1; scal->status = SEMB_OK; }
    }
}

// r -= alpha QQ^T q (q = M A_L p, masked but not yet assembled: the gather-scatter is done here in gather form);
// rr = <r,r>, rz = <r, dinv r>; the last block closes the iteration.  (x += alpha p and p = z + beta p are done
// by the next fused axhelm launch, which reads p anyway: axhelm_kernels.cuh MODE bit 2.)
template <bool FUSED_Z>
__global__ void __launch_bounds__(VEC_BLOCK, 4)
k_update_r(int64_t n, const double* __restrict__ q, double* __restrict__ r, gs_lists L,
           const double* __restrict__ dinv, semb_scalars* __restrict__ scal, double* __restrict__ partials,
           double* __restrict__ hist, int hist_cap)
{
    __shared__ double red[32];
    if (STOPPED(scal)) return;
    const double alpha = scal->alpha;
    double rr = 0.0, rz = 0.0;
    int32_t cn[GS_U];
    gs_codes(L, blockIdx.x * (int64_t)(GS_U * VEC_BLOCK) + threadIdx.x, n, cn);
    GS_CHUNKS(l0, n) {
        double qa[GS_U], wgt[GS_U], rv[GS_U], dv[GS_U], own[GS_U], pv[GS_U];
        int32_t c[GS_U];
#pragma unroll
        for (int u = 0; u < GS_U; ++u) c[u] = cn[u];
        gs_partners(q, c, pv);
        gs_codes(L, l0 + GS_STEP, n, cn);                       // next chunk's codes, in flight during this one
#pragma unroll
        for (int u = 0; u < GS_U; ++u) {
            const int64_t l = l0 + u * VEC_BLOCK;
            own[u] = (l < n) ? q[l] : 0.0;
            rv[u] = (l < n) ? r[l] : 0.0;
            dv[u] = (FUSED_Z && dinv && l < n) ? dinv[l] : 1.0;
        }
        gs_gathered(c, own, pv, qa, wgt);
#pragma unroll
        for (int u = 0; u < GS_U; ++u) {
            const int64_t l = l0 + u * VEC_BLOCK;
            if (l < n) {
                const double rl = rv[u] - alpha * qa[u];
                r[l] = rl;
                const double t = rl * rl * wgt[u];
                rr += t;
                if (FUSED_Z) rz += dv[u] * t;
            }
        }
    }
    double v[2] = { block_sum(rr, red), block_sum(rz, red) }, tot[2];
    if (grid_sum<2>(v, partials, &scal->ticket[2], tot, red) && threadIdx.x == 0) {
        const int it = scal->iter + 1;
        scal->iter = it;
        scal->rr = tot[0]; scal->rnorm = sqrt(tot[0]);
        if (hist && it < hist_cap) hist[it] = scal->rnorm;
        scal->rho_old = scal->rho_new;
        if (FUSED_Z) { scal->rho_new = tot[1]; scal->rz = tot[1]; scal->beta = tot[1] / scal->rho_old; }
        if (scal->rnorm <= scal->target) { scal->done = 1; scal->status = SEMB_OK; }
        else if (it >= scal->maxit) { scal->done = 1; scal->status = SEMB_MAXIT; }
    }
}

// Small meshes (n <= SEMB_SMALL_N nodes): an iteration of the loop above is five dependent launches of a few microseconds each
// and nothing else (configs[0]: 30 us per iteration for 32 768 nodes, all of it launch latency).  ONE launch does everything that
// follows the operator (a cluster of 8 blocks, hardware cluster barriers between the phases): p.Ap from the per-block partials and alpha; the Dirichlet mask; the class sums of the edge / corner nodes;
// r -= alpha QQ^T q with the face partner gathered; <r,r>, <r,z>; beta and the stop test.  Block-wide barriers replace four kernel
// boundaries; every sum has a fixed order, so the iterates are reproducible run to run.
#define SEMB_SMALL_N 65536
#define SMALL_BLOCK 1024
#define SMALL_CL 8              // blocks of the thread-block cluster that shares the work (hardware cluster barrier between the phases)
template <bool FUSED_Z>
__global__ void __cluster_dims__(SMALL_CL, 1, 1) __launch_bounds__(SMALL_BLOCK)
k_iter_small(int64_t n, int64_t ndot, const double* __restrict__ ax_dot, int64_t nmask, const int32_t* __restrict__ masklist,
             int64_t n_hi, const int32_t* __restrict__ hi, const int32_t* __restrict__ off, const int32_t* __restrict__ ids,
             double* q, double* __restrict__ r, const int32_t* __restrict__ code, const double* __restrict__ dinv,
             semb_scalars* __restrict__ scal, double* __restrict__ partials, double* __restrict__ hist, int hist_cap)
{
    __shared__ double red[32];
    namespace cg = cooperative_groups;
    cg::cluster_group cl = cg::this_cluster();
    if (STOPPED(scal)) return;                                     // uniform over the cluster: written only at the end of an iteration
    const int64_t tid = blockIdx.x * (int64_t)SMALL_BLOCK + threadIdx.x, nthr = (int64_t)SMALL_CL * SMALL_BLOCK;
    double s = 0.0;
    for (int64_t t = threadIdx.x; t < ndot; t += SMALL_BLOCK) s += ax_dot[t];       // every block sums all partials: same order, same bits
    const double pAp = block_sum(s, red);
    if (!(pAp > 0.0) || !isfinite(pAp)) {
        if (tid == 0) { scal->pAp = pAp; scal->status = SEMB_EBREAKDOWN; scal->done = 1; scal->x_pending = 0; }
        return;
    }
    const double alpha = scal->rho_new / pAp;
    for (int64_t t = tid; t < nmask; t += nthr) q[masklist[t]] = 0.0;
    cl.sync();
    for (int64_t t = tid; t < n_hi; t += nthr) {
        const int32_t g = hi[t], a = off[g], b = off[g + 1];
        if (b - a <= 8) {                                          // member ids, then member values, as two batches of independent loads
            int32_t id[8]; double v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) id[u] = (a + u < b) ? ids[a + u] : -1;
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = (id[u] >= 0) ? q[id[u]] : 0.0;
            double c = 0.0;
#pragma unroll
            for (int u = 0; u < 8; ++u) if (id[u] >= 0) c += v[u];
#pragma unroll
            for (int u = 0; u < 8; ++u) if (id[u] >= 0) q[id[u]] = c;
        } else {
            double c = 0.0;
            for (int32_t u = a; u < b; ++u) c += q[ids[u]];
            for (int32_t u = a; u < b; ++u) q[ids[u]] = c;
        }
    }
    cl.sync();
    double rr = 0.0, rz = 0.0;
    for (int64_t l0 = tid; l0 < n; l0 += 4 * nthr) {               // four independent nodes per pass: two exposed latencies
        int32_t c[4]; double own[4], rv[4], dv[4], pv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { const int64_t l = l0 + u * nthr; c[u] = (l < n) ? code[l] : -1; }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int64_t l = l0 + u * nthr;
            own[u] = (l < n) ? q[l] : 0.0; rv[u] = (l < n) ? r[l] : 0.0; dv[u] = (FUSED_Z && dinv && l < n) ? dinv[l] : 1.0;
            pv[u] = (c[u] <= -2) ? q[-(c[u] + 2)] : 0.0;
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int64_t l = l0 + u * nthr;
            if (l < n) {
                const double w = (c[u] <= -2) ? 0.5 : (c[u] >= 3) ? 1.0 / (double)c[u] : 1.0;
                const double rl = rv[u] - alpha * (own[u] + pv[u]);
                r[l] = rl;
                const double t = rl * rl * w;
                rr += t;
                if (FUSED_Z) rz += dv[u] * t;
            }
        }
    }
    rr = block_sum(rr, red);
    rz = block_sum(rz, red);
    if (threadIdx.x == 0) { partials[blockIdx.x] = rr; partials[SEMB_MAX_BLOCKS + blockIdx.x] = rz; }
    cl.sync();
    if (tid == 0) {
        double trr = 0.0, trz = 0.0;
        for (int bq = 0; bq < SMALL_CL; ++bq) { trr += partials[bq]; trz += partials[SEMB_MAX_BLOCKS + bq]; }
        scal->pAp = pAp; scal->alpha = alpha; scal->x_pending = 1;
        const int it = scal->iter + 1;
        scal->iter = it;
        scal->rr = trr; scal->rnorm = sqrt(trr);
        if (hist && it < hist_cap) hist[it] = scal->rnorm;
        scal->rho_old = scal->rho_new;
        if (FUSED_Z) { scal->rho_new = trz; scal->rz = trz; scal->beta = trz / scal->rho_old; }
        if (scal->rnorm <= scal->target) { scal->done = 1; scal->status = SEMB_OK; }
        else if (it >= scal->maxit) { scal->done = 1; scal->status = SEMB_MAXIT; }
    }
}

// the x-update of the last iteration, still pending when the loop stops
__global__ void __launch_bounds__(VEC_BLOCK)
k_final_x(int64_t n, const double* __restrict__ p, double* __restrict__ x, const semb_scalars* __restrict__ scal)
{
    if (!scal->x_pending) return;
    const double alpha = scal->alpha;
    GSTRIDE(l, n) x[l] += alpha * p[l];
}

// rho_new = <r,z>, beta = rho_new / rho_old (0 in the first iteration)   [Chebyshev path]
__global__ void __launch_bounds__(VEC_BLOCK)
k_dot_rz(int64_t n, const double* __restrict__ r, const double* __restrict__ z, const double* __restrict__ invmult,
         semb_scalars* __restrict__ scal, double* __restrict__ partials)
{
    __shared__ double red[32];
    if (STOPPED(scal)) return;
    double s = 0.0;
    GSTRIDE(l, n) s += r[l] * z[l] * invmult[l];
    double v[1] = { block_sum(s, red) }, tot[1];
    if (grid_sum<1>(v, partials, &scal->ticket[3], tot, red) && threadIdx.x == 0) {
        scal->rho_new = tot[0]; scal->rz = tot[0];
        scal->beta = (scal->iter == 0) ? 0.0 : tot[0] / scal->rho_old;
    }
}

// plain weighted dot product into scal->aux (Lanczos, tests)
__global__ void __launch_bounds__(VEC_BLOCK)
k_dot_aux(int64_t n, const double* __restrict__ a, const double* __restrict__ b, const double* __restrict__ invmult,
          semb_scalars* __restrict__ scal, double* __restrict__ partials)
{
    __shared__ double red[32];
    double s = 0.0;
    GSTRIDE(l, n) s += a[l] * b[l] * invmult[l];
    double v[1] = { block_sum(s, red) }, tot[1];
    if (grid_sum<1>(v, partials, &scal->ticket[4], tot, red) && threadIdx.x == 0) scal->aux = tot[0];
}

// ---- Chebyshev-Jacobi(k), 1st-kind recurrence on [0.1 lmax, lmax] (reading R9):
// z = 0; res = r; d = dinv o res / theta; k x { z += d; res -= A d; d = c1 d + c2 dinv o res }; z += d
__global__ void __launch_bounds__(VEC_BLOCK)
k_cheb_init(int64_t n, const double* __restrict__ r, const double* __restrict__ dinv, double itheta,
            double* __restrict__ res, double* __restrict__ d, double* __restrict__ z, int last,
            const semb_scalars* __restrict__ scal)
{
    if (scal && STOPPED(scal)) return;
    GSTRIDE(l, n) {
        const double rl = r[l], dl = dinv[l] * rl * itheta;
        res[l] = rl; d[l] = dl; z[l] = last ? dl : 0.0;
    }
}
// One step of the recurrence.  Ad = M A_L d, masked but not assembled: QQ^T is applied here in gather form.
//   FIRST: res_in is the PCG residual r itself and z is 0 (neither res nor z was initialised: the first d was
//          formed inside the axhelm launch, semb_axhelm_scaled_launch);
//   LAST:  z += d + d_new is final, res and d are dead and not written; with rpcg != NULL the same pass
//          accumulates rho = <rpcg, z> and its last block sets beta (what k_dot_rz did in a pass of its own).
template <bool FIRST, bool LAST, typename ST>
__global__ void __launch_bounds__(VEC_BLOCK, 3)
k_cheb_step(int64_t n, const ST* __restrict__ Ad, gs_lists L, const ST* __restrict__ dinv, double c1, double c2,
            const ST* res_in, ST* res, ST* __restrict__ d, ST* __restrict__ z,
            const double* rpcg, semb_scalars* __restrict__ scal, double* __restrict__ partials, int zacc)
{
    typedef ST CT;
    __shared__ double red[32];
    if (scal && STOPPED(scal)) return;
    int32_t cn[GS_U];
    double rz = 0.0;
    const CT k1 = (CT)c1, k2 = (CT)c2;
    gs_codes(L, blockIdx.x * (int64_t)(GS_U * VEC_BLOCK) + threadIdx.x, n, cn);
    GS_CHUNKS(l0, n) {
        CT qa[GS_U], wgt[GS_U], dl[GS_U], zl[GS_U], rl[GS_U], dv[GS_U], own[GS_U], pv[GS_U];
        double rp[GS_U];
        int32_t c[GS_U];
#pragma unroll
        for (int u = 0; u < GS_U; ++u) c[u] = cn[u];
        gs_partners(Ad, c, pv);
        gs_codes(L, l0 + GS_STEP, n, cn);
#pragma unroll
        for (int u = 0; u < GS_U; ++u) {
            const int64_t l = l0 + u * VEC_BLOCK;
            own[u] = (CT)0; zl[u] = (CT)0; rp[u] = 0.0;
            if (l < n) {
                own[u] = Ad[l]; dl[u] = d[l]; rl[u] = res_in[l]; dv[u] = dinv[l];
                if (!FIRST || zacc) zl[u] = z[l];          // zacc: the smoother's result is ADDED to the z passed in
                if (LAST && !FIRST && rpcg) rp[u] = rpcg[l];
            }
        }
        gs_gathered(c, own, pv, qa, wgt);
#pragma unroll
        for (int u = 0; u < GS_U; ++u) {
            const int64_t l = l0 + u * VEC_BLOCK;
            if (l < n) {
                CT zn = zl[u] + dl[u];
                const CT rn = rl[u] - qa[u];
                const CT dn = k1 * dl[u] + k2 * (dv[u] * rn);
                if (!LAST) { res[l] = rn; d[l] = dn; }
                else {
                    zn += dn;
                    if (rpcg) rz += (FIRST ? (double)rl[u] : rp[u]) * (double)zn * (double)wgt[u];
                }
                z[l] = zn;
            }
        }
    }
    if (LAST && rpcg) {
        double v[1] = { block_sum(rz, red) }, tot[1];
        if (grid_sum<1>(v, partials, &scal->ticket[3], tot, red) && threadIdx.x == 0) {
            scal->rho_new = tot[0]; scal->rz = tot[0];
            scal->beta = (scal->iter == 0) ? 0.0 : tot[0] / scal->rho_old;
        }
    }
}

// ---- small vector kernels for Lanczos / operator application
__global__ void k_copy(int64_t n, const double* __restrict__ a, double* __restrict__ out) { GSTRIDE(l, n) out[l] = a[l]; }
__global__ void k_scale(int64_t n, double c, const double* __restrict__ a, double* __restrict__ out) { GSTRIDE(l, n) out[l] = c * a[l]; }
__global__ void k_sqrt_scale(int64_t n, const double* __restrict__ dinv, const double* __restrict__ a, double* __restrict__ out)
{ GSTRIDE(l, n) out[l] = sqrt(dinv[l]) * a[l]; }
// w = sqrt(dinv) w - bprev vold
__global__ void k_lanczos_a(int64_t n, const double* __restrict__ dinv, double bprev, const double* __restrict__ vold, double* __restrict__ w)
{ GSTRIDE(l, n) w[l] = sqrt(dinv[l]) * w[l] - bprev * vold[l]; }
__global__ void k_axpy(int64_t n, double a, const double* __restrict__ x, double* __restrict__ y) { GSTRIDE(l, n) y[l] += a * x[l]; }

int semb_ensure_work(semb_mesh* h, int64_t vecs)
{
    if (!h->scal) {
        h->scal = (semb_scalars*)semb_dev_alloc(h, sizeof(semb_scalars));
        h->partials = (double*)semb_dev_alloc(h, sizeof(double) * 4 * SEMB_MAX_BLOCKS);
        if (!h->scal || !h->partials) return semb_fail(h, SEMB_ENOMEM, "solver scalars");
        SEMB_CUDA(h, cudaMemset(h->scal, 0, sizeof(semb_scalars)));
        SEMB_CUDA(h, cudaMallocHost((void**)&h->scal_host, sizeof(semb_scalars)));
    }
    if (vecs > h->work_vecs) {
        if (h->work) semb_dev_free(h, h->work);
        h->work = (double*)semb_dev_alloc(h, sizeof(double) * (size_t)vecs * (size_t)h->n);
        if (!h->work) { h->work_vecs = 0; return semb_fail(h, SEMB_ENOMEM, "solver workspace: %lld vectors", (long long)vecs); }
        h->work_vecs = vecs;
    }
    return SEMB_OK;
}

// out = M QQ^T A_L (M v); tmp: one work vector
static int apply_A(semb_mesh* h, double lambda, const semb_mask_entry& m, const double* v_masked, double* out,
                   semb_scalars* scal, cudaStream_t s)
{
    int rc = semb_axhelm_launch(h, lambda, nullptr, nullptr, v_masked, out, 1, scal, s); if (rc) return rc;
    rc = semb_gs_launch(h, out, 1, s); if (rc) return rc;
    return semb_mask_launch(h, m, out, 1, s);
}

// res = r - M QQ^T A_L z  (z continuous and masked; tmp: scratch [n]): the gather-scatter in gather form as in k_update_r
template <typename ST>
__global__ void __launch_bounds__(VEC_BLOCK, 4)
k_residual(int64_t n, const ST* __restrict__ q, gs_lists L, const ST* __restrict__ r, ST* __restrict__ res,
           const semb_scalars* __restrict__ scal)
{
    if (scal && STOPPED(scal)) return;
    int32_t cn[GS_U];
    gs_codes(L, blockIdx.x * (int64_t)(GS_U * VEC_BLOCK) + threadIdx.x, n, cn);
    GS_CHUNKS(l0, n) {
        ST qa[GS_U], wgt[GS_U], rv[GS_U], own[GS_U], pv[GS_U];
        int32_t c[GS_U];
#pragma unroll
        for (int u = 0; u < GS_U; ++u) c[u] = cn[u];
        gs_partners(q, c, pv);
        gs_codes(L, l0 + GS_STEP, n, cn);
#pragma unroll
        for (int u = 0; u < GS_U; ++u) {
            const int64_t l = l0 + u * VEC_BLOCK;
            own[u] = (l < n) ? q[l] : (ST)0;
            rv[u] = (l < n) ? r[l] : (ST)0;
        }
        gs_gathered(c, own, pv, qa, wgt);
#pragma unroll
        for (int u = 0; u < GS_U; ++u) {
            const int64_t l = l0 + u * VEC_BLOCK;
            if (l < n) res[l] = rv[u] - qa[u];
        }
    }
}
int semb_residual_launch(semb_mesh* h, double lambda, const semb_mask_entry& m, const double* z, const double* r, double* res,
                         double* tmp, semb_scalars* scal, cudaStream_t s)
{
    int rc = semb_axhelm_launch(h, lambda, nullptr, nullptr, z, tmp, 1, nullptr, s); if (rc) return rc;
    rc = semb_mask_launch(h, m, tmp, 1, s); if (rc) return rc;
    rc = semb_gs_hi_launch(h, tmp, scal, s); if (rc) return rc;
    k_residual<double><<<vec_grid(h->n), VEC_BLOCK, 0, s>>>(h->n, tmp, gs_lists{h->gs_code}, r, res, scal);
    h->launches += 1;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}

// ---- fp32-storage variants for the multigrid levels (mg.cu): same kernels, float vectors, float arithmetic (R21)
int semb_residual_launch_f(semb_mesh* h, double lambda, const float* geo, const semb_mask_entry& m, const float* z, const float* r,
                           float* res, float* tmp, semb_scalars* scal, cudaStream_t s)
{
    int rc = semb_axhelm_launch_f(h, lambda, geo, z, tmp, nullptr, s); if (rc) return rc;
    rc = semb_mask_launch_f(h, m, tmp, s); if (rc) return rc;
    rc = semb_gs_hi_launch_f(h, tmp, scal, s); if (rc) return rc;
    k_residual<float><<<vec_grid(h->n), VEC_BLOCK, 0, s>>>(h->n, tmp, gs_lists{h->gs_code}, r, res, scal);
    h->launches += 1;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}
// z (+)= Cheb_k(r), k >= 1
int semb_cheb_apply_f(semb_mesh* h, double lambda, const float* geo, const semb_mask_entry& m, const float* dinv, int k,
                      const semb_cheb_coef& c, const float* r, float* z, float* res, float* d, float* Ad, semb_scalars* scal,
                      cudaStream_t s, bool zacc)
{
    const int64_t n = h->n; const unsigned G = vec_grid(n);
    if (k < 1) return semb_fail(h, SEMB_EINVAL, "cheb_apply (fp32): k >= 1 required");
    const gs_lists L{h->gs_code};
    int rc = semb_axhelm_scaled_launch_f(h, lambda, geo, r, dinv, c.itheta, d, Ad, scal, s); if (rc) return rc;
    for (int it = 0; it < k; ++it) {
        if (it > 0) { rc = semb_axhelm_launch_f(h, lambda, geo, d, Ad, nullptr, s); if (rc) return rc; }
        rc = semb_mask_launch_f(h, m, Ad, s); if (rc) return rc;
        rc = semb_gs_hi_launch_f(h, Ad, scal, s); if (rc) return rc;
        const bool first = (it == 0), last = (it == k - 1);
        const float* rin = first ? r : res;
#define SEMB_CHEB_STEP_F(F, La) k_cheb_step<F, La, float><<<G, VEC_BLOCK, 0, s>>>(n, Ad, L, dinv, c.c1[it], c.c2[it], rin, res, d, z, nullptr, scal, h->partials, zacc ? 1 : 0)
        if (first && last) SEMB_CHEB_STEP_F(true, true);
        else if (first)    SEMB_CHEB_STEP_F(true, false);
        else if (last)     SEMB_CHEB_STEP_F(false, true);
        else               SEMB_CHEB_STEP_F(false, false);
#undef SEMB_CHEB_STEP_F
        h->launches += 1;
    }
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}

int semb_dot_rz_launch(semb_mesh* h, const double* r, const double* z, semb_scalars* scal, cudaStream_t s)
{
    k_dot_rz<<<vec_grid(h->n), VEC_BLOCK, 0, s>>>(h->n, r, z, h->invmult, scal, h->partials);
    h->launches += 1;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}

int semb_operator_run(semb_mesh* h, double lambda, const semb_mask_entry& m, const double* v, double* out, cudaStream_t s)
{
    int rc = semb_ensure_work(h, 1); if (rc) return rc;
    double* tmp = h->work;
    k_copy<<<vec_grid(h->n), VEC_BLOCK, 0, s>>>(h->n, v, tmp);
    rc = semb_mask_launch(h, m, tmp, 1, s); if (rc) return rc;
    return apply_A(h, lambda, m, tmp, out, nullptr, s);
}

typedef semb_cheb_coef cheb_coef;
semb_cheb_coef semb_cheb_coefficients(int k, double lmax, int kind, double lmin_frac)
{
    cheb_coef c;
    if (kind == 4) {
        // fourth-kind Chebyshev smoother: d_0 = (4/3)(1/lmax) dinv o r,
        // d_i = ((2i-1)/(2i+3)) d_{i-1} + ((8i+4)/(2i+3)) (1/lmax) dinv o res_i
        c.itheta = 4.0 / (3.0 * lmax);
        for (int i = 1; i <= k && i <= SEMB_MAX_CHEB; ++i) {
            c.c1[i - 1] = (2.0 * i - 1.0) / (2.0 * i + 3.0);
            c.c2[i - 1] = (8.0 * i + 4.0) / ((2.0 * i + 3.0) * lmax);
        }
        return c;
    }
    const double lmin = ((lmin_frac > 0.0 && lmin_frac < 1.0) ? lmin_frac : 0.1) * lmax, theta = 0.5 * (lmax + lmin), delta = 0.5 * (lmax - lmin), sigma = theta / delta;
    double rho = 1.0 / sigma;
    c.itheta = 1.0 / theta;
    for (int it = 0; it < k && it < SEMB_MAX_CHEB; ++it) {
        const double rho1 = 1.0 / (2.0 * sigma - rho);
        c.c1[it] = rho1 * rho; c.c2[it] = 2.0 * rho1 / delta;
        rho = rho1;
    }
    return c;
}

// z = Cheb_k(r);  res, d, Ad: work vectors.  in_pcg: also leave rho = <r,z> and beta in scal (PCG loop).
// Per application (k >= 1): axhelm with the first d formed in its prologue (80 B/node), then per step k_mask,
// k_gs_hi, k_cheb_step (first 60, middle 68, last 60 B/node) and, between steps, a plain axhelm (64).
int semb_cheb_apply(semb_mesh* h, double lambda, const semb_mask_entry& m, const double* dinv, int k, const cheb_coef& c,
                      const double* r, double* z, double* res, double* d, double* Ad, semb_scalars* scal, bool in_pcg, cudaStream_t s,
                      bool zacc)
{
    const int64_t n = h->n; const unsigned G = vec_grid(n);
    if (zacc && k == 0) return semb_fail(h, SEMB_EINVAL, "cheb_apply: accumulation needs k >= 1");
    if (k == 0) {
        k_cheb_init<<<G, VEC_BLOCK, 0, s>>>(n, r, dinv, c.itheta, res, d, z, 1, scal);
        h->launches += 1;
        if (in_pcg) { k_dot_rz<<<G, VEC_BLOCK, 0, s>>>(n, r, z, h->invmult, scal, h->partials); h->launches += 1; }
        SEMB_CUDA(h, cudaGetLastError());
        return SEMB_OK;
    }
    const gs_lists L{h->gs_code};
    const double* rp = in_pcg ? r : nullptr;
    int rc = semb_axhelm_scaled_launch(h, lambda, r, dinv, c.itheta, d, Ad, scal, s); if (rc) return rc;
    for (int it = 0; it < k; ++it) {
        if (it > 0) { rc = semb_axhelm_launch(h, lambda, nullptr, nullptr, d, Ad, 1, nullptr, s); if (rc) return rc; }
        rc = semb_mask_launch(h, m, Ad, 1, s); if (rc) return rc;       // every copy of a Dirichlet node is masked => sum 0
        rc = semb_gs_hi_launch(h, Ad, scal, s); if (rc) return rc;      // edges and corners; faces in k_cheb_step
        const bool first = (it == 0), last = (it == k - 1);
        const double* rin = first ? r : res;
#define SEMB_CHEB_STEP(F, La) k_cheb_step<F, La, double><<<G, VEC_BLOCK, 0, s>>>(n, Ad, L, dinv, c.c1[it], c.c2[it], rin, res, d, z, rp, scal, h->partials, zacc ? 1 : 0)
        if (first && last) SEMB_CHEB_STEP(true, true);
        else if (first)    SEMB_CHEB_STEP(true, false);
        else if (last)     SEMB_CHEB_STEP(false, true);
        else               SEMB_CHEB_STEP(false, false);
#undef SEMB_CHEB_STEP
        h->launches += 1;
    }
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}

int semb_cheb_run(semb_mesh* h, double lambda, uint32_t tags, int k, double lmax, const double* r, double* z, cudaStream_t s)
{
    if (k < 0 || k > SEMB_MAX_CHEB || !(lmax > 0.0)) return semb_fail(h, SEMB_EINVAL, "cheb_jacobi: k=%d lmax=%g", k, lmax);
    semb_mask_entry m; double* dinv;
    int rc = semb_get_mask(h, tags, &m, s); if (rc) return rc;
    rc = semb_get_dinv(h, lambda, tags, &dinv, s); if (rc) return rc;
    rc = semb_ensure_work(h, 3); if (rc) return rc;
    const int64_t n = h->n;
    return semb_cheb_apply(h, lambda, m, dinv, k, semb_cheb_coefficients(k, lmax), r, z, h->work, h->work + n, h->work + 2 * n, nullptr, false, s);
}

// largest eigenvalue of the symmetric tridiagonal (a[0..m), b[0..m-1)) by bisection on the Sturm count
static double tridiag_lmax(int m, const double* a, const double* b);
double semb_tridiag_lmax(int m, const double* a, const double* b) { return tridiag_lmax(m, a, b); }
static double tridiag_lmax(int m, const double* a, const double* b)
{
    double lo = a[0], hi = a[0];
    for (int i = 0; i < m; ++i) {
        const double rad = (i > 0 ? fabs(b[i - 1]) : 0.0) + (i + 1 < m ? fabs(b[i]) : 0.0);
        if (a[i] - rad < lo) lo = a[i] - rad;
        if (a[i] + rad > hi) hi = a[i] + rad;
    }
    for (int it = 0; it < 200 && hi - lo > 1e-15 * fmax(fabs(hi), fabs(lo)); ++it) {
        const double mid = 0.5 * (lo + hi);
        int below = 0; double q = a[0] - mid;               // number of eigenvalues < mid
        if (q < 0.0) ++below;
        for (int i = 1; i < m; ++i) {
            if (q == 0.0) q = 1e-300;
            q = a[i] - mid - b[i - 1] * b[i - 1] / q;
            if (q < 0.0) ++below;
        }
        if (below == m) hi = mid; else lo = mid;
    }
    return 0.5 * (lo + hi);
}

static int dot_to_host(semb_mesh* h, const double* a, const double* b, double* out, cudaStream_t s)
{
    k_dot_aux<<<vec_grid(h->n), VEC_BLOCK, 0, s>>>(h->n, a, b, h->invmult, h->scal, h->partials);
    SEMB_CUDA(h, cudaMemcpyAsync(h->scal_host, h->scal, sizeof(semb_scalars), cudaMemcpyDeviceToHost, s));
    SEMB_CUDA(h, cudaStreamSynchronize(s));
    *out = h->scal_host->aux;
    return SEMB_OK;
}

// Lanczos on D^-1/2 A D^-1/2: v = v0/||v0||; per step  t = D^-1/2 v; w = D^-1/2 A t - beta_{j-1} v_{j-1};
// alpha_j = <w,v>; w -= alpha_j v; beta_j = ||w||; v_{j+1} = w / beta_j.   lmax = 1.1 x largest Ritz value.
int semb_lanczos_run(semb_mesh* h, double lambda, uint32_t tags, const double* v0, int steps, double* lmax, cudaStream_t s)
{
    if (steps < 1 || steps > 64) return semb_fail(h, SEMB_EINVAL, "lanczos steps=%d", steps);
    semb_mask_entry m; double* dinv;
    int rc = semb_get_mask(h, tags, &m, s); if (rc) return rc;
    rc = semb_get_dinv(h, lambda, tags, &dinv, s); if (rc) return rc;
    rc = semb_ensure_work(h, 4); if (rc) return rc;
    const int64_t n = h->n; const unsigned G = vec_grid(n);
    double *v = h->work, *vold = v + n, *w = v + 2 * n, *t = v + 3 * n;
    double nrm2, a[64], b[64];
    rc = dot_to_host(h, v0, v0, &nrm2, s); if (rc) return rc;
    k_scale<<<G, VEC_BLOCK, 0, s>>>(n, 1.0 / sqrt(nrm2), v0, v);
    SEMB_CUDA(h, cudaMemsetAsync(vold, 0, sizeof(double) * (size_t)n, s));
    double bprev = 0.0; int msteps = 0;
    for (int j = 0; j < steps; ++j) {
        k_sqrt_scale<<<G, VEC_BLOCK, 0, s>>>(n, dinv, v, t);
        rc = apply_A(h, lambda, m, t, w, nullptr, s); if (rc) return rc;
        k_lanczos_a<<<G, VEC_BLOCK, 0, s>>>(n, dinv, bprev, vold, w);
        rc = dot_to_host(h, w, v, &a[j], s); if (rc) return rc;
        k_axpy<<<G, VEC_BLOCK, 0, s>>>(n, -a[j], v, w);
        double bb; rc = dot_to_host(h, w, w, &bb, s); if (rc) return rc;
        b[j] = sqrt(bb);
        msteps = j + 1;
        if (!(b[j] > 0.0)) break;
        k_copy<<<G, VEC_BLOCK, 0, s>>>(n, v, vold);
        k_scale<<<G, VEC_BLOCK, 0, s>>>(n, 1.0 / b[j], w, v);
        bprev = b[j];
    }
    SEMB_CUDA(h, cudaGetLastError());
    *lmax = 1.1 * tridiag_lmax(msteps, a, b);
    return SEMB_OK;
}

int semb_pcg_run(semb_mesh* h, const semb_pcg_opts* o, const double* b, double* x, semb_pcg_stats* st, cudaStream_t s)
{
    const int64_t n = h->n; const unsigned G = vec_grid(n);
    const int64_t launches0 = h->launches;
    if (o->precond < 0 || o->precond > 3 || o->maxit < 0 || (o->precond == 2 && (o->cheb_degree < 0 || o->cheb_degree > SEMB_MAX_CHEB)))
        return semb_fail(h, SEMB_EINVAL, "pcg: precond=%d cheb_degree=%d maxit=%d", o->precond, o->cheb_degree, o->maxit);
    semb_mask_entry m; double* dinv = nullptr;
    int rc = semb_get_mask(h, o->dirichlet_tags, &m, s); if (rc) return rc;
    if (o->precond >= 1) { rc = semb_get_dinv(h, o->lambda, o->dirichlet_tags, &dinv, s); if (rc) return rc; }
    semb_mg_ctx mgctx{};
    if (o->precond == 3) { rc = semb_mg_prepare(h, o, &mgctx, s); if (rc) return rc; }   // may use h->work (lambda_max estimate)
    rc = semb_ensure_work(h, o->precond == 2 ? 6 : (o->precond == 3 ? 4 : 3)); if (rc) return rc;
    double *r = h->work, *p = r + n, *q = r + 2 * n;
    double *z = nullptr, *res = nullptr, *d = nullptr;
    if (o->precond == 2) { z = r + 3 * n; res = r + 4 * n; d = r + 5 * n; }
    if (o->precond == 3) z = r + 3 * n;

    double lmax = o->cheb_lmax;
    cheb_coef cc{};
    if (o->precond == 2) {
        if (!(lmax > 0.0)) {
            // start vector of the estimator: the right-hand side (continuous, masked)
            rc = semb_lanczos_run(h, o->lambda, o->dirichlet_tags, b, 10, &lmax, s); if (rc) return rc;
            r = h->work; p = r + n; q = r + 2 * n; z = r + 3 * n; res = r + 4 * n; d = r + 5 * n;
        }
        cc = semb_cheb_coefficients(o->cheb_degree, lmax);
    }
    // history buffer
    const int want_hist = (st && st->hist_host_or_null && st->hist_len > 0) ? st->hist_len : 0;
    if (want_hist > h->hist_cap) {
        if (h->hist_dev) semb_dev_free(h, h->hist_dev);
        h->hist_dev = (double*)semb_dev_alloc(h, sizeof(double) * (size_t)want_hist);
        if (!h->hist_dev) { h->hist_cap = 0; return semb_fail(h, SEMB_ENOMEM, "residual history"); }
        h->hist_cap = want_hist;
    }
    double* hist = want_hist ? h->hist_dev : nullptr;

    semb_scalars init; memset(&init, 0, sizeof(init));
    init.rtol = o->rtol; init.atol = o->atol; init.maxit = o->maxit; init.status = SEMB_MAXIT;
    SEMB_CUDA(h, cudaMemcpyAsync(h->scal, &init, sizeof(init), cudaMemcpyHostToDevice, s));

    const double* dz = (o->precond == 1) ? dinv : nullptr;      // fused z = dinv o r
    const int nm = o->null_mean ? 1 : 0;
    if (nm) {
        if (m.count != 0 || o->lambda != 0.0)
            return semb_fail(h, SEMB_EINVAL, "pcg: null_mean needs lambda = 0 and a tag set without Dirichlet nodes");
        k_mean<<<G, VEC_BLOCK, 0, s>>>(n, b, h->invmult, 1.0 / (double)h->n_unique, h->scal, h->partials);
        h->launches += 1;
    }
    if (!o->x0_is_zero) {
        rc = apply_A(h, o->lambda, m, x, q, nullptr, s); if (rc) return rc;
        k_pcg_init<<<G, VEC_BLOCK, 0, s>>>(n, b, q, x, r, h->invmult, dz, h->scal, h->partials, hist, nm);
    } else {
        k_pcg_init<<<G, VEC_BLOCK, 0, s>>>(n, b, nullptr, x, r, h->invmult, dz, h->scal, h->partials, hist, nm);
    }
    SEMB_CUDA(h, cudaGetLastError());

    h->launches += 1;
    // optional event pairs around the axhelm launches of the first iterations (no synchronisation added)
    const int nprof = o->profile ? (o->maxit < 64 ? o->maxit : 64) : 0;
    while ((int)h->prof_ev.size() < 2 * nprof) {
        cudaEvent_t ev; SEMB_CUDA(h, cudaEventCreate(&ev)); h->prof_ev.push_back(ev);
    }
    const int check = o->check_every > 0 ? o->check_every : 16;
    bool finished = (o->maxit == 0);
    // small meshes: two launches per iteration instead of five (k_iter_small)
    const bool small = n <= SEMB_SMALL_N && o->precond <= 1 && !o->profile;
    const int64_t ndot = small ? semb_axhelm_dot_count(h) : 0;
    // ... and where one block per element fits on the device at once, the whole loop is ONE cooperative launch (pcg_persist.cu)
    const char* persist_env = getenv("SEMB_PCG_PERSIST");          // "0": keep the launch-per-phase loop (A/B runs, tests of that path)
    const bool persist_on = persist_env ? atoi(persist_env) != 0 : true;
    if (persist_on && o->precond <= 1 && !o->profile && !finished) {        // eligibility (elements, residency) is decided in there
        rc = semb_pcg_persist_run(h, o->lambda, m, o->dirichlet_tags, dz, r, x, p, q, hist, want_hist, s);
        if (rc < 0) return rc;
        if (rc == 1) {
            SEMB_CUDA(h, cudaMemcpyAsync(h->scal_host, h->scal, sizeof(semb_scalars), cudaMemcpyDeviceToHost, s));
            SEMB_CUDA(h, cudaStreamSynchronize(s));
            finished = true;
        }
    }
    for (int it0 = 0; it0 < o->maxit && !finished; it0 += check) {
        const int mbatch = (o->maxit - it0 < check) ? o->maxit - it0 : check;
        for (int i = 0; i < mbatch; ++i) {
            const double* zsrc = r;
            if (o->precond == 2) {
                rc = semb_cheb_apply(h, o->lambda, m, dinv, o->cheb_degree, cc, r, z, res, d, q, h->scal, true, s); if (rc) return rc;
                zsrc = z;
            } else if (o->precond == 3) {
                rc = semb_mg_vcycle_run(h, mgctx, 0, r, z, h->scal, s); if (rc) return rc;
                rc = semb_dot_rz_launch(h, r, z, h->scal, s); if (rc) return rc;
                zsrc = z;
            }
            const int itn = it0 + i;
            if (itn < nprof) SEMB_CUDA(h, cudaEventRecord(h->prof_ev[2 * itn], s));
            h->defer_dot_finish = small;
            rc = semb_axhelm_pcg_launch(h, o->lambda, zsrc, dz, p, x, q, h->scal, s);
            h->defer_dot_finish = false;
            if (rc) return rc;
            if (itn < nprof) SEMB_CUDA(h, cudaEventRecord(h->prof_ev[2 * itn + 1], s));
            if (small) {
                k_iter_small<true><<<SMALL_CL, SMALL_BLOCK, 0, s>>>(n, ndot, h->ax_dot, m.count, m.list, h->n_gs_hi, h->gs_hi, h->gs_off, h->gs_ids,
                                                                    q, r, h->gs_code, dz, h->scal, h->partials, hist, want_hist);     // dz == NULL: z = r
                h->launches += 1;
                continue;
            }
            rc = semb_mask_launch(h, m, q, 1, s); if (rc) return rc;     // every copy of a Dirichlet node is masked => sum 0
            rc = semb_gs_hi_launch(h, q, h->scal, s); if (rc) return rc; // edges and corners; faces in k_update_r
            const gs_lists L{h->gs_code};
            if (o->precond >= 2) k_update_r<false><<<G, VEC_BLOCK, 0, s>>>(n, q, r, L, nullptr, h->scal, h->partials, hist, want_hist);
            else                 k_update_r<true><<<G, VEC_BLOCK, 0, s>>>(n, q, r, L, dz, h->scal, h->partials, hist, want_hist);
            h->launches += 1;
        }
        SEMB_CUDA(h, cudaGetLastError());
        SEMB_CUDA(h, cudaMemcpyAsync(h->scal_host, h->scal, sizeof(semb_scalars), cudaMemcpyDeviceToHost, s));
        SEMB_CUDA(h, cudaStreamSynchronize(s));
        finished = h->scal_host->done != 0;
    }
    if (o->maxit > 0) { k_final_x<<<G, VEC_BLOCK, 0, s>>>(n, p, x, h->scal); h->launches += 1; SEMB_CUDA(h, cudaGetLastError()); }
    if (nm) {                                                   // the solution of zero mean
        k_mean<<<G, VEC_BLOCK, 0, s>>>(n, x, h->invmult, 1.0 / (double)h->n_unique, h->scal, h->partials);
        k_shift<<<G, VEC_BLOCK, 0, s>>>(n, x, h->scal);
        h->launches += 2;
        SEMB_CUDA(h, cudaGetLastError());
    }
    if (o->maxit == 0 || !finished) {
        SEMB_CUDA(h, cudaMemcpyAsync(h->scal_host, h->scal, sizeof(semb_scalars), cudaMemcpyDeviceToHost, s));
        SEMB_CUDA(h, cudaStreamSynchronize(s));
    }
    const semb_scalars& S = *h->scal_host;
    int status = S.status;
    if (st) {
        st->iters = S.iter; st->status = status; st->b_norm = S.bnorm; st->r0_norm = S.r0norm; st->r_norm = S.rnorm;
        st->lmax_used = (o->precond == 3) ? mgctx.lmax[0] : lmax;
        st->launches = h->launches - launches0;
        st->profiled = 0; st->axhelm_ms = 0.0;
        const int np_ = S.iter < nprof ? S.iter : nprof;
        if (np_ > 0) {
            double tot = 0.0;
            for (int i = 0; i < np_; ++i) { float ms = 0.f; SEMB_CUDA(h, cudaEventElapsedTime(&ms, h->prof_ev[2 * i], h->prof_ev[2 * i + 1])); tot += ms; }
            st->profiled = np_; st->axhelm_ms = tot / np_;
        }
        if (want_hist) {
            const int cnt = (S.iter + 1 < want_hist) ? S.iter + 1 : want_hist;
            SEMB_CUDA(h, cudaMemcpyAsync(st->hist_host_or_null, hist, sizeof(double) * cnt, cudaMemcpyDeviceToHost, s));
            SEMB_CUDA(h, cudaStreamSynchronize(s));
        }
    }
    if (status == SEMB_EBREAKDOWN) return semb_fail(h, SEMB_EBREAKDOWN, "pcg breakdown: p.Ap = %g at iteration %d", S.pAp, S.iter + 1);
    return status;
}
