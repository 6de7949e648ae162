// Jacobi-PCG of a SMALL mesh as ONE persistent kernel (round-1 verdict item 6 "kill the latency floors").
//
// Below ~10^5 nodes an iteration of the launch-per-phase loop (pcg.cu) is nothing but latency: configs[0] (64 elements, N = 7,
// 32 768 nodes) took 30 us per iteration with five launches and 23 us with two (k_iter_small).  Here the whole solve is one
// cooperative launch: one block per element, n1^2 threads, the element's geometric factors in shared memory and its part of
// r, p, x, D^-1 and the gather-scatter codes in registers for the whole solve.  An iteration is
//     p = D^-1 r + beta p;  w = A_e p (line contractions as in k_axhelm_line);  partial p.w;  shared nodes of w -> q      | all-sum = barrier
//     p.Ap (every block, same order, same bits);  alpha;  Ap = w + partner / class members of q;
//     x += alpha p;  r -= alpha Ap;  partial <r,r>, <r,z>                                                              | all-sum = barrier
//     beta;  stop test (uniform over the grid)
// i.e. two grid-wide synchronisations per iteration, each fused with the sum it exists for (pp_allsum below); the cooperative
// launch guarantees that all blocks are resident.  Values written by other blocks are read with ld.global.cg (L1 is not coherent).
// All sums have a fixed order: iterates are reproducible run to run.
#include <vector>

#include "axhelm_launch.cuh"

#define PP_FACE   (1 << 28)
#define PP_SHARED (1 << 29)
#define PP_CH 10          // remote copies a thread fetches per batch: one batch covers 10 n1^2 entries (a hexahedron inside a box mesh needs ~9 n1^2)

struct pp_args {
    int64_t E, n;
    const double* geo; double lambda; const double* dinv;            // dinv == NULL: no preconditioner (z = r)
    const int32_t *code, *noff, *rlist; const unsigned char* msk;     // gather-scatter code per node; remote-copy lists (below); Dirichlet flags
    double *r, *x, *p, *q;
    semb_scalars* scal; double* part; unsigned int* bar;              // part[3][E]: per-block partial sums; arrival counter of the grid barrier
    double* hist; int hist_cap;
};

// ---- grid barrier + all-reduce: block b leaves its K partial sums in part[k][b], arrives at the counter (release: bar.sync,
// fence, atomic by thread 0), waits until all gridDim.x blocks of this phase have arrived (ld.acquire spin by thread 0,
// bar.sync) and adds all partials in a fixed order: every thread of every block gets the same bits.
// Measured and rejected on B200 (configs[0], 64 blocks): publishing each partial in self-validating {phase : half of the double}
// words that all threads poll, so that the poll is the data load (one round trip instead of three): 15.4 -> 18.8 us per
// iteration -- 4096 polling threads delay the very stores they wait for.
// K block-wide sums with one pair of barriers (block_sum of reduce.cuh, K values at a time; the same fixed order per value)
template <int K>
__device__ __forceinline__ void pp_block_sum(double (&v)[K], double* red)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    const int live = min(32, (int)blockDim.x - (wid << 5));
#pragma unroll
    for (int k = 0; k < K; ++k) v[k] = warp_sum_live(v[k], lane, live);
    __syncthreads();                       // red may still be read from a previous call
    if (lane == 0) {
#pragma unroll
        for (int k = 0; k < K; ++k) red[k * 32 + wid] = v[k];
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < K; ++k) {
        double t = 0.0;
        for (int w = 0; w < nw; ++w) t += red[k * 32 + w];
        v[k] = t;
    }
}

template <int K>
__device__ __forceinline__ void pp_allsum(double* part, unsigned* bar, int64_t E, const double (&v)[K], double (&tot)[K], unsigned phase, double* red)
{
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < K; ++k) __stcg(part + k * E + blockIdx.x, v[k]);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(bar, 1u);
        unsigned seen;
        do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(bar) : "memory"); } while (seen < phase * gridDim.x);
    }
    __syncthreads();
    double s[K];
#pragma unroll
    for (int k = 0; k < K; ++k) s[k] = 0.0;
    for (int64_t t = threadIdx.x; t < E; t += blockDim.x) {
#pragma unroll
        for (int k = 0; k < K; ++k) s[k] += __ldcg(part + k * E + t);
    }
    pp_block_sum<K>(s, red);
#pragma unroll
    for (int k = 0; k < K; ++k) tot[k] = s[k];
}

template <int n1, bool HELM>
__global__ void __launch_bounds__(n1 * n1)
k_pcg_persist(pp_args A)
{
    constexpr int n2 = n1 * n1, Np = n2 * n1, NG = HELM ? 7 : 6;
    using T = ax_tile<n1>;
    extern __shared__ __align__(16) double pp_sm[];
    double* __restrict__ Gs = pp_sm;                       // [NG][Np]: slot = factor plane + thread, conflict free
    double* __restrict__ Su = Gs + NG * Np;
    double* __restrict__ Sr = Su + T::sizeA;
    double* __restrict__ Ss = Sr + T::sizeA;
    double* red = Ss + T::sizeB;                           // 2 x 32 doubles
    double* __restrict__ Sg = red + 64;                    // the remote copies this element needs in the assembly (<= max over elements)
    semb_scalars* __restrict__ scal = A.scal;
    if (*(volatile const int32_t*)&scal->done) return;     // set before the launch only (k_pcg_init): uniform over the grid
    const int tl = threadIdx.x, a = tl % n1, b = tl / n1;
    int ra = a, rb = b, sa = a, sb = b;
    if (T::permuted) {
        const int rq = c_perm[n1 - 1][0][tl], sq = c_perm[n1 - 1][1][tl];
        ra = rq % n1; rb = rq / n1; sa = sq % n1; sb = sq / n1;
    }
    const int64_t e = blockIdx.x, E = A.E, l0 = e * Np + tl;
    // ---- the state that stays on the SM for the whole solve
    {
        const double* __restrict__ g = A.geo + e * 7 * (int64_t)Np + tl;
#pragma unroll
        for (int c = 0; c < NG; ++c) {
#pragma unroll
            for (int k = 0; k < n1; ++k) Gs[c * Np + k * n2 + tl] = __ldg(g + c * Np + k * n2);
        }
    }
    double r[n1], p[n1], x[n1], dv[n1];
    double wq[n1];                                         // 1 / multiplicity: weight of the node in sums over local nodes
    int32_t pos[n1];                                       // start of the node's entries in Sg | number of entries << 20 | PP_FACE | PP_SHARED
    unsigned mbits = 0u;
    const int32_t ebase = __ldg(A.noff + e * Np), ecnt = __ldg(A.noff + (e + 1) * Np) - ebase;
#pragma unroll
    for (int k = 0; k < n1; ++k) {
        const int64_t l = l0 + k * n2;
        r[k] = A.r[l]; x[k] = A.x[l]; p[k] = 0.0;
        dv[k] = A.dinv ? A.dinv[l] : 1.0;
        const int32_t cd = A.code[l];
        wq[k] = (cd <= -2) ? 0.5 : (cd >= 3) ? 1.0 / (double)cd : 1.0;
        const int32_t n0 = __ldg(A.noff + l), nn = __ldg(A.noff + l + 1) - n0;
        pos[k] = (n0 - ebase) | (nn << 20) | (cd <= -2 ? PP_FACE : 0) | (cd != -1 ? PP_SHARED : 0);
        if (A.msk[l]) { mbits |= 1u << k; pos[k] &= PP_SHARED; }    // Dirichlet node: w = 0 is published, nothing is added
    }
    double rho = scal->rho_new, beta = 0.0, alpha = 0.0, pAp = 0.0, rnorm = scal->rnorm, trr = scal->rr;
    const double target = scal->target, lambda = A.lambda;
    const int maxit = scal->maxit;
    int iter = 0, status = SEMB_MAXIT;
    unsigned phase = 0u;
    double* __restrict__ partA = A.part; double* __restrict__ partB = A.part + E;              // [1][E] and [2][E]
#pragma unroll 1
    for (int it = 0; it < maxit; ++it) {
        // ---- p = z + beta p, z = D^-1 r;  w = A_e p
#pragma unroll
        for (int k = 0; k < n1; ++k) { p[k] = dv[k] * r[k] + beta * p[k]; Su[T::idx(k, b, a)] = p[k]; }
        __syncthreads();
        {
            double ln[n1], out[n1];
#pragma unroll
            for (int i = 0; i < n1; ++i) ln[i] = Su[T::idx(rb, ra, i)];
            ax_line<n1, 0, double>(ln, out);
#pragma unroll
            for (int i = 0; i < n1; ++i) Sr[T::idx(rb, ra, i)] = out[i];
#pragma unroll
            for (int j = 0; j < n1; ++j) ln[j] = Su[T::idx(sb, j, sa)];
            ax_line<n1, 0, double>(ln, out);
#pragma unroll
            for (int j = 0; j < n1; ++j) Ss[T::idxB(sb, j, sa)] = out[j];
        }
        double w[n1];
        {
            double ut[n1], gt[n1];
            ax_line<n1, 0, double>(p, ut);
            __syncthreads();
#pragma unroll
            for (int k = 0; k < n1; ++k) {
                const int s = T::idx(k, b, a), sB = T::idxB(k, b, a), g = k * n2 + tl;
                const double ur = Sr[s], us = Ss[sB];
                const double Grr = Gs[g], Grs = Gs[Np + g], Grt = Gs[2 * Np + g], Gss = Gs[3 * Np + g], Gst = Gs[4 * Np + g], Gtt = Gs[5 * Np + g];
                Sr[s] = Grr * ur + Grs * us + Grt * ut[k];
                Ss[sB] = Grs * ur + Gss * us + Gst * ut[k];
                gt[k] = Grt * ur + Gst * us + Gtt * ut[k];
            }
            __syncthreads();
            double ln[n1], out[n1];
#pragma unroll
            for (int i = 0; i < n1; ++i) ln[i] = Sr[T::idx(rb, ra, i)];
            ax_line<n1, 1, double>(ln, out);
#pragma unroll
            for (int i = 0; i < n1; ++i) Sr[T::idx(rb, ra, i)] = out[i];
#pragma unroll
            for (int j = 0; j < n1; ++j) ln[j] = Ss[T::idxB(sb, j, sa)];
            ax_line<n1, 1, double>(ln, out);
#pragma unroll
            for (int j = 0; j < n1; ++j) Ss[T::idxB(sb, j, sa)] = out[j];
            ax_line<n1, 1, double>(gt, w);
            if (HELM) {
#pragma unroll
                for (int k = 0; k < n1; ++k) w[k] += lambda * Gs[(HELM ? 6 : 0) * Np + k * n2 + tl] * p[k];
            }
            __syncthreads();
        }
        double dot = 0.0;
#pragma unroll
        for (int k = 0; k < n1; ++k) {
            w[k] += Sr[T::idx(k, b, a)] + Ss[T::idxB(k, b, a)];
            dot += p[k] * w[k];                            // p is continuous and zero at Dirichlet nodes: sum over elements = p.Ap
            if (mbits >> k & 1u) w[k] = 0.0;               // Dirichlet mask before the assembly
            if (pos[k] & PP_SHARED) __stcg(A.q + l0 + k * n2, w[k]);
        }
        {
            const double v[1] = { block_sum(dot, red) };
            double tot[1];
            pp_allsum<1>(partA, A.bar, E, v, tot, ++phase, red);
            pAp = tot[0];
        }
        // ---- alpha;  Ap = QQ^T w at the thread's nodes;  x, r;  partial <r,r>, <r,z>
        if (!(pAp > 0.0) || !isfinite(pAp)) { status = SEMB_EBREAKDOWN; break; }        // uniform: every block has the same bits
        alpha = rho / pAp;
        // every remote copy the element's shared nodes need (face partners; all members of the edge / corner classes, in class
        // order, own copies included), fetched by all threads together in batches of independent loads
#pragma unroll 1
        for (int i0 = 0; i0 < ecnt; i0 += PP_CH * n2) {
            int32_t id[PP_CH]; double v[PP_CH];
#pragma unroll
            for (int u = 0; u < PP_CH; ++u) { const int i = i0 + u * n2 + tl; id[u] = (i < ecnt) ? __ldg(A.rlist + ebase + i) : -1; }
#pragma unroll
            for (int u = 0; u < PP_CH; ++u) v[u] = (id[u] >= 0) ? __ldcg(A.q + id[u]) : 0.0;
#pragma unroll
            for (int u = 0; u < PP_CH; ++u) if (id[u] >= 0) Sg[i0 + u * n2 + tl] = v[u];
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < n1; ++k) {
            const int st = pos[k] & 0xfffff, cnt = (pos[k] >> 20) & 0xff;
            if (cnt) {
                double c = (pos[k] & PP_FACE) ? w[k] : 0.0;     // face: own + partner;  class: its members in list order, the same bits in every copy
                for (int u = 0; u < cnt; ++u) c += Sg[st + u];
                w[k] = c;
            }
        }
        double rr = 0.0, rz = 0.0;
#pragma unroll
        for (int k = 0; k < n1; ++k) {
            x[k] += alpha * p[k];
            r[k] -= alpha * w[k];
            const double t = r[k] * r[k] * wq[k];
            rr += t; rz += dv[k] * t;
        }
        double trz;
        {
            double v[2] = { rr, rz };
            pp_block_sum<2>(v, red);
            double tot[2];
            pp_allsum<2>(partB, A.bar, E, v, tot, ++phase, red);
            trr = tot[0]; trz = tot[1];
        }
        rnorm = sqrt(trr);
        iter = it + 1;
        if (e == 0 && tl == 0 && A.hist && iter < A.hist_cap) A.hist[iter] = rnorm;
        beta = trz / rho;
        rho = trz;
        if (rnorm <= target) { status = SEMB_OK; break; }
    }
    // ---- hand the state back
#pragma unroll
    for (int k = 0; k < n1; ++k) { const int64_t l = l0 + k * n2; A.r[l] = r[k]; A.x[l] = x[k]; A.p[l] = p[k]; }
    if (e == 0 && tl == 0) {
        scal->iter = iter; scal->rr = trr; scal->rnorm = rnorm; scal->rho_new = rho; scal->rz = rho; scal->beta = beta;
        scal->pAp = pAp; scal->alpha = alpha; scal->x_pending = 0; scal->status = status; scal->done = 1;
    }
}

// ---- host side ------------------------------------------------------------------------------------------------------
static __global__ void k_pp_mask(int64_t count, const int32_t* __restrict__ list, unsigned char* __restrict__ msk)
{
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t < count) msk[list[t]] = 1;
}

template <int n1> static size_t pp_smem(bool helm, int maxcnt)
{
    using T = ax_tile<n1>;
    return sizeof(double) * ((size_t)(helm ? 7 : 6) * n1 * n1 * n1 + 2 * T::sizeA + T::sizeB + 64 + (size_t)maxcnt);
}

// 1: launched;  0: not eligible (the caller runs the launch-per-phase loop);  < 0: error
template <int n1>
static int pp_launch(semb_mesh* h, const pp_args& A, bool helm, cudaStream_t s)
{
    const size_t smem = pp_smem<n1>(helm, h->pp_maxcnt);
    const void* kern = helm ? (const void*)k_pcg_persist<n1, true> : (const void*)k_pcg_persist<n1, false>;
    int dev = 0, optin = 0, nb = 0, coop = 0;
    SEMB_CUDA(h, cudaGetDevice(&dev));
    SEMB_CUDA(h, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    SEMB_CUDA(h, cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    if (!coop || smem > (size_t)optin) return 0;
    SEMB_CUDA(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    SEMB_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, n1 * n1, smem));
    if ((int64_t)nb * semb_sm_count() < h->E) return 0;                  // all blocks must be resident
    pp_args args = A;
    void* params[] = { (void*)&args };
    SEMB_CUDA(h, cudaMemsetAsync(A.bar, 0, sizeof(unsigned int), s));
    SEMB_CUDA(h, cudaLaunchCooperativeKernel(kern, dim3((unsigned)h->E), dim3(n1 * n1), params, smem, s));
    h->launches += 1;
    return 1;
}

// Remote-copy lists, built once per handle on the host (n <= 65 536 nodes): node l needs rlist[noff[l] .. noff[l+1]) --
// a face node its partner, a node of a class with >= 3 members all members of the class in class order (itself included),
// an unshared node nothing.  The entries of an element are contiguous (nodes are numbered element by element).
static int pp_build_lists(semb_mesh* h, cudaStream_t s)
{
    const int64_t n = h->n, Np = (int64_t)h->n1 * h->n1 * h->n1;
    std::vector<int32_t> code((size_t)n), off((size_t)h->n_gs + 1), ids((size_t)h->n_shared + 1), noff((size_t)n + 1, 0);
    SEMB_CUDA(h, cudaMemcpyAsync(code.data(), h->gs_code, sizeof(int32_t) * (size_t)n, cudaMemcpyDeviceToHost, s));
    if (h->n_gs > 0) {
        SEMB_CUDA(h, cudaMemcpyAsync(off.data(), h->gs_off, sizeof(int32_t) * ((size_t)h->n_gs + 1), cudaMemcpyDeviceToHost, s));
        SEMB_CUDA(h, cudaMemcpyAsync(ids.data(), h->gs_ids, sizeof(int32_t) * (size_t)h->n_shared, cudaMemcpyDeviceToHost, s));
    }
    SEMB_CUDA(h, cudaStreamSynchronize(s));
    for (int64_t l = 0; l < n; ++l) noff[l + 1] = noff[l] + (code[l] <= -2 ? 1 : code[l] >= 3 ? code[l] : 0);
    std::vector<int32_t> rl((size_t)noff[n] + 1, 0);
    for (int64_t l = 0; l < n; ++l) if (code[l] <= -2) rl[noff[l]] = -(code[l] + 2);
    for (int64_t g = 0; g < h->n_gs; ++g) {
        const int32_t a = off[g], b = off[g + 1];
        if (b - a < 3) continue;
        for (int32_t t = a; t < b; ++t)
            for (int32_t u = a; u < b; ++u) rl[noff[ids[t]] + (u - a)] = ids[u];
    }
    int maxcnt = 0;
    for (int64_t e = 0; e < h->E; ++e) { const int c = noff[(e + 1) * Np] - noff[e * Np]; if (c > maxcnt) maxcnt = c; }
    if (maxcnt >= (1 << 20)) return semb_fail(h, SEMB_EINVAL, "persistent PCG: %d remote copies in one element", maxcnt);
    for (int64_t l = 0; l < n; ++l) if (code[l] > 255) { h->pp_maxcnt = -1; return SEMB_OK; }      // a class of more than 255 copies: not eligible
    h->pp_maxcnt = maxcnt;
    h->pp_noff = (int32_t*)semb_dev_alloc(h, sizeof(int32_t) * ((size_t)n + 1));
    h->pp_rlist = (int32_t*)semb_dev_alloc(h, sizeof(int32_t) * rl.size());
    h->pp_msk = (unsigned char*)semb_dev_alloc(h, (size_t)n);
    h->pp_part = (double*)semb_dev_alloc(h, sizeof(double) * (3 * (size_t)h->E + 2));
    if (!h->pp_noff || !h->pp_rlist || !h->pp_msk || !h->pp_part) {
        semb_dev_free(h, h->pp_noff); semb_dev_free(h, h->pp_rlist); semb_dev_free(h, h->pp_msk); semb_dev_free(h, h->pp_part);
        h->pp_noff = h->pp_rlist = nullptr; h->pp_msk = nullptr; h->pp_part = nullptr;
        return semb_fail(h, SEMB_ENOMEM, "persistent PCG: node tables");
    }
    SEMB_CUDA(h, cudaMemcpyAsync(h->pp_noff, noff.data(), sizeof(int32_t) * ((size_t)n + 1), cudaMemcpyHostToDevice, s));
    SEMB_CUDA(h, cudaMemcpyAsync(h->pp_rlist, rl.data(), sizeof(int32_t) * rl.size(), cudaMemcpyHostToDevice, s));
    SEMB_CUDA(h, cudaStreamSynchronize(s));                              // the host vectors go out of scope
    h->pp_msk_valid = false;
    return SEMB_OK;
}

int semb_pcg_persist_run(semb_mesh* h, double lambda, const semb_mask_entry& m, uint32_t tags, const double* dinv, double* r, double* x, double* p,
                         double* q, double* hist, int hist_cap, cudaStream_t s)
{
    const int64_t n = h->n, E = h->E;
    // stored fp64 factors; blocks of at least 16 threads; a barrier over at most 768 blocks (measured on B200, ~30 000-node boxes:
    // N = 3, 512 elements 21.8 -> 14.8 us per iteration, N = 2, 1000 elements 23.8 -> 51 us: those stay on the launch-per-phase loop)
    if (h->geo_mode != 0 || h->n1 < 4 || E > 768) return 0;
    if (!h->pp_noff && h->pp_maxcnt >= 0) {
        int rc = ax_upload_basis_tu(h); if (rc) return rc;               // this translation unit's copy of the constant tables
        rc = pp_build_lists(h, s); if (rc) return rc;
    }
    if (h->pp_maxcnt < 0) return 0;
    if (!h->pp_msk_valid || h->pp_msk_tags != tags) {
        SEMB_CUDA(h, cudaMemsetAsync(h->pp_msk, 0, (size_t)n, s));
        if (m.count > 0) k_pp_mask<<<(unsigned)((m.count + 255) / 256), 256, 0, s>>>(m.count, m.list, h->pp_msk);
        SEMB_CUDA(h, cudaGetLastError());
        h->pp_msk_tags = tags; h->pp_msk_valid = true;
    }
    pp_args A;
    A.E = E; A.n = n; A.geo = h->geo; A.lambda = lambda; A.dinv = dinv;
    A.code = h->gs_code; A.noff = h->pp_noff; A.rlist = h->pp_rlist; A.msk = h->pp_msk;
    A.r = r; A.x = x; A.p = p; A.q = q; A.scal = h->scal; A.part = h->pp_part; A.bar = (unsigned int*)(h->pp_part + 3 * E);
    A.hist = hist; A.hist_cap = hist_cap;
    const bool helm = lambda != 0.0;
    switch (h->n1) {
        case 3:  return pp_launch<3>(h, A, helm, s);
        case 4:  return pp_launch<4>(h, A, helm, s);
        case 5:  return pp_launch<5>(h, A, helm, s);
        case 6:  return pp_launch<6>(h, A, helm, s);
        case 7:  return pp_launch<7>(h, A, helm, s);
        case 8:  return pp_launch<8>(h, A, helm, s);
        case 9:  return pp_launch<9>(h, A, helm, s);
        case 10: return pp_launch<10>(h, A, helm, s);
        case 11: return pp_launch<11>(h, A, helm, s);
    }
    return 0;
}
