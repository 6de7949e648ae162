// axhelm: the matrix-free local operator  w = D^T G D u + lambda B u  per hexahedral element
// (BASELINE.json:north_star; §2.2 "matrix-free ... tensor-product contractions with
// (p+1)x(p+1) operator matrices identical for all elements", O(N_e p^4) work on O(N_e p^3) data).
//
//   u_r = sum_m D_im u(m,j,k)   u_s = sum_m D_jm u(i,m,k)   u_t = sum_m D_km u(i,j,m)
//   g_r = G_rr u_r + G_rs u_s + G_rt u_t,  g_s = G_rs u_r + G_ss u_s + G_st u_t,  g_t = G_rt u_r + G_st u_s + G_tt u_t
//   w(i,j,k) = sum_m D_mi g_r(m,j,k) + sum_m D_mj g_s(i,m,k) + sum_m D_mk g_t(i,j,m) + lambda B u
//
// Algorithmic bytes per node: 8 (u) + 8 (w) + 48 (G) = 64, + 8 (B) when lambda != 0.
#include "reduce.cuh"
#include "semb_internal.h"

// D for every order 1..SEMB_MAX_N, row-major n1 x n1 at c_D[N]; filled at setup.
__constant__ double c_D[SEMB_MAX_N + 1][SEMB_MAXN1 * SEMB_MAXN1];

int semb_axhelm_upload_basis(semb_mesh* h)
{
    SEMB_CUDA(h, cudaMemcpyToSymbol(c_D, h->D, sizeof(double) * h->n1 * h->n1,
                                    sizeof(double) * SEMB_MAXN1 * SEMB_MAXN1 * (size_t)h->N));
    return SEMB_OK;
}

int semb_axhelm_prepare_geo(semb_mesh* h, cudaStream_t) { h->geoK = h->geo; return SEMB_OK; }

// ---------------------------------------------------------------------------------------------
// generic kernel, any order: one element at a time per block of n1 x n1 threads (thread = (i,j) column),
// k-loop with the t-direction column in registers and the r,s-direction plane in shared memory.
template <int n1, bool HELM>
__global__ void __launch_bounds__(n1 * n1)
k_axhelm_slab(int64_t E, int64_t n, const double* __restrict__ geo, double lambda,
              const double* __restrict__ lam0, const double* __restrict__ lam1,
              const double* __restrict__ u, double* __restrict__ w, int nfields,
              semb_scalars* __restrict__ scal, double* __restrict__ partials)
{
    constexpr int N = n1 - 1, Np = n1 * n1 * n1, n2 = n1 * n1;
    __shared__ double sD[n1][n1 + 1];
    __shared__ double su[n1][n1 + 1], sgr[n1][n1 + 1], sgs[n1][n1 + 1];
    __shared__ double red[32];
    if (scal && *(volatile int32_t*)&scal->done) return;
    const int i = threadIdx.x % n1, j = threadIdx.x / n1;
    sD[j][i] = c_D[N][j * n1 + i];
    double dot = 0.0;
    for (int64_t ef = blockIdx.x; ef < E * nfields; ef += gridDim.x) {
        const int64_t e = ef % E, f = ef / E;
        const double* __restrict__ ue = u + f * n + e * Np;
        double* __restrict__ we = w + f * n + e * Np;
        const double* __restrict__ g = geo + e * 7 * (int64_t)Np;
        double ru[n1], rw[n1];
#pragma unroll
        for (int k = 0; k < n1; ++k) { ru[k] = ue[k * n2 + j * n1 + i]; rw[k] = 0.0; }
#pragma unroll
        for (int k = 0; k < n1; ++k) {
            const int l = k * n2 + j * n1 + i;
            __syncthreads();
            su[j][i] = ru[k];
            __syncthreads();
            double ur = 0.0, us = 0.0, ut = 0.0;
#pragma unroll
            for (int m = 0; m < n1; ++m) {
                ur += sD[i][m] * su[j][m];
                us += sD[j][m] * su[m][i];
                ut += sD[k][m] * ru[m];
            }
            double Grr = g[0 * Np + l], Grs = g[1 * Np + l], Grt = g[2 * Np + l];
            double Gss = g[3 * Np + l], Gst = g[4 * Np + l], Gtt = g[5 * Np + l];
            if (lam0) { const double c = lam0[e * Np + l]; Grr *= c; Grs *= c; Grt *= c; Gss *= c; Gst *= c; Gtt *= c; }
            const double gr = Grr * ur + Grs * us + Grt * ut;
            const double gs = Grs * ur + Gss * us + Gst * ut;
            const double gt = Grt * ur + Gst * us + Gtt * ut;
            sgr[j][i] = gr; sgs[j][i] = gs;
#pragma unroll
            for (int m = 0; m < n1; ++m) rw[m] += sD[k][m] * gt;
            if (HELM) {
                const double lam = lam1 ? lam1[e * Np + l] : lambda;
                rw[k] += lam * g[6 * Np + l] * ru[k];
            }
            __syncthreads();
            double a = 0.0;
#pragma unroll
            for (int m = 0; m < n1; ++m) a += sD[m][i] * sgr[j][m] + sD[m][j] * sgs[m][i];
            rw[k] += a;
        }
#pragma unroll
        for (int k = 0; k < n1; ++k) { we[k * n2 + j * n1 + i] = rw[k]; dot += ru[k] * rw[k]; }
    }
    if (scal) {
        double v[1] = { block_sum(dot, red) }, tot[1];
        if (grid_sum<1>(v, partials, &scal->ticket[0], tot, red) && threadIdx.x == 0) {
            const double gamma = tot[0];
            scal->pAp = gamma;
            if (!(gamma > 0.0) || !isfinite(gamma)) { scal->status = SEMB_EBREAKDOWN; scal->done = 1; }
            else scal->alpha = scal->rho_new / gamma;
        }
    }
}

template <int n1>
static int launch_slab(semb_mesh* h, bool helm, double lambda, const double* lam0, const double* lam1,
                       const double* u, double* w, int nfields, semb_scalars* scal, cudaStream_t s)
{
    int64_t blocks = h->E * nfields;
    const int64_t cap = scal ? SEMB_MAX_BLOCKS : (int64_t)148 * 64;
    if (blocks > cap) blocks = cap;
    if (helm) k_axhelm_slab<n1, true><<<(unsigned)blocks, n1 * n1, 0, s>>>(h->E, h->n, h->geoK, lambda, lam0, lam1, u, w, nfields, scal, h->partials);
    else      k_axhelm_slab<n1, false><<<(unsigned)blocks, n1 * n1, 0, s>>>(h->E, h->n, h->geoK, lambda, lam0, lam1, u, w, nfields, scal, h->partials);
    SEMB_CUDA(h, cudaGetLastError());
    h->launches += 1;
    return SEMB_OK;
}

int semb_axhelm_launch(semb_mesh* h, double lambda, const double* lam0, const double* lam1,
                       const double* u, double* w, int nfields, semb_scalars* scal, cudaStream_t s)
{
    const bool helm = (lambda != 0.0) || lam1;
    switch (h->n1) {
        case 2:  return launch_slab<2>(h, helm, lambda, lam0, lam1, u, w, nfields, scal, s);
        case 3:  return launch_slab<3>(h, helm, lambda, lam0, lam1, u, w, nfields, scal, s);
        case 4:  return launch_slab<4>(h, helm, lambda, lam0, lam1, u, w, nfields, scal, s);
        case 5:  return launch_slab<5>(h, helm, lambda, lam0, lam1, u, w, nfields, scal, s);
        case 6:  return launch_slab<6>(h, helm, lambda, lam0, lam1, u, w, nfields, scal, s);
        case 7:  return launch_slab<7>(h, helm, lambda, lam0, lam1, u, w, nfields, scal, s);
        case 8:  return launch_slab<8>(h, helm, lambda, lam0, lam1, u, w, nfields, scal, s);
        case 9:  return launch_slab<9>(h, helm, lambda, lam0, lam1, u, w, nfields, scal, s);
        case 10: return launch_slab<10>(h, helm, lambda, lam0, lam1, u, w, nfields, scal, s);
        case 11: return launch_slab<11>(h, helm, lambda, lam0, lam1, u, w, nfields, scal, s);
    }
    return semb_fail(h, SEMB_EINVAL, "unsupported order N=%d", h->N);
}
