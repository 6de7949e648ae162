// axhelm: the matrix-free local operator  w = D^T G D u + lambda B u  per hexahedral element
// (BASELINE.json:north_star; §2.2 "matrix-free ... tensor-product contractions with
// (p+1)x(p+1) operator matrices identical for all elements", O(N_e p^4) work on O(N_e p^3) data).
//
//   u_r = sum_m D_im u(m,j,k)   u_s = sum_m D_jm u(i,m,k)   u_t = sum_m D_km u(i,j,m)
//   g_r = G_rr u_r + G_rs u_s + G_rt u_t,  g_s = G_rs u_r + G_ss u_s + G_st u_t,  g_t = G_rt u_r + G_st u_s + G_tt u_t
//   w(i,j,k) = sum_m D_mi g_r(m,j,k) + sum_m D_mj g_s(i,m,k) + sum_m D_mk g_t(i,j,m) + lambda B u
//
// Algorithmic bytes per node: 8 (u) + 8 (w) + 48 (G) = 64, + 8 (B) when lambda != 0.
#include "axhelm_kernels.cuh"

template <int n1> static void perm_of(unsigned char perm[2][SEMB_MAXN1 * SEMB_MAXN1 + 7])
{
    using T = ax_tile<n1>;
    ax_perm_build(n1, T::P1, T::P2, T::P2B, T::permuted, perm);
}
static int upload_perm(semb_mesh* h)
{
    unsigned char perm[2][SEMB_MAXN1 * SEMB_MAXN1 + 7] = {{0}};
    switch (h->n1) {
        case 2: perm_of<2>(perm); break;   case 3: perm_of<3>(perm); break;   case 4: perm_of<4>(perm); break;
        case 5: perm_of<5>(perm); break;   case 6: perm_of<6>(perm); break;   case 7: perm_of<7>(perm); break;
        case 8: perm_of<8>(perm); break;   case 9: perm_of<9>(perm); break;   case 10: perm_of<10>(perm); break;
        case 11: perm_of<11>(perm); break;
        default: return semb_fail(h, SEMB_EINVAL, "unsupported order N=%d", h->N);
    }
    SEMB_CUDA(h, cudaMemcpyToSymbol(c_perm, perm, sizeof(perm), sizeof(perm) * (size_t)h->N));
    return SEMB_OK;
}

int semb_axhelm_upload_basis(semb_mesh* h)
{
    SEMB_CUDA(h, cudaMemcpyToSymbol(c_D, h->D, sizeof(double) * h->n1 * h->n1,
                                    sizeof(double) * SEMB_MAXN1 * SEMB_MAXN1 * (size_t)h->N));
    ax_eo_tab tab[2];
    ax_eo_build(h->n1, h->D, tab);
    SEMB_CUDA(h, cudaMemcpyToSymbol(c_EO, tab, sizeof(tab), sizeof(ax_eo_tab) * 2 * (size_t)h->N));
    ax_eo_tab_f tabf[2];
    for (int t = 0; t < 2; ++t) {
        for (int q = 0; q < SEMB_EO_H2 * SEMB_EO_H; ++q) { tabf[t].P[q] = (float)tab[t].P[q]; tabf[t].M[q] = (float)tab[t].M[q]; }
        for (int q = 0; q < SEMB_EO_H2; ++q) tabf[t].mid[q] = (float)tab[t].mid[q];
    }
    SEMB_CUDA(h, cudaMemcpyToSymbol(c_EOf, tabf, sizeof(tabf), sizeof(ax_eo_tab_f) * 2 * (size_t)h->N));
    return upload_perm(h);
}

int semb_axhelm_prepare_geo(semb_mesh* h, cudaStream_t) { h->geoK = h->geo; return SEMB_OK; }

// resident blocks per SM asked of the compiler (register budget): measured on B200, N = 7: 4 blocks x 166
// registers beat 8 x 128 (the 48 geometric-factor loads of a thread stay in flight without spills).
#ifndef SEMB_MINB10
#define SEMB_MINB10 3
#endif
// elements per block (axhelm_kernels.cuh): small orders pack several elements into one block of ~128 threads
template <int n1> struct ax_epb { static constexpr int v = (n1 == 2) ? 32 : (n1 == 3) ? 14 : (n1 == 4) ? 8 : 1; };
template <int n1> struct ax_minb { static constexpr int v = (n1 <= 4) ? 8 : (n1 <= 6) ? 8 : (n1 <= 8) ? 4 : (n1 == 9) ? 4 : (n1 == 10) ? SEMB_MINB10 : 3; };

template <int n1, typename ST>
static int launch_line(semb_mesh* h, const ST* geo, int mode, double lambda, const double* lam0, const double* lam1,
                       const ST* u, ST* w, int nfields, semb_scalars* scal, bool want_dot, const ax_pcg_args_t<ST>& pcg, cudaStream_t s)
{
    constexpr int MB = ax_minb<n1>::v, EPB = ax_epb<n1>::v;
    const unsigned grid = (unsigned)((h->E * nfields + EPB - 1) / EPB);
    double* dot = (scal && want_dot) ? h->ax_dot : nullptr;
    // L2 prefetch distance in elements: about 8 MB of this launch's traffic ahead of the block that issues it.
    // Measured on B200 (N = 3, 5, 7, 9, stand-alone and PCG-fused): 4-20 MB ahead is flat (N = 7 Poisson 6.2 -> 7.05 TB/s,
    // N = 9 4.5 -> 5.7 TB/s), beyond ~30 MB the prefetched lines are evicted before use and the launch gets SLOWER
    // than without prefetch.
    const int64_t bytes_per_elem = (int64_t)n1 * n1 * n1 * ((mode & 4) ? (pcg.plain ? 80 : 104) : (mode & 2) ? 88 : (mode & 1) ? 72 : 64)
                                   * (int64_t)sizeof(ST) / 8;
    const int pf = (int)(((int64_t)8 << 20) / bytes_per_elem);
#define SEMB_AX_LAUNCH(M) k_axhelm_line<n1, M, MB, EPB, ST><<<grid, n1 * n1 * EPB, 0, s>>>(h->E, h->n, geo, lambda, lam0, lam1, u, w, scal, dot, pcg, pf, nfields)
    switch (mode) {
        case 0: SEMB_AX_LAUNCH(0); break;
        case 1: SEMB_AX_LAUNCH(1); break;
        case 3: SEMB_AX_LAUNCH(3); break;
        case 4: SEMB_AX_LAUNCH(4); break;
        case 5: SEMB_AX_LAUNCH(5); break;
        default: return semb_fail(h, SEMB_EINVAL, "axhelm: unsupported mode %d", mode);
    }
#undef SEMB_AX_LAUNCH
    h->launches += 1;
    if (dot) {
        // p.Ap = sum of the per-element partials, alpha = rho / p.Ap (fixed order: bit-reproducible)
        int64_t blocks = ((int64_t)grid + 2047) / 2048;
        if (blocks > 128) blocks = 128;
        k_ax_dot_finish<<<(unsigned)blocks, 256, 0, s>>>((int64_t)grid, dot, scal, h->partials);     // one partial per block
        h->launches += 1;
    }
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}

template <typename ST>
static int axhelm_dispatch(semb_mesh* h, const ST* geo, int mode, double lambda, const double* lam0, const double* lam1,
                           const ST* u, ST* w, int nfields, semb_scalars* scal, bool want_dot, const ax_pcg_args_t<ST>& pcg, cudaStream_t s)
{
    if (sizeof(ST) < 8 && (mode & 2)) return semb_fail(h, SEMB_EINVAL, "axhelm: coefficient fields need fp64 storage");
    if (scal && nfields != 1) return semb_fail(h, SEMB_EINVAL, "axhelm: fused p.Ap needs nfields == 1");
    if (scal && want_dot && !h->ax_dot) {
        h->ax_dot = (double*)semb_dev_alloc(h, sizeof(double) * (size_t)h->E);
        if (!h->ax_dot) return semb_fail(h, SEMB_ENOMEM, "axhelm: p.Ap partials");
    }
    switch (h->n1) {
        case 2:  return launch_line<2, ST>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 3:  return launch_line<3, ST>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 4:  return launch_line<4, ST>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 5:  return launch_line<5, ST>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 6:  return launch_line<6, ST>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 7:  return launch_line<7, ST>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 8:  return launch_line<8, ST>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 9:  return launch_line<9, ST>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 10: return launch_line<10, ST>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 11: return launch_line<11, ST>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
    }
    return semb_fail(h, SEMB_EINVAL, "unsupported order N=%d", h->N);
}

int semb_axhelm_launch(semb_mesh* h, double lambda, const double* lam0, const double* lam1,
                       const double* u, double* w, int nfields, semb_scalars* scal, cudaStream_t s)
{
    const int mode = (lam0 || lam1) ? 3 : (lambda != 0.0) ? 1 : 0;
    return axhelm_dispatch<double>(h, h->geoK, mode, lambda, lam0, lam1, u, w, nfields, scal, scal != nullptr, ax_pcg_args{nullptr, nullptr, nullptr, nullptr, 1.0, 0}, s);
}

// PCG-fused form (pcg.cu): x += alpha p_old (if pending), p = dinv o zsrc + beta p_old, q = A_L p, partial p.q;
// then p.Ap and alpha.  dinv may be NULL (z = zsrc).
int semb_axhelm_pcg_launch(semb_mesh* h, double lambda, const double* zsrc, const double* dinv, double* p, double* x,
                           double* q, semb_scalars* scal, cudaStream_t s)
{
    const int mode = 4 | ((lambda != 0.0) ? 1 : 0);
    return axhelm_dispatch<double>(h, h->geoK, mode, lambda, nullptr, nullptr, nullptr, q, 1, scal, true, ax_pcg_args{zsrc, dinv, p, x, 1.0, 0}, s);
}

// First Chebyshev step fused into the operator (pcg.cu: cheb_apply): d = (dinv o r) * scale, written to d, Ad = A_L d.
// scal (may be NULL) only provides the early exit of a stopped solve.  Algorithmic bytes: r, dinv, 6 G read, d, Ad written = 80.
int semb_axhelm_scaled_launch(semb_mesh* h, double lambda, const double* r, const double* dinv, double scale, double* d,
                              double* Ad, semb_scalars* scal, cudaStream_t s)
{
    const int mode = 4 | ((lambda != 0.0) ? 1 : 0);
    return axhelm_dispatch<double>(h, h->geoK, mode, lambda, nullptr, nullptr, nullptr, Ad, 1, scal, false, ax_pcg_args{r, dinv, d, nullptr, scale, 1}, s);
}

// ---- fp32-storage variants for the multigrid levels (geo: float copy of the level's factors, [E][7][Np])
int semb_axhelm_launch_f(semb_mesh* h, double lambda, const float* geo, const float* u, float* w, semb_scalars* scal, cudaStream_t s)
{
    const int mode = (lambda != 0.0) ? 1 : 0;
    return axhelm_dispatch<float>(h, geo, mode, lambda, nullptr, nullptr, u, w, 1, scal, false, ax_pcg_args_t<float>{nullptr, nullptr, nullptr, nullptr, 1.0, 0}, s);
}
int semb_axhelm_scaled_launch_f(semb_mesh* h, double lambda, const float* geo, const float* r, const float* dinv, double scale, float* d,
                                float* Ad, semb_scalars* scal, cudaStream_t s)
{
    const int mode = 4 | ((lambda != 0.0) ? 1 : 0);
    return axhelm_dispatch<float>(h, geo, mode, lambda, nullptr, nullptr, nullptr, Ad, 1, scal, false, ax_pcg_args_t<float>{r, dinv, d, nullptr, scale, 1}, s);
}
