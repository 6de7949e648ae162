// axhelm: the matrix-free local operator  w = D^T G D u + lambda B u  per hexahedral element
// (BASELINE.json:north_star; §2.2 "matrix-free ... tensor-product contractions with
// (p+1)x(p+1) operator matrices identical for all elements", O(N_e p^4) work on O(N_e p^3) data).
//
//   u_r = sum_m D_im u(m,j,k)   u_s = sum_m D_jm u(i,m,k)   u_t = sum_m D_km u(i,j,m)
//   g_r = G_rr u_r + G_rs u_s + G_rt u_t,  g_s = G_rs u_r + G_ss u_s + G_st u_t,  g_t = G_rt u_r + G_st u_s + G_tt u_t
//   w(i,j,k) = sum_m D_mi g_r(m,j,k) + sum_m D_mj g_s(i,m,k) + sum_m D_mk g_t(i,j,m) + lambda B u
//
// Algorithmic bytes per node: 8 (u) + 8 (w) + 48 (G) = 64, + 8 (B) when lambda != 0.
#include "axhelm_launch.cuh"

int semb_axhelm_upload_basis(semb_mesh* h)
{
    int rc = ax_upload_basis_tu(h);
    if (!rc) rc = semb_axhelm_g1_upload(h);
    if (!rc) rc = semb_axhelm_g2_upload(h);
    if (!rc) rc = semb_axhelm_g3_upload(h);
    return rc;
}

int64_t semb_axhelm_dot_count(semb_mesh* h)
{
    switch (h->n1) {
        case 2: return ax_dot_count_of<2>(h);  case 3: return ax_dot_count_of<3>(h);  case 4: return ax_dot_count_of<4>(h);
        case 5: return ax_dot_count_of<5>(h);  case 6: return ax_dot_count_of<6>(h);  case 7: return ax_dot_count_of<7>(h);
        case 8: return ax_dot_count_of<8>(h);  case 9: return ax_dot_count_of<9>(h);  case 10: return ax_dot_count_of<10>(h);
        default: return ax_dot_count_of<11>(h);
    }
}

int semb_axhelm_prepare_geo(semb_mesh* h, cudaStream_t) { h->geoK = h->geo; return SEMB_OK; }

// every fp64 application on the handle's own geometry goes through here: the representation semb_set_geometry_mode selected
static int axhelm_by_mode(semb_mesh* h, int mode, double lambda, const double* lam0, const double* lam1, const double* u, double* w,
                          int nfields, semb_scalars* scal, bool want_dot, const ax_pcg_args& pcg, cudaStream_t s)
{
    if (h->geo_mode != SEMB_GEO_STORED && (mode & 2)) return semb_fail(h, SEMB_EINVAL, "axhelm: coefficient fields need the stored fp64 factors (geometry mode 0)");
    switch (h->geo_mode) {
        case SEMB_GEO_F32:       return semb_axhelm_g1_dispatch(h, h->geoF, mode, lambda, u, w, nfields, scal, want_dot, pcg, s);
        case SEMB_GEO_AFFINE:    return semb_axhelm_g2_dispatch(h, h->geoC, mode, lambda, u, w, nfields, scal, want_dot, pcg, s);
        case SEMB_GEO_TRILINEAR: return semb_axhelm_g3_dispatch(h, h->geoT, mode, lambda, u, w, nfields, scal, want_dot, pcg, s);
        default:                 return axhelm_dispatch<double, SEMB_GEO_STORED>(h, h->geoK, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
    }
}

int semb_axhelm_launch(semb_mesh* h, double lambda, const double* lam0, const double* lam1,
                       const double* u, double* w, int nfields, semb_scalars* scal, cudaStream_t s)
{
    const int mode = (lam0 || lam1) ? 3 : (lambda != 0.0) ? 1 : 0;
    return axhelm_by_mode(h, mode, lambda, lam0, lam1, u, w, nfields, scal, scal != nullptr, ax_pcg_args{nullptr, nullptr, nullptr, nullptr, 1.0, 0}, s);
}

// PCG-fused form (pcg.cu): x += alpha p_old (if pending), p = dinv o zsrc + beta p_old, q = A_L p, partial p.q;
// then p.Ap and alpha.  dinv may be NULL (z = zsrc).
int semb_axhelm_pcg_launch(semb_mesh* h, double lambda, const double* zsrc, const double* dinv, double* p, double* x,
                           double* q, semb_scalars* scal, cudaStream_t s)
{
    const int mode = 4 | ((lambda != 0.0) ? 1 : 0);
    return axhelm_by_mode(h, mode, lambda, nullptr, nullptr, nullptr, q, 1, scal, true, ax_pcg_args{zsrc, dinv, p, x, 1.0, 0}, s);
}

// First Chebyshev step fused into the operator (pcg.cu: cheb_apply): d = (dinv o r) * scale, written to d, Ad = A_L d.
// scal (may be NULL) only provides the early exit of a stopped solve.  Algorithmic bytes: r, dinv, 6 G read, d, Ad written = 80.
int semb_axhelm_scaled_launch(semb_mesh* h, double lambda, const double* r, const double* dinv, double scale, double* d,
                              double* Ad, semb_scalars* scal, cudaStream_t s)
{
    const int mode = 4 | ((lambda != 0.0) ? 1 : 0);
    return axhelm_by_mode(h, mode, lambda, nullptr, nullptr, nullptr, Ad, 1, scal, false, ax_pcg_args{r, dinv, d, nullptr, scale, 1}, s);
}

// ---- fp32-storage variants for the multigrid levels (geo: float copy of the level's factors, [E][7][Np])
int semb_axhelm_launch_f(semb_mesh* h, double lambda, const float* geo, const float* u, float* w, semb_scalars* scal, cudaStream_t s)
{
    const int mode = (lambda != 0.0) ? 1 : 0;
    return axhelm_dispatch<float, SEMB_GEO_STORED>(h, geo, mode, lambda, nullptr, nullptr, u, w, 1, scal, false, ax_pcg_args_t<float>{nullptr, nullptr, nullptr, nullptr, 1.0, 0}, s);
}
int semb_axhelm_scaled_launch_f(semb_mesh* h, double lambda, const float* geo, const float* r, const float* dinv, double scale, float* d,
                                float* Ad, semb_scalars* scal, cudaStream_t s)
{
    const int mode = 4 | ((lambda != 0.0) ? 1 : 0);
    return axhelm_dispatch<float, SEMB_GEO_STORED>(h, geo, mode, lambda, nullptr, nullptr, nullptr, Ad, 1, scal, false, ax_pcg_args_t<float>{r, dinv, d, nullptr, scale, 1}, s);
}
