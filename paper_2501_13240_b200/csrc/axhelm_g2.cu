// axhelm kernels of geometry representation SEMB_GEO_AFFINE (axhelm_kernels.cuh), their own translation unit
#include "axhelm_launch.cuh"

int semb_axhelm_g2_upload(semb_mesh* h) { return ax_upload_basis_tu(h); }

int semb_axhelm_g2_dispatch(semb_mesh* h, const void* geo, int mode, double lambda, const double* u, double* w, int nfields,
                            semb_scalars* scal, bool want_dot, const ax_pcg_args& pcg, cudaStream_t s)
{
    return axhelm_dispatch<double, SEMB_GEO_AFFINE>(h, geo, mode, lambda, nullptr, nullptr, u, w, nfields, scal, want_dot, pcg, s);
}
