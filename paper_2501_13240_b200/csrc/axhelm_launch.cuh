// Launch machinery of the axhelm kernels, shared by the translation units that instantiate them (one per geometry
// representation, so that they compile in parallel; every unit has its own copy of the __constant__ tables and uploads it).
#pragma once
#include <cstdlib>
#include "axhelm_kernels.cuh"
#ifndef SEMB_AX_STAGE
#define SEMB_AX_STAGE 1          // N = 9 stand-alone launches use k_axhelm_stage (env SEMB_AX_STAGE=0/1 overrides at run time)
#endif

// one translation unit per on-the-fly / reduced-precision geometry representation
#define SEMB_AX_GEO_TU(G) \
    int semb_axhelm_g##G##_upload(semb_mesh* h); \
    int semb_axhelm_g##G##_dispatch(semb_mesh* h, const void* geo, int mode, double lambda, const double* u, double* w, int nfields, \
                                  semb_scalars* scal, bool want_dot, const ax_pcg_args& pcg, cudaStream_t s);
SEMB_AX_GEO_TU(1) SEMB_AX_GEO_TU(2) SEMB_AX_GEO_TU(3)
#undef SEMB_AX_GEO_TU

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

static int ax_upload_basis_tu(semb_mesh* h)
{
    SEMB_CUDA(h, cudaMemcpyToSymbol(c_xi, h->xi, sizeof(double) * h->n1, sizeof(double) * SEMB_MAXN1 * (size_t)h->N));
    SEMB_CUDA(h, cudaMemcpyToSymbol(c_rho, h->rho, sizeof(double) * h->n1, sizeof(double) * SEMB_MAXN1 * (size_t)h->N));
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

// resident blocks per SM asked of the compiler (register budget): measured on B200, N = 7: 4 blocks x 166
// registers beat 8 x 128 (the 48 geometric-factor loads of a thread stay in flight without spills).
#ifndef SEMB_MINB10
#define SEMB_MINB10 3
#endif
// elements per block (axhelm_kernels.cuh): small orders pack several elements into one block of ~128 threads
#ifndef SEMB_EPB5
#define SEMB_EPB5 1
#define SEMB_MINB5 8
#endif
// N = 5 (Table 4 runs Ra = 1e11 at p = 5): one 36-thread block per element leaves the second warp with 4 live
// lanes; 3 elements per 108-thread block, 4 blocks per SM: stored 105.9 -> 111.0 GDOF/s, affine 118.8 -> 164.5 (B200, 49 M nodes).
// Measured and rejected: 4 elements (108.7 / 131.9), 7 elements (106.3 / 61.9); N = 4: 3, 5, 10 per block and N = 6: 2, 3, 5 per
// block were all slower than one element per block.
#ifndef SEMB_EPB6
#define SEMB_EPB6 3
#define SEMB_MINB6 4
#endif
#ifndef SEMB_EPB7
#define SEMB_EPB7 1
#define SEMB_MINB7 4
#endif
#ifndef SEMB_EPB10
#define SEMB_EPB10 1
#endif
template <int n1> struct ax_epb { static constexpr int v = (n1 == 2) ? 32 : (n1 == 3) ? 14 : (n1 == 4) ? 8 : (n1 == 5) ? SEMB_EPB5 : (n1 == 6) ? SEMB_EPB6 : (n1 == 7) ? SEMB_EPB7 : (n1 == 10) ? SEMB_EPB10 : 1; };
#ifndef SEMB_MINB8_G3
#define SEMB_MINB8_G3 8
#endif
#ifndef SEMB_MINB8_G2
#define SEMB_MINB8_G2 10
#endif
template <int n1, int GEO> struct ax_minb { static constexpr int v = (n1 <= 4) ? 8 : (n1 == 5) ? SEMB_MINB5 : (n1 == 6) ? SEMB_MINB6 : (n1 == 7) ? SEMB_MINB7 : (n1 <= 8) ? 4 : (n1 == 9) ? 4 : (n1 == 10) ? SEMB_MINB10 : 3; };
// the trilinear mode keeps 15 map coefficients per thread and rebuilds nine cofactors per node: the 64-register budget of
// the packed small orders spilled 100-260 bytes
template <int n1> struct ax_minb<n1, SEMB_GEO_TRILINEAR> { static constexpr int v = (n1 <= 4) ? 4 : (n1 <= 6) ? 6 : (n1 <= 8) ? SEMB_MINB8_G3 : 3; };
#ifndef SEMB_MINB8_G1
#define SEMB_MINB8_G1 8
#endif
template <int n1> struct ax_minb<n1, SEMB_GEO_F32> { static constexpr int v = (n1 <= 4) ? 8 : (n1 <= 6) ? 8 : (n1 <= 8) ? SEMB_MINB8_G1 : (n1 == 9) ? 4 : (n1 == 10) ? SEMB_MINB10 : 3; };
template <int n1> struct ax_minb<n1, SEMB_GEO_AFFINE> { static constexpr int v = (n1 <= 4) ? 8 : (n1 <= 6) ? 8 : (n1 <= 8) ? SEMB_MINB8_G2 : (n1 == 9) ? 4 : (n1 == 10) ? SEMB_MINB10 : 3; };

template <int n1, typename ST, int GEO>
static int launch_line(semb_mesh* h, const void* geo, int mode, double lambda, const double* lam0, const double* lam1,
                       const ST* u, ST* w, int nfields, semb_scalars* scal, bool want_dot, const ax_pcg_args_t<ST>& pcg, cudaStream_t s)
{
    constexpr int MB = ax_minb<n1, GEO>::v, EPB = ax_epb<n1>::v;
    const unsigned grid = (unsigned)((h->E * nfields + EPB - 1) / EPB);
    double* dot = (scal && want_dot) ? h->ax_dot : nullptr;
    // L2 prefetch distance in elements: about 8 MB of this launch's traffic ahead of the block that issues it.
    // Measured on B200 (N = 3, 5, 7, 9, stand-alone and PCG-fused): 4-20 MB ahead is flat (N = 7 Poisson 6.2 -> 7.05 TB/s,
    // N = 9 4.5 -> 5.7 TB/s), beyond ~30 MB the prefetched lines are evicted before use and the launch gets SLOWER
    // than without prefetch.
    const int gsub = (GEO == SEMB_GEO_F32) ? ((mode & 1) ? 28 : 24) : (GEO >= SEMB_GEO_AFFINE) ? ((mode & 1) ? 56 : 48) : 0;   // bytes of G this mode does not read
    const int64_t bytes_per_elem = (int64_t)n1 * n1 * n1 * (((mode & 4) ? (pcg.plain ? 80 : 104) : (mode & 2) ? 88 : (mode & 1) ? 72 : 64) - gsub)
                                   * (int64_t)sizeof(ST) / 8;
    const int pf = (int)(((int64_t)8 << 20) / bytes_per_elem);
    // N = 9, fp64 stored factors, stand-alone Poisson / Helmholtz: the persistent kernel with TMA-staged factors
    if constexpr ((n1 == 10 || n1 == 8) && sizeof(ST) == 8 && GEO == SEMB_GEO_STORED) {
        static const int stage_on = [] { const char* v = getenv("SEMB_AX_STAGE"); return v ? atoi(v) : SEMB_AX_STAGE; }();
        if (stage_on && !scal && (mode == 0 || mode == 1) && ((uintptr_t)geo & 15) == 0 && (n1 == 10 || nfields >= 2)) {       // N = 7: several fields only
            constexpr size_t smem = ax_stage_smem<n1>::bytes;
            auto kern = (mode & 1) ? k_axhelm_stage<n1, true> : k_axhelm_stage<n1, false>;
            static int per_sm[2][64] = {{0}};                      // per device: the opt-in shared-memory size is a per-device attribute
            int devid = 0;
            SEMB_CUDA(h, cudaGetDevice(&devid));
            int& nb_dev = per_sm[mode & 1][devid & 63];
            if (!nb_dev) {
                SEMB_CUDA(h, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
                int nb = 0;
                SEMB_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, n1 * n1, smem));
                nb_dev = nb > 0 ? nb : 1;
            }
            const int64_t nef = h->E, cap = (int64_t)nb_dev * semb_sm_count();                  // one block walks over elements, all fields of each
            kern<<<(unsigned)(nef < cap ? nef : cap), n1 * n1, smem, s>>>(h->E, h->n, (const double*)geo, lambda, (const double*)u, (double*)w, nfields);
            h->launches += 1;
            SEMB_CUDA(h, cudaGetLastError());
            return SEMB_OK;
        }
    }
#define SEMB_AX_LAUNCH(M) k_axhelm_line<n1, M, MB, EPB, ST, GEO><<<grid, n1 * n1 * EPB, 0, s>>>(h->E, h->n, geo, lambda, lam0, lam1, u, w, scal, dot, pcg, pf, nfields)
    switch (mode) {
        case 0: if (SEMB_AX_FIELD_FAST && nfields > 1) SEMB_AX_LAUNCH(8); else SEMB_AX_LAUNCH(0); break;
        case 1: if (SEMB_AX_FIELD_FAST && nfields > 1) SEMB_AX_LAUNCH(9); else SEMB_AX_LAUNCH(1); break;
        case 3: if constexpr (GEO == SEMB_GEO_STORED) { SEMB_AX_LAUNCH(3); break; } else return semb_fail(h, SEMB_EINVAL, "axhelm: coefficient fields need stored fp64 factors");
        case 4: SEMB_AX_LAUNCH(4); break;
        case 5: SEMB_AX_LAUNCH(5); break;
        default: return semb_fail(h, SEMB_EINVAL, "axhelm: unsupported mode %d", mode);
    }
#undef SEMB_AX_LAUNCH
    h->launches += 1;
    if (dot && !h->defer_dot_finish) {
        // p.Ap = sum of the per-element partials, alpha = rho / p.Ap (fixed order: bit-reproducible)
        int64_t blocks = ((int64_t)grid + 2047) / 2048;
        if (blocks > 128) blocks = 128;
        k_ax_dot_finish<<<(unsigned)blocks, 256, 0, s>>>((int64_t)grid, dot, scal, h->partials);     // one partial per block
        h->launches += 1;
    }
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}

template <int n1> static int64_t ax_dot_count_of(semb_mesh* h) { return (h->E + ax_epb<n1>::v - 1) / ax_epb<n1>::v; }

template <typename ST, int GEO>
static int axhelm_dispatch(semb_mesh* h, const void* geo, int mode, double lambda, const double* lam0, const double* lam1,
                           const ST* u, ST* w, int nfields, semb_scalars* scal, bool want_dot, const ax_pcg_args_t<ST>& pcg, cudaStream_t s)
{
    if (sizeof(ST) < 8 && (mode & 2)) return semb_fail(h, SEMB_EINVAL, "axhelm: coefficient fields need fp64 storage");
    if (scal && nfields != 1) return semb_fail(h, SEMB_EINVAL, "axhelm: fused p.Ap needs nfields == 1");
    if (scal && want_dot && !h->ax_dot) {
        h->ax_dot = (double*)semb_dev_alloc(h, sizeof(double) * (size_t)h->E);
        if (!h->ax_dot) return semb_fail(h, SEMB_ENOMEM, "axhelm: p.Ap partials");
    }
    switch (h->n1) {
        case 2:  return launch_line<2, ST, GEO>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 3:  return launch_line<3, ST, GEO>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 4:  return launch_line<4, ST, GEO>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 5:  return launch_line<5, ST, GEO>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 6:  return launch_line<6, ST, GEO>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 7:  return launch_line<7, ST, GEO>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 8:  return launch_line<8, ST, GEO>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 9:  return launch_line<9, ST, GEO>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 10: return launch_line<10, ST, GEO>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
        case 11: return launch_line<11, ST, GEO>(h, geo, mode, lambda, lam0, lam1, u, w, nfields, scal, want_dot, pcg, s);
    }
    return semb_fail(h, SEMB_EINVAL, "unsupported order N=%d", h->N);
}

