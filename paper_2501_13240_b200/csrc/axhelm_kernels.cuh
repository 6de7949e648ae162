// axhelm device kernels (sm_100a, fp64):  w = D^T G D u + lambda B u  per hexahedral element
// (BASELINE.json:north_star; §2.2 "matrix-free ... tensor-product contractions with
// (p+1)x(p+1) operator matrices identical for all elements").
//
//   u_r = sum_m D_im u(m,j,k)   u_s = sum_m D_jm u(i,m,k)   u_t = sum_m D_km u(i,j,m)
//   g_r = G_rr u_r + G_rs u_s + G_rt u_t,  g_s = G_rs u_r + G_ss u_s + G_st u_t,  g_t = G_rt u_r + G_st u_s + G_tt u_t
//   w(i,j,k) = sum_m D_mi g_r(m,j,k) + sum_m D_mj g_s(i,m,k) + sum_m D_mk g_t(i,j,m) + lambda B u
//
// k_axhelm_line ("line" kernel, the production path).  One block of n1 x n1 threads per element.  Every one
// of the six contractions is done by a thread that holds a WHOLE line of n1 nodes in registers, so its n1 x n1
// multiply-adds take D from the constant bank (compile-time indices -> DFMA with a c[][] operand) and touch
// shared memory only to transpose between the three line orientations:
//     thread (a,b) owns   t-line (i=a, j=b, k=*)   -- also the layout of every global load/store (coalesced)
//                         r-line (i=*, j=a, k=b)
//                         s-line (i=a, j=*, k=b)
// Shared-memory traffic is 8 transposes x 16 B + 8 B = 136 B per node (about 1.06 wavefronts per node,
// conflict-free for n1 = 8 through the XOR swizzle below), against 3.7 wavefronts per node of the slab kernel
// that ncu showed to be bound by the shared-memory pipe (profiles/r1_v1_axhelm_full.md).
#pragma once
#include "reduce.cuh"
#include "semb_internal.h"

// D for every order 1..SEMB_MAX_N, row-major n1 x n1 at c_D[N]; filled at setup.
static __constant__ double c_D[SEMB_MAX_N + 1][SEMB_MAXN1 * SEMB_MAXN1];
// GLL nodes and weights per order (the on-the-fly geometry modes rebuild W = rho_i rho_j rho_k and the trilinear map from them)
static __constant__ double c_xi[SEMB_MAX_N + 1][SEMB_MAXN1], c_rho[SEMB_MAX_N + 1][SEMB_MAXN1];

// ---- geometry representations (semb_set_geometry_mode) -----------------------------------
//   GEO 0  stored factors, geo[E][7][Np] in the storage type ST                              48 (56) B/node
//   GEO 1  the same layout in float, widened exactly on load, fp64 arithmetic                 24 (28) B/node
//   GEO 2  affine elements (parallelepipeds): 7 constants per element, geoc[E][8] =
//          (1/J) C_a.C_b for ab = rr, rs, rt, ss, st, tt, then J; G_ab = rho_i rho_j rho_k * that    64 B/element
//   GEO 3  trilinear elements (straight edges): the 8 x 3 coefficients of x = c0 + c1 r + c2 s + c3 t + c4 rs + c5 rt
//          + c6 st + c7 rst per coordinate, tri[E][3][8]; the Jacobian, its cofactors C_r = x_s x x_t, C_s = x_t x x_r,
//          C_t = x_r x x_s and J = x_r . C_r are recomputed per node and G applied in factored form
//          g_a = (W / J) C_a . (C_r u_r + C_s u_s + C_t u_t)                                        192 B/element

#ifndef SEMB_AX_RELOAD_N1
#define SEMB_AX_RELOAD_N1 10
#endif
#ifndef SEMB_AX_FIELD_FAST
#define SEMB_AX_FIELD_FAST 1          // launches on several fields use the MODE | 8 instantiations; measured on B200, 3 fields:
#endif                                // N = 7 112 -> 141 GDOF/s (Helmholtz 100 -> 137), N = 5 106 -> 123, N = 3 101 -> 157
#ifndef SEMB_AX_SPLIT_N1
#define SEMB_AX_SPLIT_N1 99          // off by default until measured
#endif

// 1 / d for d > 0 in the normal range: hardware seed (2^-23) + two Newton steps (2^-46, 2^-92 -> rounding level)
__device__ __forceinline__ double ax_rcp(double d)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    r = fma(r, fma(-d, r, 1.0), r);
    r = fma(r, fma(-d, r, 1.0), r);
    return r;
}

// ---- shared-memory layout of one element tile, index (k,j,i) -> double slot -------------------------------
// All three line orientations read/write it with 64-bit accesses; a half-warp (16 lanes) is conflict-free iff
// its 16 slots are distinct mod 16.
// Generic n1: plain strides, row stride n1 (so the t-line pattern, slot = const + thread index, is always
// conflict-free), plane strides P2A (tiles Su, Sr) and P2B (tile Ss) chosen per n1 together with the assignment of
// r- and s-lines to threads (ax_perm_build) so that the 16 lines of each half-warp start in 16 different banks
// wherever the residues of the line starts allow it (exhaustive search over P2A, P2B in [n1^2, n1^2 + 16)).
template <int n1> struct ax_tile {
    static constexpr int P1 = n1;
    static constexpr int P2 = (n1 == 4) ? 19 : (n1 == 10) ? 103 : n1 * n1;                        // Su, Sr
    static constexpr int P2B = (n1 == 4) ? 19 : (n1 == 7) ? 57 : (n1 == 10) ? 101 : n1 * n1;       // Ss
    static constexpr int size = n1 * (P2 > P2B ? P2 : P2B);
    static constexpr int sizeA = (n1 - 1) * P2 + n1 * n1, sizeB = (n1 - 1) * P2B + n1 * n1;     // what idx / idxB really reach
    // measured on B200 (A/B in one session): N = 6 +5 %, N = 9 +3 % (Poisson) / +10 % (Helmholtz), N = 10 +7 %;
    // n1 = 9 was 3 % slower with its best permuted layout and n1 <= 6 within noise: those keep thread = line.
    static constexpr bool permuted = (n1 == 7) || (n1 >= 10);
    __device__ static __forceinline__ int idx(int k, int j, int i) { return k * P2 + j * P1 + i; }
    __device__ static __forceinline__ int idxB(int k, int j, int i) { return k * P2B + j * P1 + i; }
    __device__ static __forceinline__ int idx32(int k, int j, int i) { return idx(k, j, i); }       // no 32-bit layouts searched yet
};
// n1 = 8: XOR swizzle, conflict-free in all three orientations without padding:
//   slot mod 16 = ((j^k)&1)*8 + (i ^ (((j>>1)&3) | ((k&1)<<2)))
template <> struct ax_tile<8> {
    static constexpr int size = 512, sizeA = 512, sizeB = 512;
    static constexpr int P1 = 8, P2 = 64, P2B = 64;
    static constexpr bool permuted = false;
    __device__ static __forceinline__ int idx(int k, int j, int i)
    {
        return k * 64 + ((j ^ (k & 1)) << 3) + (i ^ (((j >> 1) & 3) | ((k & 1) << 2)));
    }
    __device__ static __forceinline__ int idxB(int k, int j, int i) { return idx(k, j, i); }
    // 32-bit tiles (float arithmetic on the fp32 multigrid levels): a warp covers 8 x 4 lines; word within plane k =
    // j[2]*32 + ((j[1:0] ^ k[1:0]) << 3) + (i ^ j[2:0]) puts the 32 lanes of all three orientations into 32 different banks
    __device__ static __forceinline__ int idx32(int k, int j, int i)
    {
        return k * 64 + ((j >> 2) << 5) + (((j ^ k) & 3) << 3) + (i ^ (j & 7));
    }
};

// Which r-line (j = q % n1, k = q / n1) and which s-line (i = q % n1, k = q / n1) a thread contracts:
// c_perm[N][0][thread] and c_perm[N][1][thread], filled at setup (axhelm.cu: ax_perm_build).
static __constant__ unsigned char c_perm[SEMB_MAX_N + 1][2][SEMB_MAXN1 * SEMB_MAXN1 + 7];

// host: greedy balanced grouping.  start_bank[q] = bank (64-bit, mod 16) of the first slot of line q.  Lines are
// dealt to the half-warps (aligned groups of 16 threads) so that a group holds as few lines of equal bank as
// possible; perm[thread] = line.
static inline void ax_perm_group(int nt, const int* start_bank, unsigned char* perm)
{
    const int ng = (nt + 15) / 16;
    int fill[16] = {0}, cnt[16][16] = {{0}}, members[16][16];
    int order[16], size[16] = {0};
    for (int q = 0; q < nt; ++q) size[start_bank[q]]++;
    for (int v = 0; v < 16; ++v) order[v] = v;
    for (int x = 0; x < 16; ++x) for (int y = x + 1; y < 16; ++y)
        if (size[order[y]] > size[order[x]] || (size[order[y]] == size[order[x]] && order[y] < order[x])) { int t = order[x]; order[x] = order[y]; order[y] = t; }
    for (int oi = 0; oi < 16; ++oi) {
        const int v = order[oi];
        for (int q = 0; q < nt; ++q) {
            if (start_bank[q] != v) continue;
            int best = -1;
            for (int g = 0; g < ng; ++g) {
                const int cap = (nt - 16 * g < 16) ? nt - 16 * g : 16;
                if (fill[g] >= cap) continue;
                if (best < 0) { best = g; continue; }
                const int capb = (nt - 16 * best < 16) ? nt - 16 * best : 16;
                if (cnt[g][v] < cnt[best][v] || (cnt[g][v] == cnt[best][v] && cap - fill[g] > capb - fill[best])) best = g;
            }
            members[best][fill[best]++] = q; cnt[best][v]++;
        }
    }
    int t = 0;
    for (int g = 0; g < ng; ++g) for (int x = 0; x < fill[g]; ++x) perm[t++] = (unsigned char)members[g][x];
}
static inline void ax_perm_build(int n1, int P1, int P2A, int P2B, bool permuted, unsigned char perm[2][SEMB_MAXN1 * SEMB_MAXN1 + 7])
{
    const int nt = n1 * n1;
    int bank[SEMB_MAXN1 * SEMB_MAXN1];
    if (!permuted) { for (int q = 0; q < nt; ++q) perm[0][q] = perm[1][q] = (unsigned char)q; return; }
    for (int q = 0; q < nt; ++q) bank[q] = ((q / n1) * P2A + (q % n1) * P1) % 16;     // r-line (j, k) in Su, Sr
    ax_perm_group(nt, bank, perm[0]);
    for (int q = 0; q < nt; ++q) bank[q] = ((q / n1) * P2B + (q % n1)) % 16;          // s-line (i, k) in Ss
    ax_perm_group(nt, bank, perm[1]);
}

// PCG epilogue shared by the kernels: grid-wide sum of u.w (= p.Ap before assembly, valid because p is
// continuous and zero at masked nodes: SURVEY.md §8 a-6), then alpha = rho / p.Ap in the last block.
__device__ __forceinline__ void ax_finish_dot(double dot, semb_scalars* __restrict__ scal, double* __restrict__ partials, double* red)
{
    double v[1] = { block_sum(dot, red) }, tot[1];
    if (grid_sum<1>(v, partials, &scal->ticket[0], tot, red) && threadIdx.x == 0) {
        const double gamma = tot[0];
        scal->pAp = gamma;
        if (!(gamma > 0.0) || !isfinite(gamma)) { scal->status = SEMB_EBREAKDOWN; scal->done = 1; scal->x_pending = 0; }
        else { scal->alpha = scal->rho_new / gamma; scal->x_pending = 1; }   // x += alpha p is applied by the next fused axhelm
    }
}

// ---- even-odd form of the line contractions ------------------------------------------------------------
// D (and D^T) are centro-antisymmetric, A[N-i][N-m] = -A[i][m], so with e_m = x_m + x_{N-m}, o_m = x_m - x_{N-m}
// (m < h = n1/2),  P_im = (A_im + A_i,N-m)/2,  M_im = (A_im - A_i,N-m)/2:
//     y_i = sum_m M_im o_m + a_i,   y_{N-i} = sum_m M_im o_m - a_i,   a_i = sum_m P_im e_m (+ A_ih x_h, n1 odd)
// and, for odd n1, the middle row y_h = sum_m M_hm o_m.  That is n1^2/2 multiply-adds plus 2 n1 additions per
// line instead of n1^2, and only n1^2/2 distinct constants, all at compile-time offsets of the constant bank.
#define SEMB_EO_H  ((SEMB_MAXN1) / 2)          // max h
#define SEMB_EO_H2 ((SEMB_MAXN1 + 1) / 2)      // max number of rows i <= h
struct ax_eo_tab { double P[SEMB_EO_H2 * SEMB_EO_H], M[SEMB_EO_H2 * SEMB_EO_H], mid[SEMB_EO_H2]; };
static __constant__ ax_eo_tab c_EO[SEMB_MAX_N + 1][2];      // [N][0] for D, [N][1] for D^T

// host: fill the two tables of order N from D (row-major n1 x n1)
static inline void ax_eo_build(int n1, const double* D, ax_eo_tab tab[2])
{
    const int N = n1 - 1, h = n1 / 2, h2 = (n1 + 1) / 2;
    for (int tr = 0; tr < 2; ++tr) {
        ax_eo_tab& T = tab[tr];
        for (auto& v : T.P) v = 0.0;
        for (auto& v : T.M) v = 0.0;
        for (auto& v : T.mid) v = 0.0;
        for (int i = 0; i < h2; ++i) {
            for (int m = 0; m < h; ++m) {
                const double x = tr ? D[m * n1 + i] : D[i * n1 + m], y = tr ? D[(N - m) * n1 + i] : D[i * n1 + (N - m)];
                T.P[i * SEMB_EO_H + m] = 0.5 * (x + y);
                T.M[i * SEMB_EO_H + m] = 0.5 * (x - y);
            }
            if (n1 & 1) T.mid[i] = tr ? D[h * n1 + i] : D[i * n1 + h];
        }
    }
}

// float copies of the tables for the fp32-storage multigrid levels, where the whole kernel computes in float
struct ax_eo_tab_f { float P[SEMB_EO_H2 * SEMB_EO_H], M[SEMB_EO_H2 * SEMB_EO_H], mid[SEMB_EO_H2]; };
static __constant__ ax_eo_tab_f c_EOf[SEMB_MAX_N + 1][2];
template <typename CT> struct ax_eo_sel;
template <> struct ax_eo_sel<double> { typedef ax_eo_tab tab; __device__ static __forceinline__ const ax_eo_tab& get(int N, int tr) { return c_EO[N][tr]; } };
template <> struct ax_eo_sel<float> { typedef ax_eo_tab_f tab; __device__ static __forceinline__ const ax_eo_tab_f& get(int N, int tr) { return c_EOf[N][tr]; } };

template <int n1, int TR, typename CT>
__device__ __forceinline__ void ax_line(const CT (&x)[n1], CT (&y)[n1])
{
    constexpr int N = n1 - 1, h = n1 / 2;
    constexpr bool odd = n1 & 1;
    const typename ax_eo_sel<CT>::tab& T = ax_eo_sel<CT>::get(N, TR);
    CT e[h > 0 ? h : 1], o[h > 0 ? h : 1];
#pragma unroll
    for (int m = 0; m < h; ++m) { e[m] = x[m] + x[N - m]; o[m] = x[m] - x[N - m]; }
#pragma unroll
    for (int i = 0; i < h; ++i) {
        CT a = odd ? T.mid[i] * x[h] : (CT)0, s = (CT)0;
#pragma unroll
        for (int m = 0; m < h; ++m) { a += T.P[i * SEMB_EO_H + m] * e[m]; s += T.M[i * SEMB_EO_H + m] * o[m]; }
        y[i] = s + a; y[N - i] = s - a;
    }
    if (odd) {
        CT s = (CT)0;
#pragma unroll
        for (int m = 0; m < h; ++m) s += T.M[h * SEMB_EO_H + m] * o[m];
        y[h] = s;
    }
}

// MODE bit 0: Helmholtz term lambda*B*u (7th factor);  bit 1: per-node coefficient fields lam0 / lam1;
// bit 2: PCG-fused prologue (nfields = 1): before the operator is applied the thread updates its own nodes
//     x += alpha * p_old  (the x-update of the PREVIOUS iteration, pending in scal)   and
//     p  = z + beta * p_old,  z = dinv o zsrc  (Jacobi), zsrc (none / Chebyshev's z)
// writes x and p back and applies the operator to the new p, so p is read once per iteration instead of three
// times (SURVEY.md §8 a-6 (iii),(iv) folded into (i)).  u is then unused; p_io is both input and output.
// One block per (element, field): grid = E * nfields.  dot_out != NULL: block b writes its partial sum of
// u.w to dot_out[b] (fixed summation order; reduced by k_ax_dot_finish).
// plain != 0 (first Chebyshev step): no recurrence, p = (dinv o zsrc) * scale is written to p_io and the operator is
// applied to it; x, alpha, beta are not touched.
template <typename ST, int GEO> struct ax_geo_type { typedef ST type; };
template <typename ST> struct ax_geo_type<ST, SEMB_GEO_F32> { typedef float type; };
template <typename ST> struct ax_pcg_args_t { const ST* zsrc; const ST* dinv; ST* p_io; ST* x; double scale; int plain; };
typedef ax_pcg_args_t<double> ax_pcg_args;

// L2 prefetch of one contiguous run of doubles (TMA unit, no destination in the SM):
// cp.async.bulk.prefetch.L2 needs a 16-byte aligned address and size; runs that are only 8-byte aligned (odd n1)
// are widened inward to the aligned part.  Issued by ONE thread.
template <typename ST>
__device__ __forceinline__ void ax_prefetch_l2(const ST* ptr, int count)
{
    uintptr_t a = (uintptr_t)ptr, b = a + (size_t)count * sizeof(ST);
    a = (a + 15) & ~(uintptr_t)15; b &= ~(uintptr_t)15;
    if (b > a) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(a), "r"((unsigned)(b - a)) : "memory");
}

// EPB elements per block (small orders: a block of n1^2 = 4, 9 or 16 threads per element cannot fill an SM -- the
// N = 1 level of the multigrid ran at 1 TB/s): thread group el = tl / n1^2 works on element
// blockIdx.x * EPB + el with its own shared-memory tiles; groups past the end recompute the last element and write nothing.
// ST: STORAGE type of the vectors and geometric factors in global memory (double, or float for the multigrid levels:
// PAPER.md:L102 runs the preconditioner in FP32 "to save on memory bandwidth"); float storage computes in float with 32-bit tiles,
// double storage in fp64 (R21).
template <int n1, int MODE, int MINB, int EPB, typename ST, int GEO>
__global__ void __launch_bounds__(n1 * n1 * EPB, MINB)
k_axhelm_line(int64_t E, int64_t n, const void* __restrict__ geo_v, double lambda,
              const double* __restrict__ lam0, const double* __restrict__ lam1,
              const ST* __restrict__ u, ST* __restrict__ w,
              const semb_scalars* __restrict__ scal, double* __restrict__ dot_out, ax_pcg_args_t<ST> pcg, int pf_dist, int nfields)
{
    constexpr int n2 = n1 * n1, Np = n1 * n1 * n1;
    constexpr bool HELM = MODE & 1, VAR = MODE & 2, FUSE = MODE & 4;
    constexpr int NG = HELM ? 7 : 6;
    constexpr bool STORED = GEO == SEMB_GEO_STORED || GEO == SEMB_GEO_F32;
    typedef typename ax_geo_type<ST, GEO>::type GT;             // what the stored factors are read as
    const GT* __restrict__ geo = (const GT*)geo_v;
    using T = ax_tile<n1>;
    typedef ST CT;                    // float storage => float arithmetic and 32-bit tiles (the fp64-arithmetic float-storage
                                      // kernel was bound by its 64-bit transposes at 138 GDOF/s: profiles/r1_v6_fp32_levels.md)
    constexpr bool W32 = sizeof(CT) == 4;
#define AX_I(k, j, i) (W32 ? T::idx32(k, j, i) : T::idx(k, j, i))
#define AX_IB(k, j, i) (W32 ? T::idx32(k, j, i) : T::idxB(k, j, i))
    __shared__ __align__(8) CT SuA[EPB * T::sizeA], SrA[EPB * T::sizeA], SsA[EPB * (W32 ? T::sizeA : T::sizeB)];
    if (scal && *(volatile const int32_t*)&scal->done) return;
    const int el = (EPB > 1) ? threadIdx.x / n2 : 0, tl = (EPB > 1) ? threadIdx.x - el * n2 : threadIdx.x;
    CT* __restrict__ Su = SuA + el * T::sizeA; CT* __restrict__ Sr = SrA + el * T::sizeA; CT* __restrict__ Ss = SsA + el * (W32 ? T::sizeA : T::sizeB);
    const int64_t nef = E * (int64_t)nfields;
    int64_t ef = blockIdx.x * (int64_t)EPB + el;
    const bool valid = ef < nef;
    if (!valid) ef = nef - 1;
    const int a = tl % n1, b = tl / n1;
    int ra = a, rb = b, sa = a, sb = b;                                     // r-line (j=ra, k=rb), s-line (i=sa, k=sb)
    if (T::permuted) {
        const int rq = c_perm[n1 - 1][0][tl], sq = c_perm[n1 - 1][1][tl];
        ra = rq % n1; rb = rq / n1; sa = sq % n1; sb = sq / n1;
    }
    // MODE bit 3 (launches on several fields): the fields of an element sit in neighbouring blocks, so its factors cross DRAM once and
    // the other fields read them from L2.  Single-field launches keep the instantiation without the bit: their code is unchanged.
    constexpr bool FF = (MODE & 8) != 0;
    const int64_t e = FF ? ef / nfields : ef % E, f = FF ? ef - (ef / nfields) * nfields : ef / E;
    // The element that a block pf_dist launches later will work on is pulled into L2 now: DRAM stays busy while
    // the resident blocks are in their compute phase, and that block's loads hit L2.
    if (pf_dist > 0 && tl == 0 && valid && e + pf_dist < E) {
        const int64_t ep = e + pf_dist;
        if (STORED && (!FF || f == 0)) ax_prefetch_l2(geo + ep * 7 * (int64_t)Np, NG * Np);
        if (FUSE) {
            ax_prefetch_l2(pcg.zsrc + ep * Np, Np);
            if (pcg.dinv) ax_prefetch_l2(pcg.dinv + ep * Np, Np);
            if (!pcg.plain) { ax_prefetch_l2(pcg.p_io + ep * Np, Np); ax_prefetch_l2(pcg.x + ep * Np, Np); }
        } else ax_prefetch_l2(u + f * n + ep * Np, Np);
        if (VAR && lam0) ax_prefetch_l2(lam0 + ep * Np, Np);
        if (VAR && lam1) ax_prefetch_l2(lam1 + ep * Np, Np);
    }
    ST* __restrict__ we = w + f * n + e * Np + tl;
    const GT* __restrict__ g = geo + e * 7 * (int64_t)Np + tl;
    CT ru[n1], G[STORED ? NG : 1][STORED ? n1 : 1];
    if (FUSE) {
        const int64_t l0 = e * Np + tl;
        const bool plain = pcg.plain != 0;
        const CT beta = plain ? (CT)0 : (CT)scal->beta, alpha = plain ? (CT)0 : (CT)scal->alpha;
        const bool pend = !plain && scal->x_pending != 0, first = plain || (beta == (CT)0);
        const CT pscale = (CT)pcg.scale;
        CT z[n1], po[n1];
#pragma unroll
        for (int k = 0; k < n1; ++k) z[k] = pcg.zsrc[l0 + k * n2];
        if (pcg.dinv) {
#pragma unroll
            for (int k = 0; k < n1; ++k) z[k] *= pcg.dinv[l0 + k * n2];
        }
        if (plain) {
#pragma unroll
            for (int k = 0; k < n1; ++k) z[k] *= pscale;
        }
        if (pend || !first) {
#pragma unroll
            for (int k = 0; k < n1; ++k) po[k] = pcg.p_io[l0 + k * n2];
        }
        if (pend) {
#pragma unroll
            for (int k = 0; k < n1; ++k) if (valid) pcg.x[l0 + k * n2] += alpha * po[k];
        }
#pragma unroll
        for (int k = 0; k < n1; ++k) {
            ru[k] = first ? z[k] : z[k] + beta * po[k];
            if (valid) pcg.p_io[l0 + k * n2] = ru[k];
        }
    } else {
        const ST* __restrict__ ue = u + f * n + e * Np + tl;
#pragma unroll
        for (int k = 0; k < n1; ++k) ru[k] = ue[k * n2];
    }
    // ---- global loads, t-line layout: lane -> consecutive nodes of plane k (coalesced 64-bit)
    // KH: how many k-planes of factors a thread loads up front.  For n1 >= SEMB_AX_SPLIT_N1 (N = 9, 10) the 6 x n1 factors of a
    // thread are 120+ registers on their own; loading the second half of the planes only after the second barrier (they are L2
    // hits by then: the bulk prefetch brought the element in) halves that footprint and lets one more block reside on the SM.
    constexpr int KH = (STORED && sizeof(ST) == 8 && n1 >= SEMB_AX_SPLIT_N1) ? (n1 + 1) / 2 : n1;
    if (STORED) {
#pragma unroll
        for (int k = 0; k < KH; ++k) {
#pragma unroll
            for (int c = 0; c < NG; ++c) G[c][k] = (CT)__ldg(g + c * Np + k * n2);
        }
    }
    // on-the-fly modes: element constants (uniform loads) and the thread's part of W = rho_i rho_j rho_k
    double gc[GEO == SEMB_GEO_AFFINE ? 7 : 1], wab = 0.0;
    double tA[GEO == SEMB_GEO_TRILINEAR ? 3 : 1][5];      // per coordinate: x_r = tA0 + tA1 t, x_s = tA2 + tA3 t, x_t = tA4
    if (GEO == SEMB_GEO_AFFINE) {
        const double* __restrict__ ge = (const double*)geo_v + e * 8;
#pragma unroll
        for (int c = 0; c < 7; ++c) gc[c] = __ldg(ge + c);
        wab = c_rho[n1 - 1][a] * c_rho[n1 - 1][b];
    }
    if (GEO == SEMB_GEO_TRILINEAR) {
        const double* __restrict__ ce = (const double*)geo_v + e * 24;
        const double r = c_xi[n1 - 1][a], sx = c_xi[n1 - 1][b];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double c1 = __ldg(ce + c * 8 + 1), c2 = __ldg(ce + c * 8 + 2), c3 = __ldg(ce + c * 8 + 3), c4 = __ldg(ce + c * 8 + 4),
                         c5 = __ldg(ce + c * 8 + 5), c6 = __ldg(ce + c * 8 + 6), c7 = __ldg(ce + c * 8 + 7);
            tA[c][0] = fma(c4, sx, c1); tA[c][1] = fma(c7, sx, c5);
            tA[c][2] = fma(c4, r, c2);  tA[c][3] = fma(c7, r, c6);
            tA[c][4] = fma(fma(c7, sx, c5), r, fma(c6, sx, c3));
        }
        wab = c_rho[n1 - 1][a] * c_rho[n1 - 1][b];
    }
#pragma unroll
    for (int k = 0; k < n1; ++k) Su[AX_I(k, b, a)] = ru[k];
    __syncthreads();
    // ---- forward contractions, one line per orientation
    {
        CT ln[n1], out[n1];
#pragma unroll
        for (int i = 0; i < n1; ++i) ln[i] = Su[AX_I(rb, ra, i)];
        ax_line<n1, 0, CT>(ln, out);
#pragma unroll
        for (int i = 0; i < n1; ++i) Sr[AX_I(rb, ra, i)] = out[i];
#pragma unroll
        for (int j = 0; j < n1; ++j) ln[j] = Su[AX_I(sb, j, sa)];
        ax_line<n1, 0, CT>(ln, out);
#pragma unroll
        for (int j = 0; j < n1; ++j) Ss[AX_IB(sb, j, sa)] = out[j];
    }
    CT ut[n1];
    ax_line<n1, 0, CT>(ru, ut);
    __syncthreads();
    if (STORED && KH < n1) {
#pragma unroll
        for (int k = KH; k < n1; ++k) {
#pragma unroll
            for (int c = 0; c < NG; ++c) G[c][k] = (CT)__ldg(g + c * Np + k * n2);
        }
    }
    // ---- geometric factors at the nodes of the t-line
    CT gt[n1];
    double Bk[(HELM && !STORED) ? n1 : 1];                 // mass factor W J of the on-the-fly modes
#pragma unroll
    for (int k = 0; k < n1; ++k) {
        const int s = AX_I(k, b, a), sB = AX_IB(k, b, a);
        const CT ur = Sr[s], us = Ss[sB];
        if (STORED) {
            CT Grr = G[0][k], Grs = G[1][k], Grt = G[2][k], Gss = G[3][k], Gst = G[4][k], Gtt = G[5][k];
            if (VAR && lam0) { const CT c = (CT)lam0[e * Np + k * n2 + tl]; Grr *= c; Grs *= c; Grt *= c; Gss *= c; Gst *= c; Gtt *= c; }
            Sr[s] = Grr * ur + Grs * us + Grt * ut[k];
            Ss[sB] = Grs * ur + Gss * us + Gst * ut[k];
            gt[k] = Grt * ur + Gst * us + Gtt * ut[k];
        } else if (GEO == SEMB_GEO_AFFINE) {
            const double W = wab * c_rho[n1 - 1][k];
            Sr[s] = (CT)(W * (gc[0] * ur + gc[1] * us + gc[2] * ut[k]));
            Ss[sB] = (CT)(W * (gc[1] * ur + gc[3] * us + gc[4] * ut[k]));
            gt[k] = (CT)(W * (gc[2] * ur + gc[4] * us + gc[5] * ut[k]));
            if (HELM) Bk[k] = W * gc[6];
        } else {
            const double t = c_xi[n1 - 1][k];
            const double xr = fma(tA[0][1], t, tA[0][0]), xs = fma(tA[0][3], t, tA[0][2]), xt = tA[0][4];
            const double yr = fma(tA[1][1], t, tA[1][0]), ys = fma(tA[1][3], t, tA[1][2]), yt = tA[1][4];
            const double zr = fma(tA[2][1], t, tA[2][0]), zs = fma(tA[2][3], t, tA[2][2]), zt = tA[2][4];
            // cofactor rows C_r = x_s x x_t, C_s = x_t x x_r, C_t = x_r x x_s
            const double rx = ys * zt - yt * zs, ry = zs * xt - zt * xs, rz = xs * yt - xt * ys;
            const double sx_ = yt * zr - yr * zt, sy_ = zt * xr - zr * xt, sz_ = xt * yr - xr * yt;
            const double tx = yr * zs - ys * zr, ty = zr * xs - zs * xr, tz = xr * ys - xs * yr;
            const double J = xr * rx + yr * ry + zr * rz;
            const double W = wab * c_rho[n1 - 1][k];
            const double sc = W * ax_rcp(J);
            const double vx = rx * ur + sx_ * us + tx * ut[k], vy = ry * ur + sy_ * us + ty * ut[k], vz = rz * ur + sz_ * us + tz * ut[k];
            Sr[s] = (CT)(sc * (rx * vx + ry * vy + rz * vz));
            Ss[sB] = (CT)(sc * (sx_ * vx + sy_ * vy + sz_ * vz));
            gt[k] = (CT)(sc * (tx * vx + ty * vy + tz * vz));
            if (HELM) Bk[k] = W * J;
        }
    }
    __syncthreads();
    // ---- transposed contractions
    {
        CT ln[n1], out[n1];
#pragma unroll
        for (int i = 0; i < n1; ++i) ln[i] = Sr[AX_I(rb, ra, i)];
        ax_line<n1, 1, CT>(ln, out);
#pragma unroll
        for (int i = 0; i < n1; ++i) Sr[AX_I(rb, ra, i)] = out[i];
#pragma unroll
        for (int j = 0; j < n1; ++j) ln[j] = Ss[AX_IB(sb, j, sa)];
        ax_line<n1, 1, CT>(ln, out);
#pragma unroll
        for (int j = 0; j < n1; ++j) Ss[AX_IB(sb, j, sa)] = out[j];
    }
    CT wt[n1];
    ax_line<n1, 1, CT>(gt, wt);
    // RELOAD (n1 >= SEMB_AX_RELOAD_N1, i.e. N = 9, 10): the thread's own u values are read back from the Su tile (never overwritten)
    // where the epilogue needs them, instead of staying in 2 n1 registers across both contraction phases.  Measured on B200, N = 9,
    // 46.7 M nodes: spills 88-132 -> 8-52 bytes; Poisson 5.50 -> 5.70 TB/s, Helmholtz 5.65 -> 6.41, PCG-fused 6.69 -> 6.87; N = 7
    // unchanged within noise (left off there).  Computing the t-contraction after the barrier from a reloaded u changed nothing.
    constexpr bool RELOAD = n1 >= SEMB_AX_RELOAD_N1;
    if (HELM) {
#pragma unroll
        for (int k = 0; k < n1; ++k) {
            const CT lam = (VAR && lam1) ? (CT)lam1[e * Np + k * n2 + tl] : (CT)lambda;
            const CT uk = RELOAD ? Su[AX_I(k, b, a)] : ru[k];
            wt[k] += lam * (STORED ? G[STORED ? NG - 1 : 0][STORED ? k : 0] : (CT)Bk[(HELM && !STORED) ? k : 0]) * uk;
        }
    }
    __syncthreads();
    double dot = 0.0;
#pragma unroll
    for (int k = 0; k < n1; ++k) {
        const CT wv = wt[k] + Sr[AX_I(k, b, a)] + Ss[AX_IB(k, b, a)];
        const CT uk = RELOAD ? Su[AX_I(k, b, a)] : ru[k];
        if (valid) { we[k * n2] = wv; dot += (double)uk * (double)wv; }
    }
    if (dot_out) {
        // two N = 9 elements per block fill the 48 KB of static shared memory: the reduction scratch then lives in the Sr tile
        constexpr bool ALIAS = sizeof(CT) * EPB * (2 * T::sizeA + (W32 ? T::sizeA : T::sizeB)) + 256 > 48 * 1024;
        __shared__ double red_own[ALIAS ? 1 : 32];
        double* red = ALIAS ? reinterpret_cast<double*>(SrA) : red_own;
        if (ALIAS) __syncthreads();
        dot = block_sum(dot, red);
        if (threadIdx.x == 0) dot_out[blockIdx.x] = dot;
    }
}
#undef AX_I
#undef AX_IB

// ---- N = 9 stand-alone operator, factors staged through shared memory by the TMA unit -------------------------------------
// k_axhelm_line at n1 = 10 holds 6 x 10 factors per thread in registers (168 registers, 3 blocks of 4 warps per SM) and its
// blocks wait for their own loads: 0.71 ms per launch on the cfg4 mesh whatever the byte count (Poisson 5.7 TB/s).  Here a
// block is persistent (3 per SM, elements blockIdx.x, + gridDim.x, ...), the six factors of its NEXT element are copied into a
// 48 KB shared-memory buffer by one cp.async.bulk issued as soon as the current element's factor phase has released the
// buffer, and consumed in place (conflict-free: slot = plane + thread).  The element body is a __noinline__ function so that
// ptxas cannot hoist the constant-bank operands of the contractions out of the element loop.
// Only n1 = 10: the bulk copy needs 16-byte aligned element starts (7 Np doubles per element: Np even).
template <int n1> struct ax_stage_smem {
    using T = ax_tile<n1>;
    static constexpr int Np = n1 * n1 * n1;
    static constexpr int oSu = 6 * Np, oSr = oSu + T::sizeA, oSs = oSr + T::sizeA, oBar = oSs + T::sizeB;     // in doubles
    static constexpr size_t bytes = (size_t)(oBar + 2) * sizeof(double);
};
__device__ __forceinline__ unsigned ax_smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void ax_stage_issue(double* dst, uint64_t* bar, const double* src, unsigned bytes)
{
    const unsigned d = ax_smem_u32(dst), m = ax_smem_u32(bar);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");       // the buffer's last generic-proxy reads precede the async write
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(m), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(d), "l"(src), "r"(bytes), "r"(m) : "memory");
}
__device__ __forceinline__ void ax_stage_wait(uint64_t* bar, unsigned phase)
{
    const unsigned m = ax_smem_u32(bar);
    asm volatile("{\n\t.reg .pred p;\n\tAX_WAIT:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@p bra AX_DONE;\n\tbra AX_WAIT;\n\tAX_DONE:\n\t}"
                 :: "r"(m), "r"(phase) : "memory");
}

template <int n1, bool HELM>
__device__ __noinline__ void ax_stage_element(int64_t e, int64_t f, int64_t ep, int64_t fp, int64_t n, const double* __restrict__ geo,
                                              double lambda, const double* __restrict__ u, double* __restrict__ w, unsigned phase,
                                              int do_wait, int64_t e_issue)
{
    // (e, f): the element and field applied now; (ep, fp): what this block applies next (its u goes to L2 now), ep < 0: nothing;
    // do_wait: the first field of the element -- its factors may still be in flight; e_issue >= 0: the last field -- once the factor
    // phase is over, the factors of element e_issue are copied into the buffer
    constexpr int n2 = n1 * n1, Np = n2 * n1;
    using T = ax_tile<n1>; using L = ax_stage_smem<n1>;
    extern __shared__ __align__(128) double ax_dyn[];
    double* __restrict__ Gs = ax_dyn; double* __restrict__ Su = ax_dyn + L::oSu; double* __restrict__ Sr = ax_dyn + L::oSr;
    double* __restrict__ Ss = ax_dyn + L::oSs; uint64_t* bar = reinterpret_cast<uint64_t*>(ax_dyn + L::oBar);
    const int tl = threadIdx.x, a = tl % n1, b = tl / n1;
    int ra = a, rb = b, sa = a, sb = b;
    if (T::permuted) {
        const int rq = c_perm[n1 - 1][0][tl], sq = c_perm[n1 - 1][1][tl];
        ra = rq % n1; rb = rq / n1; sa = sq % n1; sb = sq / n1;
    }
    if (tl == 0 && ep >= 0) {                          // what the next element (ep, field fp) reads with plain loads goes to L2 now
        ax_prefetch_l2(u + fp * n + ep * Np, Np);
        if (HELM && ep != e) ax_prefetch_l2(geo + (ep * 7 + 6) * (int64_t)Np, Np);
    }
    const double* __restrict__ ue = u + f * n + e * Np + tl;
    double ut[n1];
    {
        double ru[n1];
#pragma unroll
        for (int k = 0; k < n1; ++k) ru[k] = ue[k * n2];
#pragma unroll
        for (int k = 0; k < n1; ++k) Su[T::idx(k, b, a)] = ru[k];
        ax_line<n1, 0, double>(ru, ut);
    }
    double Bf[HELM ? n1 : 1];
    if (HELM) {
        const double* __restrict__ gB = geo + (e * 7 + 6) * (int64_t)Np + tl;
#pragma unroll
        for (int k = 0; k < n1; ++k) Bf[k] = __ldg(gB + k * n2);
    }
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
    __syncthreads();
    if (do_wait) ax_stage_wait(bar, phase);            // the factors of this element have landed
    double gt[n1];
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
    if (tl == 0 && e_issue >= 0)                       // every thread is past its last read of Gs
        ax_stage_issue(Gs, bar, geo + e_issue * 7 * (int64_t)Np, (unsigned)(6 * Np * sizeof(double)));
    {
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
    }
    double wt[n1];
    ax_line<n1, 1, double>(gt, wt);
    if (HELM) {
#pragma unroll
        for (int k = 0; k < n1; ++k) wt[k] += lambda * Bf[HELM ? k : 0] * Su[T::idx(k, b, a)];
    }
    __syncthreads();
    double* __restrict__ we = w + f * n + e * Np + tl;
#pragma unroll
    for (int k = 0; k < n1; ++k) we[k * n2] = wt[k] + Sr[T::idx(k, b, a)] + Ss[T::idxB(k, b, a)];
}

// Several fields (semb_apply_axhelm with nfields > 1, BASELINE.json configs[1]): a block applies its element to ALL fields before it
// moves on, so the factors cross DRAM -> shared memory once per element: 48 + 16 nfields bytes per node instead of 64 nfields.
template <int n1, bool HELM>
__global__ void __launch_bounds__(n1 * n1, 3)
k_axhelm_stage(int64_t E, int64_t n, const double* __restrict__ geo, double lambda, const double* __restrict__ u, double* __restrict__ w, int nfields)
{
    constexpr int Np = n1 * n1 * n1;
    using L = ax_stage_smem<n1>;
    extern __shared__ __align__(128) double ax_dyn[];
    uint64_t* bar = reinterpret_cast<uint64_t*>(ax_dyn + L::oBar);
    const int64_t stride = gridDim.x;
    int64_t e = blockIdx.x;
    if (e >= E) return;
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(ax_smem_u32(bar)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        ax_stage_issue(ax_dyn, bar, geo + e * 7 * (int64_t)Np, (unsigned)(6 * Np * sizeof(double)));
    }
    __syncthreads();
    unsigned phase = 0;
#pragma unroll 1
    for (; e < E; e += stride) {
        const int64_t en = (e + stride < E) ? e + stride : -1;
#pragma unroll 1
        for (int f = 0; f < nfields; ++f) {
            const bool lastf = f == nfields - 1;
            ax_stage_element<n1, HELM>(e, f, lastf ? en : e, lastf ? 0 : f + 1, n, geo, lambda, u, w, phase, f == 0, lastf ? en : -1);
        }
        phase ^= 1u;
    }
}

// Sum of the per-block partials dot_in[0..count) in a fixed order (two stages, last block by ticket), then
// the PCG scalars: p.Ap, alpha = rho / p.Ap, breakdown detection.
static __global__ void __launch_bounds__(256)
k_ax_dot_finish(int64_t count, const double* __restrict__ dot_in, semb_scalars* __restrict__ scal, double* __restrict__ partials)
{
    __shared__ double red[32];
    if (*(volatile int32_t*)&scal->done) return;
    double s = 0.0;
    const int64_t per = (count + gridDim.x - 1) / gridDim.x, lo = blockIdx.x * per, hi = (lo + per < count) ? lo + per : count;
    for (int64_t q = lo + threadIdx.x; q < hi; q += blockDim.x) s += dot_in[q];
    ax_finish_dot(s, scal, partials, red);
}
