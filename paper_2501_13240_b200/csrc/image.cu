// In-situ IMAGE consumer behind semb_export_field (§5.3: the overview scene is
// "two slices on the walls, two vertical slices in the background and an isocontour", 4096 x 2048 pixels).  The paper renders
// with ASCENT / VTK-m on the mesh of hexahedral SUB-CELLS between neighbouring GLL nodes; there is no graphics API on this
// machine, so the two primitives are plain CUDA kernels on that sub-cell mesh (reading R24):
//   slice        object order: one block per element, dropped at once unless the image plane cuts it; a thread per cut
//                sub-cell inverts the cell's trilinear map at the pixel centres of its footprint (Newton) and claims the
//                pixels it contains with atomicMin on (cell id << 32 | RGBA): the smallest cell id wins, whatever the order.
//   iso-surface  marching tetrahedra (6 per sub-cell around the diagonal corner 0 - corner 7) on the linear interpolant,
//                triangles rasterised orthographically with a depth key, atomicMin on (depth << 32 | RGBA).
// Every floating-point operation that decides a byte is written with an explicit rounding (__dmul_rn, __dadd_rn, fma,
// __ddiv_rn) so that the images are reproducible bit for bit (reading R11's rule applied to images).
#include <math.h>

#include "semb_internal.h"

#define MUL(a, b) __dmul_rn((a), (b))
#define ADD(a, b) __dadd_rn((a), (b))
#define SUB(a, b) __dsub_rn((a), (b))
#define DIV(a, b) __ddiv_rn((a), (b))

struct img_cam { double o[3], u[3], v[3], w[3], du, dv, dlo, dhi; int W, H; };

__device__ __forceinline__ double img_dot(const double* a, double x, double y, double z) { return fma(a[2], z, fma(a[1], y, MUL(a[0], x))); }

__device__ __forceinline__ void img_project(const img_cam& c, double X, double Y, double Z, double& a, double& b, double& d)
{
    const double x = SUB(X, c.o[0]), y = SUB(Y, c.o[1]), z = SUB(Z, c.o[2]);
    a = DIV(img_dot(c.u, x, y, z), c.du);
    b = DIV(img_dot(c.v, x, y, z), c.dv);
    d = img_dot(c.w, x, y, z);
}

// piecewise-linear colour table, value -> RGBA8 (shade multiplies the colour channels)
__device__ __forceinline__ uint32_t img_color(const semb_colormap& cm, double val, double shade)
{
    double s = DIV(SUB(val, cm.lo), SUB(cm.hi, cm.lo));
    if (!(s > 0.0)) s = 0.0;
    if (s > 1.0) s = 1.0;
    s = MUL(s, (double)(cm.ncolors - 1));
    int m = (int)floor(s);
    if (m > cm.ncolors - 2) m = cm.ncolors - 2;
    const double frac = SUB(s, (double)m);
    uint32_t out = 0xff000000u;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double c0 = (double)cm.rgb[m][c], c1 = (double)cm.rgb[m + 1][c];
        const double ch = MUL(fma(SUB(c1, c0), frac, c0), shade);
        uint32_t q = (uint32_t)floor(ADD(ch, 0.5));
        if (q > 255u) q = 255u;
        out |= q << (8 * c);
    }
    return out;
}

__global__ void k_img_clear(int64_t np, unsigned long long* __restrict__ key, uint32_t bg)
{
    for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < np; p += (int64_t)gridDim.x * blockDim.x)
        key[p] = 0xffffffff00000000ull | (unsigned long long)bg;
}
__global__ void k_img_resolve(int64_t np, const unsigned long long* __restrict__ key, uint32_t* __restrict__ rgba)
{
    for (int64_t p = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; p < np; p += (int64_t)gridDim.x * blockDim.x)
        rgba[p] = (uint32_t)(key[p] & 0xffffffffull);
}
__global__ void k_img_colormap(int64_t n, const double* __restrict__ val, semb_colormap cm, uint32_t* __restrict__ rgba)
{
    for (int64_t l = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; l < n; l += (int64_t)gridDim.x * blockDim.x)
        rgba[l] = img_color(cm, val[l], 1.0);
}

// Newton inversion of the trilinear map of one cell at P: start at the centre, <= 12 steps, converged when the step's
// max norm is <= 1e-10 (quadratic convergence: the iterate is then exact to rounding); gives up when the iterate leaves [-4, 4]^3 or the Jacobian is singular.
__device__ bool img_invert(const double (&X)[3][8], const double (&P)[3], double (&rst)[3])
{
    double r = 0.0, s = 0.0, t = 0.0;
    for (int it = 0; it < 12; ++it) {
        const double R[2] = {MUL(0.5, SUB(1.0, r)), MUL(0.5, ADD(1.0, r))}, S[2] = {MUL(0.5, SUB(1.0, s)), MUL(0.5, ADD(1.0, s))},
                     T[2] = {MUL(0.5, SUB(1.0, t)), MUL(0.5, ADD(1.0, t))};
        const double dR[2] = {-0.5, 0.5};
        double F[3], J[3][3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            double f = 0.0, jr = 0.0, js = 0.0, jt = 0.0;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const int a = q & 1, b = (q >> 1) & 1, d = q >> 2;
                const double x = X[c][q];
                f = fma(MUL(MUL(R[a], S[b]), T[d]), x, f);
                jr = fma(MUL(MUL(dR[a], S[b]), T[d]), x, jr);
                js = fma(MUL(MUL(R[a], dR[b]), T[d]), x, js);
                jt = fma(MUL(MUL(R[a], S[b]), dR[d]), x, jt);
            }
            F[c] = SUB(f, P[c]); J[c][0] = jr; J[c][1] = js; J[c][2] = jt;
        }
        const double c00 = fma(J[1][1], J[2][2], -MUL(J[1][2], J[2][1])), c01 = fma(J[1][2], J[2][0], -MUL(J[1][0], J[2][2])),
                     c02 = fma(J[1][0], J[2][1], -MUL(J[1][1], J[2][0]));
        const double det = fma(J[0][2], c02, fma(J[0][1], c01, MUL(J[0][0], c00)));
        if (det == 0.0 || det != det) return false;
        const double c10 = fma(J[0][2], J[2][1], -MUL(J[0][1], J[2][2])), c11 = fma(J[0][0], J[2][2], -MUL(J[0][2], J[2][0])),
                     c12 = fma(J[0][1], J[2][0], -MUL(J[0][0], J[2][1]));
        const double c20 = fma(J[0][1], J[1][2], -MUL(J[0][2], J[1][1])), c21 = fma(J[0][2], J[1][0], -MUL(J[0][0], J[1][2])),
                     c22 = fma(J[0][0], J[1][1], -MUL(J[0][1], J[1][0]));
        const double dr = DIV(fma(c20, F[2], fma(c10, F[1], MUL(c00, F[0]))), det);
        const double ds = DIV(fma(c21, F[2], fma(c11, F[1], MUL(c01, F[0]))), det);
        const double dt = DIV(fma(c22, F[2], fma(c12, F[1], MUL(c02, F[0]))), det);
        r = SUB(r, dr); s = SUB(s, ds); t = SUB(t, dt);
        const double step = fmax(fabs(dr), fmax(fabs(ds), fabs(dt)));
        if (!(fabs(r) <= 4.0 && fabs(s) <= 4.0 && fabs(t) <= 4.0)) return false;
        if (step <= 1e-10) { rst[0] = r; rst[1] = s; rst[2] = t; return true; }
    }
    return false;
}

// ---- slice ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
k_img_slice(int N, int64_t n, const double* __restrict__ xyz, const double* __restrict__ field, int64_t fstride, img_cam cam,
            semb_colormap cm, unsigned long long* __restrict__ key)
{
    extern __shared__ double sh[];               // per node: image a, image b, plane distance d
    __shared__ double s_lo[4], s_hi[4];
    const int n1 = N + 1, Np = n1 * n1 * n1;
    const int64_t e = blockIdx.x, base = e * Np;
    double* sa = sh; double* sb = sh + Np; double* sd = sh + 2 * Np;
    double lo = INFINITY, hi = -INFINITY;
    for (int l = threadIdx.x; l < Np; l += blockDim.x) {
        double a, b, d;
        img_project(cam, xyz[base + l], xyz[n + base + l], xyz[2 * n + base + l], a, b, d);
        sa[l] = a; sb[l] = b; sd[l] = d;
        lo = fmin(lo, d); hi = fmax(hi, d);
    }
    for (int o = 16; o > 0; o >>= 1) { lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o)); hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o)); }
    if ((threadIdx.x & 31) == 0) { s_lo[threadIdx.x >> 5] = lo; s_hi[threadIdx.x >> 5] = hi; }
    __syncthreads();
    lo = fmin(fmin(s_lo[0], s_lo[1]), fmin(s_lo[2], s_lo[3])); hi = fmax(fmax(s_hi[0], s_hi[1]), fmax(s_hi[2], s_hi[3]));
    if (!(lo <= 0.0 && hi >= 0.0)) return;       // the plane misses every node of the element, hence every sub-cell
    const int nc = N * N * N;
    for (int cl = threadIdx.x; cl < nc; cl += blockDim.x) {
        const int i = cl % N, j = (cl / N) % N, k = cl / (N * N);
        int id[8];
        double amin = INFINITY, amax = -INFINITY, bmin = INFINITY, bmax = -INFINITY, dmin = INFINITY, dmax = -INFINITY;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            id[q] = (k + (q >> 2)) * n1 * n1 + (j + ((q >> 1) & 1)) * n1 + (i + (q & 1));
            amin = fmin(amin, sa[id[q]]); amax = fmax(amax, sa[id[q]]); bmin = fmin(bmin, sb[id[q]]); bmax = fmax(bmax, sb[id[q]]);
            dmin = fmin(dmin, sd[id[q]]); dmax = fmax(dmax, sd[id[q]]);
        }
        if (!(dmin <= 0.0 && dmax >= 0.0)) continue;
        long long px0 = (long long)ceil(SUB(amin, 0.5)), px1 = (long long)floor(SUB(amax, 0.5));
        long long py0 = (long long)ceil(SUB(bmin, 0.5)), py1 = (long long)floor(SUB(bmax, 0.5));
        if (px0 < 0) px0 = 0; if (py0 < 0) py0 = 0; if (px1 > cam.W - 1) px1 = cam.W - 1; if (py1 > cam.H - 1) py1 = cam.H - 1;
        if (px1 < px0 || py1 < py0) continue;
        double X[3][8], fv[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            X[0][q] = xyz[base + id[q]]; X[1][q] = xyz[n + base + id[q]]; X[2][q] = xyz[2 * n + base + id[q]];
            fv[q] = field[(base + id[q]) * fstride];
        }
        const unsigned long long cid = (unsigned long long)(e * (int64_t)nc + cl);
        for (long long py = py0; py <= py1; ++py) for (long long px = px0; px <= px1; ++px) {
            const double ca = MUL(ADD((double)px, 0.5), cam.du), cb = MUL(ADD((double)py, 0.5), cam.dv);
            double P[3], rst[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) P[c] = fma(cb, cam.v[c], fma(ca, cam.u[c], cam.o[c]));
            if (!img_invert(X, P, rst)) continue;
            if (!(fabs(rst[0]) <= 1.0 + 1e-9 && fabs(rst[1]) <= 1.0 + 1e-9 && fabs(rst[2]) <= 1.0 + 1e-9)) continue;
            const double R[2] = {MUL(0.5, SUB(1.0, rst[0])), MUL(0.5, ADD(1.0, rst[0]))}, S[2] = {MUL(0.5, SUB(1.0, rst[1])), MUL(0.5, ADD(1.0, rst[1]))},
                         T[2] = {MUL(0.5, SUB(1.0, rst[2])), MUL(0.5, ADD(1.0, rst[2]))};
            double val = MUL(MUL(MUL(R[0], S[0]), T[0]), fv[0]);
#pragma unroll
            for (int q = 1; q < 8; ++q) val = fma(MUL(MUL(R[q & 1], S[(q >> 1) & 1]), T[q >> 2]), fv[q], val);
            atomicMin(&key[py * cam.W + px], (cid << 32) | (unsigned long long)img_color(cm, val, 1.0));
        }
    }
}

// ---- iso-surface ---------------------------------------------------------------------------------------------
struct img_vert { double a, b, d, X[3], col; };

__device__ __forceinline__ void img_edge(const img_vert& p, const img_vert& q, double fp, double fq, double iso, img_vert& o)
{
    const double tt = DIV(SUB(iso, fp), SUB(fq, fp));
    o.a = fma(SUB(q.a, p.a), tt, p.a); o.b = fma(SUB(q.b, p.b), tt, p.b); o.d = fma(SUB(q.d, p.d), tt, p.d);
#pragma unroll
    for (int c = 0; c < 3; ++c) o.X[c] = fma(SUB(q.X[c], p.X[c]), tt, p.X[c]);
    o.col = fma(SUB(q.col, p.col), tt, p.col);
}

__device__ void img_raster(const img_cam& cam, const semb_colormap& cm, const double* light, const img_vert& A, const img_vert& B,
                           const img_vert& C, unsigned long long* __restrict__ key)
{
    const double area = fma(SUB(B.a, A.a), SUB(C.b, A.b), -MUL(SUB(B.b, A.b), SUB(C.a, A.a)));
    if (area == 0.0 || area != area) return;
    const double e1[3] = {SUB(B.X[0], A.X[0]), SUB(B.X[1], A.X[1]), SUB(B.X[2], A.X[2])}, e2[3] = {SUB(C.X[0], A.X[0]), SUB(C.X[1], A.X[1]), SUB(C.X[2], A.X[2])};
    double nrm[3];
    nrm[0] = fma(e1[1], e2[2], -MUL(e1[2], e2[1])); nrm[1] = fma(e1[2], e2[0], -MUL(e1[0], e2[2])); nrm[2] = fma(e1[0], e2[1], -MUL(e1[1], e2[0]));
    const double nn = sqrt(img_dot(nrm, nrm[0], nrm[1], nrm[2]));
    if (nn == 0.0) return;
    const double shade = fma(0.75, DIV(fabs(img_dot(nrm, light[0], light[1], light[2])), nn), 0.25);
    const double amin = fmin(A.a, fmin(B.a, C.a)), amax = fmax(A.a, fmax(B.a, C.a)), bmin = fmin(A.b, fmin(B.b, C.b)), bmax = fmax(A.b, fmax(B.b, C.b));
    long long px0 = (long long)ceil(SUB(amin, 0.5)), px1 = (long long)floor(SUB(amax, 0.5)), py0 = (long long)ceil(SUB(bmin, 0.5)), py1 = (long long)floor(SUB(bmax, 0.5));
    if (px0 < 0) px0 = 0; if (py0 < 0) py0 = 0; if (px1 > cam.W - 1) px1 = cam.W - 1; if (py1 > cam.H - 1) py1 = cam.H - 1;
    const double sg = (area > 0.0) ? 1.0 : -1.0, slack = MUL(-1e-12, fabs(area));
    for (long long py = py0; py <= py1; ++py) for (long long px = px0; px <= px1; ++px) {
        const double a = ADD((double)px, 0.5), b = ADD((double)py, 0.5);
        const double w0 = fma(SUB(B.a, a), SUB(C.b, b), -MUL(SUB(B.b, b), SUB(C.a, a)));
        const double w1 = fma(SUB(C.a, a), SUB(A.b, b), -MUL(SUB(C.b, b), SUB(A.a, a)));
        const double w2 = fma(SUB(A.a, a), SUB(B.b, b), -MUL(SUB(A.b, b), SUB(B.a, a)));
        if (!(MUL(sg, w0) >= slack && MUL(sg, w1) >= slack && MUL(sg, w2) >= slack)) continue;
        const double l0 = DIV(w0, area), l1 = DIV(w1, area), l2 = DIV(w2, area);
        const double depth = fma(l2, C.d, fma(l1, B.d, MUL(l0, A.d)));
        const double col = fma(l2, C.col, fma(l1, B.col, MUL(l0, A.col)));
        double qd = DIV(SUB(depth, cam.dlo), SUB(cam.dhi, cam.dlo));
        if (!(qd > 0.0)) qd = 0.0;
        if (qd > 1.0) qd = 1.0;
        const unsigned long long dq = (unsigned long long)floor(MUL(qd, 4294967295.0));
        atomicMin(&key[py * cam.W + px], (dq << 32) | (unsigned long long)img_color(cm, col, shade));
    }
}

__constant__ int c_tet[6][4] = { {0, 1, 3, 7}, {0, 3, 2, 7}, {0, 2, 6, 7}, {0, 6, 4, 7}, {0, 4, 5, 7}, {0, 5, 1, 7} };

__global__ void __launch_bounds__(128)
k_img_iso(int N, int64_t n, const double* __restrict__ xyz, const double* __restrict__ field, int64_t fstride, double iso,
          const double* __restrict__ cfield, int64_t cstride, img_cam cam, semb_colormap cm, double lx, double ly, double lz,
          unsigned long long* __restrict__ key)
{
    extern __shared__ double sh[];               // the element's field values
    __shared__ double s_lo[4], s_hi[4];
    const int n1 = N + 1, Np = n1 * n1 * n1;
    const int64_t e = blockIdx.x, base = e * Np;
    double lo = INFINITY, hi = -INFINITY;
    for (int l = threadIdx.x; l < Np; l += blockDim.x) { const double f = field[(base + l) * fstride]; sh[l] = f; lo = fmin(lo, f); hi = fmax(hi, f); }
    for (int o = 16; o > 0; o >>= 1) { lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o)); hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o)); }
    if ((threadIdx.x & 31) == 0) { s_lo[threadIdx.x >> 5] = lo; s_hi[threadIdx.x >> 5] = hi; }
    __syncthreads();
    lo = fmin(fmin(s_lo[0], s_lo[1]), fmin(s_lo[2], s_lo[3])); hi = fmax(fmax(s_hi[0], s_hi[1]), fmax(s_hi[2], s_hi[3]));
    if (!(lo < iso && hi >= iso)) return;
    const double light[3] = {lx, ly, lz};
    const int nc = N * N * N;
    for (int cl = threadIdx.x; cl < nc; cl += blockDim.x) {
        const int i = cl % N, j = (cl / N) % N, k = cl / (N * N);
        int id[8]; double fv[8], fl = INFINITY, fh = -INFINITY;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            id[q] = (k + (q >> 2)) * n1 * n1 + (j + ((q >> 1) & 1)) * n1 + (i + (q & 1));
            fv[q] = sh[id[q]]; fl = fmin(fl, fv[q]); fh = fmax(fh, fv[q]);
        }
        if (!(fl < iso && fh >= iso)) continue;
        img_vert V[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            V[q].X[0] = xyz[base + id[q]]; V[q].X[1] = xyz[n + base + id[q]]; V[q].X[2] = xyz[2 * n + base + id[q]];
            img_project(cam, V[q].X[0], V[q].X[1], V[q].X[2], V[q].a, V[q].b, V[q].d);
            V[q].col = cfield ? cfield[(base + id[q]) * cstride] : iso;
        }
        for (int tt = 0; tt < 6; ++tt) {
            int up[4], dn[4], nu = 0, nd = 0;
            for (int c = 0; c < 4; ++c) { const int q = c_tet[tt][c]; if (fv[q] >= iso) up[nu++] = q; else dn[nd++] = q; }
            if (nu == 0 || nd == 0) continue;
            img_vert P[4];
            if (nu == 1 || nd == 1) {
                const int apex = (nu == 1) ? up[0] : dn[0];
                const int* oth = (nu == 1) ? dn : up;
                for (int c = 0; c < 3; ++c) img_edge(V[apex], V[oth[c]], fv[apex], fv[oth[c]], iso, P[c]);
                img_raster(cam, cm, light, P[0], P[1], P[2], key);
            } else {
                img_edge(V[up[0]], V[dn[0]], fv[up[0]], fv[dn[0]], iso, P[0]);
                img_edge(V[up[0]], V[dn[1]], fv[up[0]], fv[dn[1]], iso, P[1]);
                img_edge(V[up[1]], V[dn[1]], fv[up[1]], fv[dn[1]], iso, P[2]);
                img_edge(V[up[1]], V[dn[0]], fv[up[1]], fv[dn[0]], iso, P[3]);
                img_raster(cam, cm, light, P[0], P[1], P[2], key);
                img_raster(cam, cm, light, P[0], P[2], P[3], key);
            }
        }
    }
}

// ---- entry points --------------------------------------------------------------------------------------------
static int img_check(semb_mesh* h, const semb_field_desc* f, const semb_image_view* vw, const semb_colormap* cm, const void* key, img_cam* cam)
{
    if (!f || !vw || !cm || !key) return semb_fail(h, SEMB_EINVAL, "image: bad argument");
    if (!f->ptr || f->memspace != SEMB_MEM_DEVICE || f->dtype != SEMB_F64 || f->stride < 1 || f->count != h->n)
        return semb_fail(h, SEMB_EINVAL, "image: the field must be a device fp64 array over the mesh's local nodes (PAPER.md:L171-177)");
    if (vw->width < 1 || vw->height < 1 || (int64_t)vw->width * vw->height > ((int64_t)1 << 28) || !(vw->du > 0.0) || !(vw->dv > 0.0))
        return semb_fail(h, SEMB_EINVAL, "image: bad view");
    if (cm->ncolors < 2 || cm->ncolors > 16 || !(cm->hi > cm->lo)) return semb_fail(h, SEMB_EINVAL, "image: bad colour map");
    if (!h->xyz) return semb_fail(h, SEMB_EINVAL, "image: the handle holds no coordinates");
    if (h->E * (int64_t)h->N * h->N * h->N >= ((int64_t)1 << 32) - 1) return semb_fail(h, SEMB_EINVAL, "image: too many sub-cells for a 32-bit cell id");
    for (int c = 0; c < 3; ++c) { cam->o[c] = vw->origin[c]; cam->u[c] = vw->u[c]; cam->v[c] = vw->v[c]; }
    // w = u x v with the same roundings as everywhere: fma(a, b, -(c d))
    cam->w[0] = fma(vw->u[1], vw->v[2], -(vw->u[2] * vw->v[1]));
    cam->w[1] = fma(vw->u[2], vw->v[0], -(vw->u[0] * vw->v[2]));
    cam->w[2] = fma(vw->u[0], vw->v[1], -(vw->u[1] * vw->v[0]));
    cam->du = vw->du; cam->dv = vw->dv; cam->dlo = vw->depth_lo; cam->dhi = vw->depth_hi; cam->W = vw->width; cam->H = vw->height;
    return SEMB_OK;
}

static unsigned img_grid(int64_t n) { int64_t b = (n + 1023) / 1024, cap = (int64_t)semb_sm_count() * 8; return (unsigned)(b < 1 ? 1 : (b > cap ? cap : b)); }

extern "C" int semb_colormap_apply(const semb_colormap* cm, const double* val_dev, int64_t n, uint32_t* rgba_dev, void* stream)
{
    if (!cm || !val_dev || !rgba_dev || n < 1 || cm->ncolors < 2 || cm->ncolors > 16 || !(cm->hi > cm->lo)) return SEMB_EINVAL;
    k_img_colormap<<<img_grid(n), 256, 0, (cudaStream_t)stream>>>(n, val_dev, *cm, rgba_dev);
    return cudaGetLastError() == cudaSuccess ? SEMB_OK : SEMB_ECUDA;
}

extern "C" int semb_image_slice(semb_handle h, const semb_field_desc* f, const semb_image_view* vw, const semb_colormap* cm,
                                uint64_t* key_dev, uint32_t* rgba_dev, void* stream)
{
    if (!h) return SEMB_EINVAL;
    img_cam cam;
    int rc = img_check(h, f, vw, cm, key_dev, &cam); if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t np = (int64_t)cam.W * cam.H;
    k_img_clear<<<img_grid(np), 256, 0, s>>>(np, (unsigned long long*)key_dev, cm->background);
    k_img_slice<<<(unsigned)h->E, 128, sizeof(double) * 3 * (size_t)h->Np, s>>>(h->N, h->n, h->xyz, (const double*)f->ptr, f->stride, cam, *cm,
                                                                               (unsigned long long*)key_dev);
    if (rgba_dev) k_img_resolve<<<img_grid(np), 256, 0, s>>>(np, (const unsigned long long*)key_dev, rgba_dev);
    h->launches += 3;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}

extern "C" int semb_image_isosurface(semb_handle h, const semb_field_desc* f, double iso, const semb_field_desc* color_or_null,
                                     const semb_image_view* vw, const semb_colormap* cm, const double* light, uint64_t* key_dev,
                                     uint32_t* rgba_dev, void* stream)
{
    if (!h) return SEMB_EINVAL;
    img_cam cam;
    int rc = img_check(h, f, vw, cm, key_dev, &cam); if (rc) return rc;
    if (!light || !(vw->depth_hi > vw->depth_lo)) return semb_fail(h, SEMB_EINVAL, "image_isosurface: light and a depth range are needed");
    const semb_field_desc* cf = color_or_null;
    if (cf && (!cf->ptr || cf->memspace != SEMB_MEM_DEVICE || cf->dtype != SEMB_F64 || cf->stride < 1 || cf->count != h->n))
        return semb_fail(h, SEMB_EINVAL, "image_isosurface: bad colour field");
    cudaStream_t s = (cudaStream_t)stream;
    const int64_t np = (int64_t)cam.W * cam.H;
    k_img_clear<<<img_grid(np), 256, 0, s>>>(np, (unsigned long long*)key_dev, cm->background);
    k_img_iso<<<(unsigned)h->E, 128, sizeof(double) * (size_t)h->Np, s>>>(h->N, h->n, h->xyz, (const double*)f->ptr, f->stride, iso,
                                                                         cf ? (const double*)cf->ptr : nullptr, cf ? cf->stride : 1, cam, *cm,
                                                                         light[0], light[1], light[2], (unsigned long long*)key_dev);
    if (rgba_dev) k_img_resolve<<<img_grid(np), 256, 0, s>>>(np, (const unsigned long long*)key_dev, rgba_dev);
    h->launches += 3;
    SEMB_CUDA(h, cudaGetLastError());
    return SEMB_OK;
}
