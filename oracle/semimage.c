/*
 * semimage.c -- CPU oracle of the in-situ IMAGE consumer (§5.3: "The overview scene
 * ... is composed of several partial images, two slices on the walls, two vertical slices in the background and an
 * isocontour.  4096 pixels were used ... for the longest side", 2048 for the shorter one).
 *
 * TEST INFRASTRUCTURE ONLY: used by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg.  Plain C, fp64, loops in
 * Pins (tests/test_oracle_image.py): colour ramps in closed form; the claiming sub-cell against a numpy search of the node planes and
 * the value of a linear field; the disc footprint of the cylinder; iso-plane exact, iso-sphere to second order.  Parity unpinned: none.
 * the order the definitions below state; shares no code with the CUDA path (csrc/image.cu).
 *
 * The paper renders with ASCENT / VTK-m, which see the spectral-element field as an unstructured mesh of hexahedral
 * SUB-CELLS (the N^3 cells between neighbouring GLL nodes of every element, "connectivity") with trilinear
 * interpolation inside a cell.  No graphics API exists on this machine, so the two image primitives are restated as
 * arithmetic on that sub-cell mesh (reading R24).  Sub-cell id c = e*N^3 + (k*N + j)*N + i, corners = the 8 nodes
 * (i+a, j+b, k+c); corner q = a + 2 b + 4 c.
 *
 * View: pixel (px, py), 0 <= px < W, 0 <= py < H, has the centre  P = origin + ((px + 0.5) du) u + ((py + 0.5) dv) v ;
 * w = u x v is the viewing direction; the signed distance of a point X to the image plane is d = (X - origin) . w.
 *
 * All products and sums below are written out with explicit fma() where a fused operation is meant and are otherwise
 * rounded one by one (compile with -ffp-contract=off); the CUDA path fixes the same forms, so bytes compare EXACTLY.
 *
 * (1) slice: the image plane cuts the mesh.  For every sub-cell in ascending id whose corner distances satisfy
 *     min d <= 0 <= max d, and every pixel of the bounding box of its corners' image coordinates: invert the cell's
 *     trilinear map at P by Newton (start 0, at most 12 steps, stop when the step's max norm is <= 1e-10: Newton is quadratic, the next iterate is exact to rounding; 1e-13 is below the rounding noise of the residual on the smallest cells of a 64^3 mesh); the pixel is
 *     inside when every reference coordinate has |.| <= 1 + 1e-9; the first (= smallest id) cell claims the pixel; its
 *     value is the trilinear interpolant of the field; colour by the map (3).
 * (2) iso-surface: every sub-cell is split into the 6 tetrahedra around its diagonal corner 0 - corner 7; each tetrahedron
 *     yields the triangles of the level set {f = iso} of the LINEAR interpolant (0, 1 or 2 triangles); triangles are
 *     projected orthographically along w, rasterised at pixel centres (inside when all three edge functions have the sign
 *     of the area, are zero, or miss that by at most 1e-12 |area|), depth = distance d interpolated barycentrically, flat Lambert shading |n . light|
 *     (0.25 ambient + 0.75 diffuse) of the colour that the map gives to a second field (or to the iso value).  Per pixel
 *     the smallest key (depth quantised to 2^-32 of the depth range, then RGBA) wins, which is independent of the order in
 *     which triangles are drawn.
 * (3) colour map: s = clamp((v - lo) / (hi - lo), 0, 1) * (ncolors - 1); segment m = min(floor(s), ncolors - 2);
 *     channel = floor((c_m + (c_{m+1} - c_m) (s - m)) + 0.5), alpha 255; packed r | g << 8 | b << 16 | a << 24.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t width, height;
    double origin[3], u[3], v[3];
    double du, dv;
} img_view;

typedef struct {
    double lo, hi;
    int32_t ncolors;
    uint8_t rgb[16][3];
    uint32_t background;
} img_cmap;

static uint32_t orc_color(const img_cmap* cm, double val, double shade)
{
    double s = (val - cm->lo) / (cm->hi - cm->lo);
    if (!(s > 0.0)) s = 0.0;
    if (s > 1.0) s = 1.0;
    s = s * (double)(cm->ncolors - 1);
    int m = (int)floor(s);
    if (m > cm->ncolors - 2) m = cm->ncolors - 2;
    const double frac = s - (double)m;
    uint32_t out = 0xff000000u;
    for (int c = 0; c < 3; ++c) {
        const double c0 = (double)cm->rgb[m][c], c1 = (double)cm->rgb[m + 1][c];
        double ch = fma(c1 - c0, frac, c0) * shade;
        uint32_t q = (uint32_t)floor(ch + 0.5);
        if (q > 255u) q = 255u;
        out |= q << (8 * c);
    }
    return out;
}

void orc_colormap(const img_cmap* cm, int64_t n, const double* val, uint32_t* rgba)
{
    for (int64_t l = 0; l < n; ++l) rgba[l] = orc_color(cm, val[l], 1.0);
}

static double dot3(const double* a, double bx, double by, double bz)      /* fma(a2, bz, fma(a1, by, a0*bx)) */
{
    return fma(a[2], bz, fma(a[1], by, a[0] * bx));
}

static void cross3(const double* a, const double* b, double* c)
{
    c[0] = fma(a[1], b[2], -(a[2] * b[1]));
    c[1] = fma(a[2], b[0], -(a[0] * b[2]));
    c[2] = fma(a[0], b[1], -(a[1] * b[0]));
}

/* corners of sub-cell (e; i, j, k): local node ids */
static void cell_nodes(int N, int64_t e, int i, int j, int k, int64_t* id)
{
    const int n1 = N + 1; const int64_t Np = (int64_t)n1 * n1 * n1;
    for (int q = 0; q < 8; ++q) {
        const int a = q & 1, b = (q >> 1) & 1, c = q >> 2;
        id[q] = e * Np + (int64_t)(k + c) * n1 * n1 + (j + b) * n1 + (i + a);
    }
}

/* trilinear weights of corner q at (r, s, t) in [-1,1]^3: (1 +- r)(1 +- s)(1 +- t) / 8 */
static void tri_weights(double r, double s, double t, double* wq)
{
    const double rm = 0.5 * (1.0 - r), rp = 0.5 * (1.0 + r), sm = 0.5 * (1.0 - s), sp = 0.5 * (1.0 + s),
                 tm = 0.5 * (1.0 - t), tp = 0.5 * (1.0 + t);
    const double R[2] = {rm, rp}, S[2] = {sm, sp}, T[2] = {tm, tp};
    for (int q = 0; q < 8; ++q) wq[q] = (R[q & 1] * S[(q >> 1) & 1]) * T[q >> 2];
}

/* value of sum_q w_q c_q accumulated in ascending q with fma */
static double tri_eval(const double* wq, const double* c)
{
    double s = wq[0] * c[0];
    for (int q = 1; q < 8; ++q) s = fma(wq[q], c[q], s);
    return s;
}

/* Newton inversion of the trilinear map X(r,s,t) = P.  X[3][8] corner coordinates.  Returns 1 when converged. */
static int tri_invert(const double X[3][8], const double* P, double* rst)
{
    double r = 0.0, s = 0.0, t = 0.0;
    for (int it = 0; it < 12; ++it) {
        const double R[2] = {0.5 * (1.0 - r), 0.5 * (1.0 + r)}, S[2] = {0.5 * (1.0 - s), 0.5 * (1.0 + s)}, T[2] = {0.5 * (1.0 - t), 0.5 * (1.0 + t)};
        const double dR[2] = {-0.5, 0.5};
        double F[3], J[3][3];
        for (int c = 0; c < 3; ++c) {
            double f = 0.0, jr = 0.0, js = 0.0, jt = 0.0;
            for (int q = 0; q < 8; ++q) {
                const int a = q & 1, b = (q >> 1) & 1, d = q >> 2;
                const double x = X[c][q];
                f = fma((R[a] * S[b]) * T[d], x, f);
                jr = fma((dR[a] * S[b]) * T[d], x, jr);
                js = fma((R[a] * dR[b]) * T[d], x, js);
                jt = fma((R[a] * S[b]) * dR[d], x, jt);
            }
            F[c] = f - P[c]; J[c][0] = jr; J[c][1] = js; J[c][2] = jt;
        }
        /* solve J delta = F by Cramer's rule with the cofactors written out */
        const double c00 = fma(J[1][1], J[2][2], -(J[1][2] * J[2][1])), c01 = fma(J[1][2], J[2][0], -(J[1][0] * J[2][2])),
                     c02 = fma(J[1][0], J[2][1], -(J[1][1] * J[2][0]));
        const double det = fma(J[0][2], c02, fma(J[0][1], c01, J[0][0] * c00));
        if (det == 0.0 || det != det) return 0;
        const double c10 = fma(J[0][2], J[2][1], -(J[0][1] * J[2][2])), c11 = fma(J[0][0], J[2][2], -(J[0][2] * J[2][0])),
                     c12 = fma(J[0][1], J[2][0], -(J[0][0] * J[2][1]));
        const double c20 = fma(J[0][1], J[1][2], -(J[0][2] * J[1][1])), c21 = fma(J[0][2], J[1][0], -(J[0][0] * J[1][2])),
                     c22 = fma(J[0][0], J[1][1], -(J[0][1] * J[1][0]));
        const double dr = fma(c20, F[2], fma(c10, F[1], c00 * F[0])) / det;
        const double ds = fma(c21, F[2], fma(c11, F[1], c01 * F[0])) / det;
        const double dt = fma(c22, F[2], fma(c12, F[1], c02 * F[0])) / det;
        r -= dr; s -= ds; t -= dt;
        const double step = fmax(fabs(dr), fmax(fabs(ds), fabs(dt)));
        if (!(fabs(r) <= 4.0 && fabs(s) <= 4.0 && fabs(t) <= 4.0)) return 0;        /* diverging: not this cell */
        if (step <= 1e-10) { rst[0] = r; rst[1] = s; rst[2] = t; return 1; }
    }
    return 0;
}

/* image coordinates (in pixels, continuous) and plane distance of a point */
static void project(const img_view* vw, const double* w, double X, double Y, double Z, double* a, double* b, double* d)
{
    const double x = X - vw->origin[0], y = Y - vw->origin[1], z = Z - vw->origin[2];
    *a = dot3(vw->u, x, y, z) / vw->du;
    *b = dot3(vw->v, x, y, z) / vw->dv;
    *d = dot3(w, x, y, z);
}

/* (1) slice.  rgba [W*H]; cell_of [W*H] (may be NULL): the sub-cell id that claimed the pixel, -1 = background. */
void orc_image_slice(int64_t E, int N, const double* x, const double* y, const double* z, const double* field,
                     const img_view* vw, const img_cmap* cm, uint32_t* rgba, int64_t* cell_of)
{
    const int W = vw->width, H = vw->height;
    double w[3];
    cross3(vw->u, vw->v, w);
    for (int64_t p = 0; p < (int64_t)W * H; ++p) { rgba[p] = cm->background; if (cell_of) cell_of[p] = -1; }
    unsigned char* claimed = (unsigned char*)calloc((size_t)W * H, 1);
    for (int64_t e = 0; e < E; ++e)
        for (int k = 0; k < N; ++k) for (int j = 0; j < N; ++j) for (int i = 0; i < N; ++i) {
            int64_t id[8];
            cell_nodes(N, e, i, j, k, id);
            double X[3][8], fv[8], a[8], b[8], d[8];
            double amin = INFINITY, amax = -INFINITY, bmin = INFINITY, bmax = -INFINITY, dmin = INFINITY, dmax = -INFINITY;
            for (int q = 0; q < 8; ++q) {
                X[0][q] = x[id[q]]; X[1][q] = y[id[q]]; X[2][q] = z[id[q]]; fv[q] = field[id[q]];
                project(vw, w, X[0][q], X[1][q], X[2][q], &a[q], &b[q], &d[q]);
                amin = fmin(amin, a[q]); amax = fmax(amax, a[q]); bmin = fmin(bmin, b[q]); bmax = fmax(bmax, b[q]);
                dmin = fmin(dmin, d[q]); dmax = fmax(dmax, d[q]);
            }
            if (!(dmin <= 0.0 && dmax >= 0.0)) continue;
            /* pixels whose centre px + 0.5 lies in [amin, amax] */
            int64_t px0 = (int64_t)ceil(amin - 0.5), px1 = (int64_t)floor(amax - 0.5);
            int64_t py0 = (int64_t)ceil(bmin - 0.5), py1 = (int64_t)floor(bmax - 0.5);
            if (px0 < 0) px0 = 0; if (py0 < 0) py0 = 0; if (px1 > W - 1) px1 = W - 1; if (py1 > H - 1) py1 = H - 1;
            const int64_t cid = e * (int64_t)N * N * N + ((int64_t)k * N + j) * N + i;
            for (int64_t py = py0; py <= py1; ++py) for (int64_t px = px0; px <= px1; ++px) {
                const int64_t p = py * W + px;
                if (claimed[p]) continue;
                const double ca = ((double)px + 0.5) * vw->du, cb = ((double)py + 0.5) * vw->dv;
                double P[3], rst[3];
                for (int c = 0; c < 3; ++c) P[c] = fma(cb, vw->v[c], fma(ca, vw->u[c], vw->origin[c]));
                if (!tri_invert(X, P, rst)) continue;
                if (!(fabs(rst[0]) <= 1.0 + 1e-9 && fabs(rst[1]) <= 1.0 + 1e-9 && fabs(rst[2]) <= 1.0 + 1e-9)) continue;
                double wq[8];
                tri_weights(rst[0], rst[1], rst[2], wq);
                rgba[p] = orc_color(cm, tri_eval(wq, fv), 1.0);
                claimed[p] = 1;
                if (cell_of) cell_of[p] = cid;
            }
        }
    free(claimed);
}

/* the 6 tetrahedra of a hexahedron around the diagonal corner 0 - corner 7 (corner q = a + 2 b + 4 c) */
static const int TET[6][4] = { {0, 1, 3, 7}, {0, 3, 2, 7}, {0, 2, 6, 7}, {0, 6, 4, 7}, {0, 4, 5, 7}, {0, 5, 1, 7} };

typedef struct { double a, b, d, X[3], col; } img_vert;      /* image coordinates, depth, world position, colour value */

static void edge_point(const img_vert* p, const img_vert* q, double fp, double fq, double iso, img_vert* o)
{
    const double tt = (iso - fp) / (fq - fp);
    o->a = fma(q->a - p->a, tt, p->a); o->b = fma(q->b - p->b, tt, p->b); o->d = fma(q->d - p->d, tt, p->d);
    for (int c = 0; c < 3; ++c) o->X[c] = fma(q->X[c] - p->X[c], tt, p->X[c]);
    o->col = fma(q->col - p->col, tt, p->col);
}

static void raster_tri(const img_view* vw, const img_cmap* cm, const double* light, double dlo, double dhi,
                       const img_vert* A, const img_vert* B, const img_vert* C, uint64_t* key)
{
    const int W = vw->width, H = vw->height;
    const double area = fma(B->a - A->a, C->b - A->b, -((B->b - A->b) * (C->a - A->a)));
    if (area == 0.0 || area != area) return;
    /* flat normal from the world positions; shade = 0.25 + 0.75 |n . light| / |n| (light is a unit vector) */
    const double e1[3] = {B->X[0] - A->X[0], B->X[1] - A->X[1], B->X[2] - A->X[2]}, e2[3] = {C->X[0] - A->X[0], C->X[1] - A->X[1], C->X[2] - A->X[2]};
    double nrm[3];
    cross3(e1, e2, nrm);
    const double nn = sqrt(dot3(nrm, nrm[0], nrm[1], nrm[2]));
    if (nn == 0.0) return;
    const double shade = fma(0.75, fabs(dot3(nrm, light[0], light[1], light[2])) / nn, 0.25);
    const double amin = fmin(A->a, fmin(B->a, C->a)), amax = fmax(A->a, fmax(B->a, C->a));
    const double bmin = fmin(A->b, fmin(B->b, C->b)), bmax = fmax(A->b, fmax(B->b, C->b));
    int64_t px0 = (int64_t)ceil(amin - 0.5), px1 = (int64_t)floor(amax - 0.5), py0 = (int64_t)ceil(bmin - 0.5), py1 = (int64_t)floor(bmax - 0.5);
    if (px0 < 0) px0 = 0; if (py0 < 0) py0 = 0; if (px1 > W - 1) px1 = W - 1; if (py1 > H - 1) py1 = H - 1;
    for (int64_t py = py0; py <= py1; ++py) for (int64_t px = px0; px <= px1; ++px) {
        const double a = (double)px + 0.5, b = (double)py + 0.5;
        /* edge functions = twice the signed areas of (P, B, C), (A, P, C), (A, B, P) */
        const double w0 = fma(B->a - a, C->b - b, -((B->b - b) * (C->a - a)));
        const double w1 = fma(C->a - a, A->b - b, -((C->b - b) * (A->a - a)));
        const double w2 = fma(A->a - a, B->b - b, -((A->b - b) * (B->a - a)));
        /* inside or on the boundary; a pixel centre exactly on an edge shared by two triangles must not fall between them
           when the two roundings of that edge function disagree in sign: slack 1e-12 |area| */
        const double sg = (area > 0.0) ? 1.0 : -1.0, slack = -1e-12 * fabs(area);
        const int in = (sg * w0 >= slack && sg * w1 >= slack && sg * w2 >= slack);
        if (!in) continue;
        const double l0 = w0 / area, l1 = w1 / area, l2 = w2 / area;
        const double depth = fma(l2, C->d, fma(l1, B->d, l0 * A->d));
        const double col = fma(l2, C->col, fma(l1, B->col, l0 * A->col));
        double qd = (depth - dlo) / (dhi - dlo);
        if (!(qd > 0.0)) qd = 0.0;
        if (qd > 1.0) qd = 1.0;
        const uint64_t dq = (uint64_t)floor(qd * 4294967295.0);
        const uint64_t kk = (dq << 32) | (uint64_t)orc_color(cm, col, shade);
        if (kk < key[py * W + px]) key[py * W + px] = kk;
    }
}

/* (2) iso-surface of `field` at `iso`, coloured by `cfield` (NULL: by the iso value).  depth range [dlo, dhi] of the
 * scene along w (the caller passes the range of (X - origin) . w over the mesh).  rgba [W*H]. */
void orc_image_isosurface(int64_t E, int N, const double* x, const double* y, const double* z, const double* field,
                          double iso, const double* cfield, const img_view* vw, const img_cmap* cm, const double* light,
                          double dlo, double dhi, uint32_t* rgba, uint64_t* key_out)
{
    const int W = vw->width, H = vw->height;
    double w[3];
    cross3(vw->u, vw->v, w);
    uint64_t* key = (uint64_t*)malloc(sizeof(uint64_t) * (size_t)W * H);
    for (int64_t p = 0; p < (int64_t)W * H; ++p) key[p] = 0xffffffff00000000ull | (uint64_t)cm->background;
    for (int64_t e = 0; e < E; ++e)
        for (int k = 0; k < N; ++k) for (int j = 0; j < N; ++j) for (int i = 0; i < N; ++i) {
            int64_t id[8];
            cell_nodes(N, e, i, j, k, id);
            double fv[8], fmin_ = INFINITY, fmax_ = -INFINITY;
            for (int q = 0; q < 8; ++q) { fv[q] = field[id[q]]; fmin_ = fmin(fmin_, fv[q]); fmax_ = fmax(fmax_, fv[q]); }
            if (!(fmin_ < iso && fmax_ >= iso)) continue;
            img_vert V[8];
            for (int q = 0; q < 8; ++q) {
                V[q].X[0] = x[id[q]]; V[q].X[1] = y[id[q]]; V[q].X[2] = z[id[q]];
                project(vw, w, V[q].X[0], V[q].X[1], V[q].X[2], &V[q].a, &V[q].b, &V[q].d);
                V[q].col = cfield ? cfield[id[q]] : iso;
            }
            for (int tt = 0; tt < 6; ++tt) {
                /* corners above (f >= iso) and below the level, in the tetrahedron's own order */
                int up[4], dn[4], nu = 0, nd = 0;
                for (int c = 0; c < 4; ++c) { const int q = TET[tt][c]; if (fv[q] >= iso) up[nu++] = q; else dn[nd++] = q; }
                if (nu == 0 || nd == 0) continue;
                img_vert P[4];
                if (nu == 1 || nd == 1) {
                    /* one corner on its own: a triangle on the three edges leaving it */
                    const int apex = (nu == 1) ? up[0] : dn[0];
                    const int* oth = (nu == 1) ? dn : up;
                    for (int c = 0; c < 3; ++c) edge_point(&V[apex], &V[oth[c]], fv[apex], fv[oth[c]], iso, &P[c]);
                    raster_tri(vw, cm, light, dlo, dhi, &P[0], &P[1], &P[2], key);
                } else {
                    /* two and two: a quadrilateral u0d0, u0d1, u1d1, u1d0 split along u0d0 - u1d1 */
                    edge_point(&V[up[0]], &V[dn[0]], fv[up[0]], fv[dn[0]], iso, &P[0]);
                    edge_point(&V[up[0]], &V[dn[1]], fv[up[0]], fv[dn[1]], iso, &P[1]);
                    edge_point(&V[up[1]], &V[dn[1]], fv[up[1]], fv[dn[1]], iso, &P[2]);
                    edge_point(&V[up[1]], &V[dn[0]], fv[up[1]], fv[dn[0]], iso, &P[3]);
                    raster_tri(vw, cm, light, dlo, dhi, &P[0], &P[1], &P[2], key);
                    raster_tri(vw, cm, light, dlo, dhi, &P[0], &P[2], &P[3], key);
                }
            }
        }
    for (int64_t p = 0; p < (int64_t)W * H; ++p) { rgba[p] = (uint32_t)(key[p] & 0xffffffffull); if (key_out) key_out[p] = key[p]; }
    free(key);
}
