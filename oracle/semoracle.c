/*
 * semoracle.c — plain, slow, obviously-correct CPU oracle for the spectral-element
 * Poisson/Helmholtz hot path (axhelm, gather-scatter, mask, Jacobi / Chebyshev-Jacobi,
 * PCG, min/max/histogram consumer).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code,
 * header, table or constant generator with the CUDA path (paper_2501_13240_b200/csrc).
 *
 * What it follows.  The paper states the method only in prose:
 *   PAPER.md:L85  (§2.2) SEM of order p, GLL quadrature, tensor-product (ijk) ordering
 *                 on [-1,1]^3, n ~ N_e p^3 unknowns;
 *   PAPER.md:L100 (§2.2) operators = dense contractions with (p+1)x(p+1) matrices that
 *                 are the same for all elements; deformed elements via the chain rule;
 *   PAPER.md:L102 (§2.2) surface data exchanged/summed between elements (direct-stiffness
 *                 summation); pressure Poisson solve is the stiffest sub-step; Chebyshev
 *                 acceleration of the smoother;
 *   PAPER.md:L238 (§4.1) isothermal, no-slip plates (Dirichlet), periodic x,y;
 *   PAPER.md:L128, L138-159 (§2.3, §3.1) zero-copy hand-off of device arrays.
 * The operator w = D^T G D u + lambda B u, QQ^T, masking, Jacobi/Chebyshev-Jacobi and PCG
 * are named by BASELINE.json:north_star; the formulas are the standard SEM ones, written
 * out in SURVEY.md §8(c) items c-1 .. c-11, which every function below cites.
 * Readings taken where the paper is silent are listed in DESIGN.md ("Readings").
 *
 * Everything is fp64, loops are in the order the definitions state (m ascending, local
 * index l ascending), no blocking, no fusion.  The only pragma is a trivial OpenMP
 * "parallel for" over elements in axhelm/geo/diag which does not change
 * any result (elements are independent).
 *
 * Layout: local node l = e*Np + k*n1*n1 + j*n1 + i, i fastest ("(ijk) ordering").
 * geo[e][g][Np], g = 0..6 : G_rr, G_rs, G_rt, G_ss, G_st, G_tt, B.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P1-P16 of SURVEY.md §8(c).  The "next" rows built so far follow the
 * same rule: p-multigrid V-cycle (f-1, R19: orc_interp_matrix, orc_interp3, orc_mg_*; pins: Vandermonde
 * interpolation, Kronecker transfer, adjointness, dense V-cycle composition, bounds covering the dense spectrum),
 * fourth-kind Chebyshev smoother (closed-form residual polynomial), FP32-storage levels (R21: a float-rounding
 * perturbation of the pinned fp64 cycle), all-Neumann solves (R20, in semoracle.py: pseudo-inverse solution).
 * Functions with no independent pin: none ("parity unpinned" list is empty; see DESIGN.md §Oracle pins).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_MAXN1 16

/* ------------------------------------------------------------------------------------ */
/* c-1  GLL nodes and weights ("GLL quadrature").              */
/* Legendre P_N and P_{N-1} by the three-term recurrence.                                */
static void legendre(int N, double x, double* PN, double* PNm1)
{
    double p0 = 1.0, p1 = x;
    if (N == 0) { *PN = 1.0; *PNm1 = 0.0; return; }
    for (int n = 1; n < N; ++n) {
        double p2 = ((2.0 * n + 1.0) * x * p1 - n * p0) / (n + 1.0);
        p0 = p1; p1 = p2;
    }
    *PN = p1; *PNm1 = p0;
}

/* xi[0..N], rho[0..N].  Interior nodes = roots of P'_N by Newton from the
 * Chebyshev-Lobatto guess; rho_i = 2 / (N (N+1) P_N(xi_i)^2); then symmetrised. */
int orc_gll(int N, double* xi, double* rho)
{
    if (N < 1 || N + 1 > ORC_MAXN1) return -1;
    const double pi = 3.14159265358979323846;
    xi[0] = -1.0; xi[N] = 1.0;
    for (int i = 1; i < N; ++i) {
        double x = -cos(pi * i / N);
        for (int it = 0; it < 100; ++it) {
            double PN, PNm1;
            legendre(N, x, &PN, &PNm1);
            /* P'_N = N (x P_N - P_{N-1}) / (x^2 - 1);
             * (1-x^2) P''_N = 2 x P'_N - N (N+1) P_N   (Legendre ODE) */
            double dP  = N * (x * PN - PNm1) / (x * x - 1.0);
            double d2P = (2.0 * x * dP - N * (N + 1.0) * PN) / (1.0 - x * x);
            double dx  = dP / d2P;
            x -= dx;
            if (fabs(dx) <= 1e-16 * (1.0 + fabs(x))) break;
        }
        xi[i] = x;
    }
    for (int i = 0; i <= N / 2; ++i) {           /* symmetrise xi_{N-i} = -xi_i */
        double a = 0.5 * (xi[N - i] - xi[i]);
        xi[i] = -a; xi[N - i] = a;
    }
    if (N % 2 == 0) xi[N / 2] = 0.0;
    for (int i = 0; i <= N; ++i) {
        double PN, PNm1;
        legendre(N, xi[i], &PN, &PNm1);
        rho[i] = 2.0 / (N * (N + 1.0) * PN * PN);
    }
    for (int i = 0; i <= N / 2; ++i) {
        double a = 0.5 * (rho[i] + rho[N - i]);
        rho[i] = a; rho[N - i] = a;
    }
    return 0;
}

/* c-2  D[i*n1+j] = l'_j(xi_i) = P_N(xi_i) / (P_N(xi_j) (xi_i - xi_j)), i != j;
 * diagonal = minus the sum of the off-diagonal row entries (reading R2:
 * rows sum to 0 exactly up to the rounding of that sum, so that A*const = 0). */
int orc_dhat(int N, const double* xi, double* D)
{
    int n1 = N + 1;
    if (N < 1 || n1 > ORC_MAXN1) return -1;
    double P[ORC_MAXN1];
    for (int i = 0; i < n1; ++i) { double t; legendre(N, xi[i], &P[i], &t); }
    for (int i = 0; i < n1; ++i) {
        double s = 0.0;
        for (int j = 0; j < n1; ++j) {
            if (j == i) continue;
            D[i * n1 + j] = P[i] / (P[j] * (xi[i] - xi[j]));
            s += D[i * n1 + j];
        }
        D[i * n1 + i] = -s;
    }
    return 0;
}

/* ------------------------------------------------------------------------------------ */
/* c-3  geometric factors ("chain rule" folded with the GLL weights of L85).
 * Returns -1 if all Jacobians are positive, else the first element with J <= 0.         */
int64_t orc_geo(int64_t E, int N, const double* x, const double* y, const double* z,
                const double* D, const double* rho, double* geo)
{
    const int n1 = N + 1, Np = n1 * n1 * n1;
    int64_t bad = -1;
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < E; ++e) {
        const double* X = x + e * Np; const double* Y = y + e * Np; const double* Z = z + e * Np;
        double* g = geo + e * 7 * (int64_t)Np;
        for (int k = 0; k < n1; ++k)
        for (int j = 0; j < n1; ++j)
        for (int i = 0; i < n1; ++i) {
            double xr = 0, xs = 0, xt = 0, yr = 0, ys = 0, yt = 0, zr = 0, zs = 0, zt = 0;
            for (int m = 0; m < n1; ++m) {
                int ir = k * n1 * n1 + j * n1 + m;
                int is = k * n1 * n1 + m * n1 + i;
                int it = m * n1 * n1 + j * n1 + i;
                xr += D[i * n1 + m] * X[ir]; xs += D[j * n1 + m] * X[is]; xt += D[k * n1 + m] * X[it];
                yr += D[i * n1 + m] * Y[ir]; ys += D[j * n1 + m] * Y[is]; yt += D[k * n1 + m] * Y[it];
                zr += D[i * n1 + m] * Z[ir]; zs += D[j * n1 + m] * Z[is]; zt += D[k * n1 + m] * Z[it];
            }
            double J = xr * (ys * zt - yt * zs) - xs * (yr * zt - yt * zr) + xt * (yr * zs - ys * zr);
            if (!(J > 0.0)) {
#pragma omp critical
                { if (bad < 0 || e < bad) bad = e; }
            }
            double rx =  (ys * zt - yt * zs) / J, ry = -(xs * zt - xt * zs) / J, rz =  (xs * yt - xt * ys) / J;
            double sx = -(yr * zt - yt * zr) / J, sy =  (xr * zt - xt * zr) / J, sz = -(xr * yt - xt * yr) / J;
            double tx =  (yr * zs - ys * zr) / J, ty = -(xr * zs - xs * zr) / J, tz =  (xr * ys - xs * yr) / J;
            double W = rho[i] * rho[j] * rho[k];
            int l = k * n1 * n1 + j * n1 + i;
            g[0 * Np + l] = W * J * (rx * rx + ry * ry + rz * rz);
            g[1 * Np + l] = W * J * (rx * sx + ry * sy + rz * sz);
            g[2 * Np + l] = W * J * (rx * tx + ry * ty + rz * tz);
            g[3 * Np + l] = W * J * (sx * sx + sy * sy + sz * sz);
            g[4 * Np + l] = W * J * (sx * tx + sy * ty + sz * tz);
            g[5 * Np + l] = W * J * (tx * tx + ty * ty + tz * tz);
            g[6 * Np + l] = W * J;
        }
    }
    return bad;
}

/* ------------------------------------------------------------------------------------ */
/* c-4  axhelm, the plain definition (north_star: w = D^T G D u + lambda B u).
 * lam0/lam1 (may be NULL): per-node coefficients, w = D^T (lam0 G) D u + lam1 B u
 * (reading R3 / SURVEY A3); with both NULL the scalar lambda multiplies B.      */
void orc_axhelm(int64_t E, int N, const double* geo, const double* D, double lambda,
                const double* lam0, const double* lam1, const double* u, double* w)
{
    const int n1 = N + 1, Np = n1 * n1 * n1;
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < E; ++e) {
        const double* U = u + e * Np;
        const double* g = geo + e * 7 * (int64_t)Np;
        double* W = w + e * Np;
        double* gr = (double*)malloc(sizeof(double) * 3 * Np);
        double* gs = gr + Np; double* gt = gs + Np;
        for (int k = 0; k < n1; ++k)
        for (int j = 0; j < n1; ++j)
        for (int i = 0; i < n1; ++i) {
            double ur = 0, us = 0, ut = 0;
            for (int m = 0; m < n1; ++m) {
                ur += D[i * n1 + m] * U[k * n1 * n1 + j * n1 + m];
                us += D[j * n1 + m] * U[k * n1 * n1 + m * n1 + i];
                ut += D[k * n1 + m] * U[m * n1 * n1 + j * n1 + i];
            }
            int l = k * n1 * n1 + j * n1 + i;
            double c = lam0 ? lam0[e * Np + l] : 1.0;
            double Grr = c * g[0 * Np + l], Grs = c * g[1 * Np + l], Grt = c * g[2 * Np + l];
            double Gss = c * g[3 * Np + l], Gst = c * g[4 * Np + l], Gtt = c * g[5 * Np + l];
            gr[l] = Grr * ur + Grs * us + Grt * ut;
            gs[l] = Grs * ur + Gss * us + Gst * ut;
            gt[l] = Grt * ur + Gst * us + Gtt * ut;
        }
        for (int k = 0; k < n1; ++k)
        for (int j = 0; j < n1; ++j)
        for (int i = 0; i < n1; ++i) {
            double s = 0;
            for (int m = 0; m < n1; ++m) {
                s += D[m * n1 + i] * gr[k * n1 * n1 + j * n1 + m];
                s += D[m * n1 + j] * gs[k * n1 * n1 + m * n1 + i];
                s += D[m * n1 + k] * gt[m * n1 * n1 + j * n1 + i];
            }
            int l = k * n1 * n1 + j * n1 + i;
            double lam = lam1 ? lam1[e * Np + l] : lambda;
            W[l] = s + lam * g[6 * Np + l] * U[l];
        }
        free(gr);
    }
}

/* ------------------------------------------------------------------------------------ */
/* smallest distance between neighbouring GLL nodes of any element (along r, s and t);
 * the matching tolerance of c-6 is 1e-8 times this.                      */
double orc_min_spacing(int64_t E, int N, const double* x, const double* y, const double* z)
{
    const int n1 = N + 1, Np = n1 * n1 * n1;
    double best = INFINITY;
    for (int64_t e = 0; e < E; ++e)
        for (int k = 0; k < n1; ++k)
        for (int j = 0; j < n1; ++j)
        for (int i = 0; i < n1; ++i) {
            int64_t l = e * Np + k * n1 * n1 + j * n1 + i;
            int64_t nb[3] = { i + 1 < n1 ? l + 1 : -1, j + 1 < n1 ? l + n1 : -1, k + 1 < n1 ? l + n1 * n1 : -1 };
            for (int d = 0; d < 3; ++d) {
                if (nb[d] < 0) continue;
                double dx = x[nb[d]] - x[l], dy = y[nb[d]] - y[l], dz = z[nb[d]] - z[l];
                double dist = sqrt(dx * dx + dy * dy + dz * dz);
                if (dist < best) best = dist;
            }
        }
    return best;
}

/* c-6  global numbering.  Two local nodes are the same global node iff their coordinates
 * agree within tol in every direction after wrapping periodic directions (PAPER.md:L102 is
 * the only description of the inter-element exchange; L238 gives the periodic x,y).  The
 * canonical ("first-touch") id of a class is the rank of its smallest local index.
 * Candidates are found through a sorted cell list (cell edge hc >= 4 tol; a match lies in
 * the same or a face/edge/corner-adjacent cell).  Returns n_unique, or -1 if "within tol"
 * turned out not to be an equivalence relation on this mesh (tolerance unusable).        */
typedef struct { int64_t c[3]; int64_t l; } orc_cell;

static int cell_cmp(const void* a, const void* b)
{
    const orc_cell* A = (const orc_cell*)a; const orc_cell* B = (const orc_cell*)b;
    for (int d = 0; d < 3; ++d) { if (A->c[d] < B->c[d]) return -1; if (A->c[d] > B->c[d]) return 1; }
    return (A->l < B->l) ? -1 : (A->l > B->l);
}

static double wrap_coord(double c, double period, double tol)
{
    if (period > 0.0) {
        c -= period * floor(c / period);
        if (c >= period - tol) c -= period;      /* seam copies land next to 0 */
    }
    return c;
}

int64_t orc_numbering(int64_t E, int N, const double* x, const double* y, const double* z,
                      const double* period, double tol, int32_t* gid)
{
    const int n1 = N + 1, Np = n1 * n1 * n1;
    const int64_t n = E * Np;
    const double* X[3] = { x, y, z };
    const double hc = 16.0 * tol;
    /* surface nodes only: an element-interior node has no copy */
    int64_t ns = 0;
    orc_cell* cells = (orc_cell*)malloc(sizeof(orc_cell) * (size_t)n);
    double* cw = (double*)malloc(sizeof(double) * 3 * (size_t)n);
    int64_t* label = (int64_t*)malloc(sizeof(int64_t) * (size_t)n);
    for (int64_t l = 0; l < n; ++l) {
        int loc = (int)(l % Np), i = loc % n1, j = (loc / n1) % n1, k = loc / (n1 * n1);
        label[l] = l;
        for (int d = 0; d < 3; ++d) cw[3 * l + d] = wrap_coord(X[d][l], period[d], tol);
        if (i == 0 || i == N || j == 0 || j == N || k == 0 || k == N) {
            for (int d = 0; d < 3; ++d) cells[ns].c[d] = (int64_t)floor(cw[3 * l + d] / hc);
            cells[ns].l = l; ++ns;
        }
    }
    qsort(cells, (size_t)ns, sizeof(orc_cell), cell_cmp);
    for (int64_t s = 0; s < ns; ++s) {
        int64_t l = cells[s].l, best = l;
        for (int ox = -1; ox <= 1; ++ox) for (int oy = -1; oy <= 1; ++oy) for (int oz = -1; oz <= 1; ++oz) {
            orc_cell key; key.c[0] = cells[s].c[0] + ox; key.c[1] = cells[s].c[1] + oy; key.c[2] = cells[s].c[2] + oz;
            key.l = -1;
            int64_t lo = 0, hi = ns;                     /* lower bound of the cell's run */
            while (lo < hi) { int64_t mid = (lo + hi) / 2; if (cell_cmp(&cells[mid], &key) < 0) lo = mid + 1; else hi = mid; }
            for (int64_t t = lo; t < ns && cells[t].c[0] == key.c[0] && cells[t].c[1] == key.c[1] && cells[t].c[2] == key.c[2]; ++t) {
                int64_t l2 = cells[t].l;
                if (fabs(cw[3 * l2] - cw[3 * l]) <= tol && fabs(cw[3 * l2 + 1] - cw[3 * l + 1]) <= tol &&
                    fabs(cw[3 * l2 + 2] - cw[3 * l + 2]) <= tol && l2 < best) best = l2;
            }
        }
        label[l] = best;
    }
    int64_t nu = 0, ok = 1;
    for (int64_t l = 0; l < n; ++l) {
        if (label[label[l]] != label[l]) ok = 0;
        if (label[l] == l) gid[l] = (int32_t)nu++; else gid[l] = gid[label[l]];
    }
    free(cells); free(cw); free(label);
    return ok ? nu : -1;
}

/* c-7  gather-scatter QQ^T: s_g = sum of the copies in ascending local index,
 * written back to every copy.                                                            */
void orc_gs(int64_t n, const int32_t* gid, int64_t n_unique, double* w)
{
    double* s = (double*)calloc((size_t)n_unique, sizeof(double));
    for (int64_t l = 0; l < n; ++l) s[gid[l]] += w[l];
    for (int64_t l = 0; l < n; ++l) w[l] = s[gid[l]];
    free(s);
}

/* c-6/c-8  Dirichlet mask: mask[l] = 0 if the global node of l lies on a face whose
 * tag t has bit t set in tags (OR over all copies), else 1.  Faces: r-,r+,s-,s+,t-,t+.    */
void orc_mask(int64_t E, int N, const int32_t* face_tag, uint32_t tags, const int32_t* gid,
              int64_t n_unique, double* mask)
{
    const int n1 = N + 1, Np = n1 * n1 * n1;
    unsigned char* flag = (unsigned char*)calloc((size_t)n_unique, 1);
    for (int64_t e = 0; e < E; ++e)
        for (int k = 0; k < n1; ++k) for (int j = 0; j < n1; ++j) for (int i = 0; i < n1; ++i) {
            int on[6] = { i == 0, i == N, j == 0, j == N, k == 0, k == N };
            for (int f = 0; f < 6; ++f) {
                int32_t t = face_tag[e * 6 + f];
                if (on[f] && t > 0 && t < 32 && ((tags >> t) & 1u)) flag[gid[e * Np + k * n1 * n1 + j * n1 + i]] = 1;
            }
        }
    for (int64_t l = 0; l < E * Np; ++l) mask[l] = flag[gid[l]] ? 0.0 : 1.0;
    free(flag);
}

/* c-7  exact diagonal of the local operator D^T G D + lambda B.                           */
void orc_diag_local(int64_t E, int N, const double* geo, const double* D, double lambda, double* d)
{
    const int n1 = N + 1, Np = n1 * n1 * n1;
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < E; ++e) {
        const double* g = geo + e * 7 * (int64_t)Np;
        for (int k = 0; k < n1; ++k) for (int j = 0; j < n1; ++j) for (int i = 0; i < n1; ++i) {
            int l = k * n1 * n1 + j * n1 + i;
            double s = 0;
            for (int m = 0; m < n1; ++m) {
                s += D[m * n1 + i] * D[m * n1 + i] * g[0 * Np + k * n1 * n1 + j * n1 + m];
                s += D[m * n1 + j] * D[m * n1 + j] * g[3 * Np + k * n1 * n1 + m * n1 + i];
                s += D[m * n1 + k] * D[m * n1 + k] * g[5 * Np + m * n1 * n1 + j * n1 + i];
            }
            s += 2.0 * (D[i * n1 + i] * D[j * n1 + j] * g[1 * Np + l] + D[i * n1 + i] * D[k * n1 + k] * g[2 * Np + l] +
                        D[j * n1 + j] * D[k * n1 + k] * g[4 * Np + l]);
            d[e * Np + l] = s + lambda * g[6 * Np + l];
        }
    }
}

/* ------------------------------------------------------------------------------------ */
/* c-8  assembled, masked operator and inner products on local (redundant) storage.       */
typedef struct {
    int64_t E; int32_t N; int32_t pad_; int64_t n; int64_t n_unique;
    const double* geo; const double* D; const int32_t* gid;
    const double* mask;      /* 1 / 0 per local node (orc_mask) */
    const double* invmult;   /* 1 / multiplicity per local node  */
    double lambda;
} orc_op;

/* f-1, reading R21: FP32 STORAGE of the multigrid levels.  While g_r32 is set (only inside
 * orc_mg_vcycle with mg->fp32), every vector an operation of the V-cycle produces is rounded to float where it would
 * be stored; the arithmetic stays fp64.  Off everywhere else, so nothing outside the fp32 V-cycle changes. */
static int g_r32 = 0;
static void rnd32(double* v, int64_t n)
{
    if (!g_r32) return;
    for (int64_t l = 0; l < n; ++l) v[l] = (double)(float)v[l];
}

/* out = M QQ^T ( A_L ( M v ) );  tmp is scratch [n] */
void orc_apply_A(const orc_op* op, const double* v, double* out, double* tmp)
{
    for (int64_t l = 0; l < op->n; ++l) tmp[l] = op->mask[l] * v[l];
    orc_axhelm(op->E, op->N, op->geo, op->D, op->lambda, NULL, NULL, tmp, out);
    rnd32(out, op->n);
    orc_gs(op->n, op->gid, op->n_unique, out);
    for (int64_t l = 0; l < op->n; ++l) out[l] *= op->mask[l];
    rnd32(out, op->n);
}

/* <a,b> = sum_l a_l b_l / mult_l  (= dot product over unique nodes for continuous a,b) */
double orc_dot(const orc_op* op, const double* a, const double* b)
{
    double s = 0;
    for (int64_t l = 0; l < op->n; ++l) s += a[l] * b[l] * op->invmult[l];
    return s;
}

/* invmult = 1 / (QQ^T 1) */
void orc_invmult(int64_t n, const int32_t* gid, int64_t n_unique, double* invmult)
{
    for (int64_t l = 0; l < n; ++l) invmult[l] = 1.0;
    orc_gs(n, gid, n_unique, invmult);
    for (int64_t l = 0; l < n; ++l) invmult[l] = 1.0 / invmult[l];
}

/* c-7 / a-4  dinv = 1 / (QQ^T diag_local), 1 at masked nodes */
void orc_dinv(const orc_op* op, double* dinv)
{
    orc_diag_local(op->E, op->N, op->geo, op->D, op->lambda, dinv);
    orc_gs(op->n, op->gid, op->n_unique, dinv);
    for (int64_t l = 0; l < op->n; ++l) dinv[l] = (op->mask[l] == 0.0) ? 1.0 : 1.0 / dinv[l];
}

/* b = M QQ^T (B o f)  (c-8) */
void orc_assemble_rhs(const orc_op* op, const double* f, double* b)
{
    const int Np = (op->N + 1) * (op->N + 1) * (op->N + 1);
    for (int64_t e = 0; e < op->E; ++e)
        for (int l = 0; l < Np; ++l) b[e * Np + l] = op->geo[e * 7 * (int64_t)Np + 6 * Np + l] * f[e * Np + l];
    orc_gs(op->n, op->gid, op->n_unique, b);
    for (int64_t l = 0; l < op->n; ++l) b[l] *= op->mask[l];
}

/* c-10  Chebyshev-Jacobi(k) preconditioner, 1st-kind recurrence on [0.1 lmax, lmax]
 * (PAPER.md:L102 names Chebyshev acceleration; bounds and kind: DESIGN.md reading R9).
 * work: 4 vectors [n].                                                                    */
void orc_cheb_jacobi_frac(const orc_op* op, int k, double lmax, double lmin_frac, const double* dinv, const double* r,
                          double* z, double* work);
void orc_cheb_jacobi(const orc_op* op, int k, double lmax, const double* dinv, const double* r,
                     double* z, double* work)
{
    orc_cheb_jacobi_frac(op, k, lmax, 0.1, dinv, r, z, work);
}
/* the same recurrence on [lmin_frac, 1] lmax (f-1: the last multigrid level may use a smaller fraction and a higher
 * degree, which turns the smoother into an approximate coarse solver) */
void orc_cheb_jacobi_frac(const orc_op* op, int k, double lmax, double lmin_frac, const double* dinv, const double* r,
                          double* z, double* work)
{
    const int64_t n = op->n;
    double* res = work; double* d = work + n; double* Ad = work + 2 * n; double* tmp = work + 3 * n;
    const double lmin = lmin_frac * lmax, theta = 0.5 * (lmax + lmin), delta = 0.5 * (lmax - lmin);
    const double sigma = theta / delta;
    double rho = 1.0 / sigma;
    for (int64_t l = 0; l < n; ++l) { z[l] = 0.0; res[l] = r[l]; d[l] = dinv[l] * res[l] / theta; }
    rnd32(d, n);
    for (int it = 0; it < k; ++it) {
        for (int64_t l = 0; l < n; ++l) z[l] += d[l];
        rnd32(z, n);
        orc_apply_A(op, d, Ad, tmp);
        for (int64_t l = 0; l < n; ++l) res[l] -= Ad[l];
        rnd32(res, n);
        double rho1 = 1.0 / (2.0 * sigma - rho);
        for (int64_t l = 0; l < n; ++l) d[l] = rho1 * rho * d[l] + (2.0 * rho1 / delta) * (dinv[l] * res[l]);
        rnd32(d, n);
        rho = rho1;
    }
    for (int64_t l = 0; l < n; ++l) z[l] += d[l];
    rnd32(z, n);
}

/* ------------------------------------------------------------------------------------ */
/* f-1  p-multigrid V-cycle preconditioner (§2.2: "p-multigrid ... Chebyshev-accelerated
 * ... smoothers" is NekRS's pressure preconditioner; the paper gives no formulas, reading R19
 * fixes them).  Levels l = 0 (order N, the problem) .. L-1 (coarsest), each a re-discretisation of the
 * same elements at order N_l: its own geometric factors, numbering, mask and Jacobi diagonal (orc_op).
 *   prolongation   P_l : level l+1 -> l,  per element  v_f(i,j,k) = sum_abc J_ia J_jb J_kc v_c(a,b,c),
 *                  J_ia = l^(l+1)_a(xi^(l)_i)  (coarse Lagrange basis at the fine GLL nodes);
 *   restriction    R_l = M_c QQ^T_c (J^T x J^T x J^T)(invmult_f o r)   (the transpose of P_l on unique nodes);
 *   smoother       S_l = Chebyshev-Jacobi(k) of c-10 on level l;
 *   V(l, r):  coarsest: z = S(r) with degree k_coarse;  else
 *             z = S r;  res = r - A z;  z += P V(l+1, R res);  res = r - A z;  z += S res.          */
typedef struct {
    orc_op op;
    const double* dinv;
    double lmax;
    const double* J;         /* [n1_l][n1_{l+1}] row-major; NULL on the coarsest level */
} orc_mg_level;
typedef struct {
    int32_t nlevels, k_smooth, k_coarse, kind;      /* kind: 4 = fourth-kind Chebyshev smoother, else first kind (c-10) */
    double coarse_frac;                             /* first kind, last level: interval [coarse_frac, 1] lmax (0.1 = c-10) */
    orc_mg_level lev[8];
} orc_mg;

/* J[(Nto+1) x (Nfrom+1)], J_ia = a-th Lagrange polynomial on the GLL nodes of order Nfrom at the
 * i-th GLL node of order Nto (product formula: rows at coinciding nodes are exact unit vectors) */
int orc_interp_matrix(int Nfrom, int Nto, double* J)
{
    double xf[ORC_MAXN1], xt[ORC_MAXN1], w[ORC_MAXN1];
    if (orc_gll(Nfrom, xf, w) || orc_gll(Nto, xt, w)) return -1;
    for (int i = 0; i <= Nto; ++i)
        for (int a = 0; a <= Nfrom; ++a) {
            double v = 1.0;
            for (int m = 0; m <= Nfrom; ++m) if (m != a) v *= (xt[i] - xf[m]) / (xf[a] - xf[m]);
            J[i * (Nfrom + 1) + a] = v;
        }
    return 0;
}

/* per element: transpose == 0: out(i,j,k) = sum_abc J_ia J_jb J_kc in(a,b,c)   (in: nc1^3, out: nf1^3)
 *              transpose != 0: out(a,b,c) = sum_ijk J_ia J_jb J_kc in(i,j,k)   (in: nf1^3, out: nc1^3)
 * J is [nf1][nc1].  The definition written out, no sum factorisation. */
void orc_interp3(int64_t E, int nf1, int nc1, const double* J, int transpose, const double* in, double* out)
{
    const int Nf = nf1 * nf1 * nf1, Nc = nc1 * nc1 * nc1;
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < E; ++e) {
        const double* vi = in + e * (transpose ? Nf : Nc);
        double* vo = out + e * (transpose ? Nc : Nf);
        if (!transpose) {
            for (int k = 0; k < nf1; ++k) for (int j = 0; j < nf1; ++j) for (int i = 0; i < nf1; ++i) {
                double s = 0;
                for (int c = 0; c < nc1; ++c) for (int b = 0; b < nc1; ++b) for (int a = 0; a < nc1; ++a)
                    s += J[i * nc1 + a] * J[j * nc1 + b] * J[k * nc1 + c] * vi[(c * nc1 + b) * nc1 + a];
                vo[(k * nf1 + j) * nf1 + i] = s;
            }
        } else {
            for (int c = 0; c < nc1; ++c) for (int b = 0; b < nc1; ++b) for (int a = 0; a < nc1; ++a) {
                double s = 0;
                for (int k = 0; k < nf1; ++k) for (int j = 0; j < nf1; ++j) for (int i = 0; i < nf1; ++i)
                    s += J[i * nc1 + a] * J[j * nc1 + b] * J[k * nc1 + c] * vi[(k * nf1 + j) * nf1 + i];
                vo[(c * nc1 + b) * nc1 + a] = s;
            }
        }
    }
}

/* v_f = M_f P v_c */
void orc_mg_prolong(const orc_mg* mg, int l, const double* vc, double* vf)
{
    const orc_op* f = &mg->lev[l].op; const orc_op* c = &mg->lev[l + 1].op;
    orc_interp3(f->E, f->N + 1, c->N + 1, mg->lev[l].J, 0, vc, vf);
    for (int64_t q = 0; q < f->n; ++q) vf[q] *= f->mask[q];
    rnd32(vf, f->n);
}
/* r_c = M_c QQ^T_c J^T (invmult_f o r_f);  tmp: [n_f] */
void orc_mg_restrict(const orc_mg* mg, int l, const double* rf, double* rc, double* tmp)
{
    const orc_op* f = &mg->lev[l].op; const orc_op* c = &mg->lev[l + 1].op;
    for (int64_t q = 0; q < f->n; ++q) tmp[q] = f->invmult[q] * rf[q];
    orc_interp3(f->E, f->N + 1, c->N + 1, mg->lev[l].J, 1, tmp, rc);
    rnd32(rc, c->n);
    orc_gs(c->n, c->gid, c->n_unique, rc);
    for (int64_t q = 0; q < c->n; ++q) rc[q] *= c->mask[q];
    rnd32(rc, c->n);
}

/* f-1  Chebyshev-Jacobi smoother of the FOURTH kind ("fourth-kind Chebyshev-accelerated"
 * smoothers; the recurrence is the published one for polynomial smoothers that need only the upper bound lmax
 * of spec(D^-1 A), restated):
 *   z = 0; res = r; d = (4/3)(1/lmax) dinv o res;
 *   for i = 1..k { z += d; res -= A d; d = ((2i-1)/(2i+3)) d + ((8i+4)/(2i+3)) (1/lmax) dinv o res };  z += d
 * so that 1 - lam p_k(lam) = W_{k+1}(1 - 2 lam/lmax) / (2k+3), W_n the Chebyshev polynomial of the 4th kind
 * (pin: tests/test_oracle_multigrid.py).  work: 4 vectors [n].                                        */
void orc_cheb4_jacobi(const orc_op* op, int k, double lmax, const double* dinv, const double* r,
                      double* z, double* work)
{
    const int64_t n = op->n;
    double* res = work; double* d = work + n; double* Ad = work + 2 * n; double* tmp = work + 3 * n;
    for (int64_t l = 0; l < n; ++l) { z[l] = 0.0; res[l] = r[l]; d[l] = dinv[l] * res[l] * (4.0 / (3.0 * lmax)); }
    rnd32(d, n);
    for (int i = 1; i <= k; ++i) {
        for (int64_t l = 0; l < n; ++l) z[l] += d[l];
        rnd32(z, n);
        orc_apply_A(op, d, Ad, tmp);
        for (int64_t l = 0; l < n; ++l) res[l] -= Ad[l];
        rnd32(res, n);
        const double c1 = (2.0 * i - 1.0) / (2.0 * i + 3.0), c2 = (8.0 * i + 4.0) / ((2.0 * i + 3.0) * lmax);
        for (int64_t l = 0; l < n; ++l) d[l] = c1 * d[l] + c2 * (dinv[l] * res[l]);
        rnd32(d, n);
    }
    for (int64_t l = 0; l < n; ++l) z[l] += d[l];
    rnd32(z, n);
}
static void mg_smooth(const orc_mg* mg, const orc_mg_level* L, int k, const double* r, double* z, double* work)
{
    const int last = (L == &mg->lev[mg->nlevels - 1]);
    if (mg->kind == 4) orc_cheb4_jacobi(&L->op, k, L->lmax, L->dinv, r, z, work);
    else               orc_cheb_jacobi_frac(&L->op, k, L->lmax, last ? mg->coarse_frac : 0.1, L->dinv, r, z, work);
}

void orc_mg_vcycle(const orc_mg* mg, int l, const double* r, double* z)
{
    const orc_mg_level* L = &mg->lev[l];
    const int64_t n = L->op.n;
    double* work = (double*)malloc(sizeof(double) * (size_t)n * 7);
    if (l == mg->nlevels - 1) {
        mg_smooth(mg, L, mg->k_coarse, r, z, work);
        free(work);
        return;
    }
    double* res = work + 4 * n; double* Az = work + 5 * n; double* tmp = work + 6 * n;
    const int64_t nc = mg->lev[l + 1].op.n;
    double* rc = (double*)malloc(sizeof(double) * (size_t)nc * 2); double* ec = rc + nc;
    mg_smooth(mg, L, mg->k_smooth, r, z, work);                                     /* z = S r            */
    orc_apply_A(&L->op, z, Az, tmp);
    for (int64_t q = 0; q < n; ++q) res[q] = r[q] - Az[q];                          /* res = r - A z      */
    rnd32(res, n);
    orc_mg_restrict(mg, l, res, rc, tmp);
    orc_mg_vcycle(mg, l + 1, rc, ec);
    orc_mg_prolong(mg, l, ec, tmp);
    for (int64_t q = 0; q < n; ++q) z[q] += tmp[q];                                 /* z += P e           */
    rnd32(z, n);
    orc_apply_A(&L->op, z, Az, tmp);
    for (int64_t q = 0; q < n; ++q) res[q] = r[q] - Az[q];                          /* res = r - A z      */
    rnd32(res, n);
    mg_smooth(mg, L, mg->k_smooth, res, Az, work);                                  /* Az = S res         */
    for (int64_t q = 0; q < n; ++q) z[q] += Az[q];
    rnd32(z, n);
    free(rc); free(work);
}

/* z = V(0, r) with FP32 storage (R21): r is rounded on entry, every stored vector inside the cycle is rounded, the
 * level operators mg32 must have been built from float-rounded geometric factors, diagonals and multiplicities. */
void orc_mg_vcycle_fp32(const orc_mg* mg32, const double* r, double* z)
{
    const int64_t n = mg32->lev[0].op.n;
    double* r32 = (double*)malloc(sizeof(double) * (size_t)n);
    for (int64_t l = 0; l < n; ++l) r32[l] = (double)(float)r[l];
    g_r32 = 1;
    orc_mg_vcycle(mg32, 0, r32, z);
    g_r32 = 0;
    free(r32);
}

/* z = M^-1 r : precond 0 = identity, 1 = Jacobi, 2 = Chebyshev-Jacobi(cheb_k), 3 = p-multigrid V-cycle */
static void precond_apply(const orc_op* op, int precond, int cheb_k, double lmax, const double* dinv, const orc_mg* mg,
                          const double* r, double* z, double* work)
{
    if (precond == 0)      for (int64_t l = 0; l < op->n; ++l) z[l] = r[l];
    else if (precond == 1) for (int64_t l = 0; l < op->n; ++l) z[l] = dinv[l] * r[l];
    else if (precond == 2) orc_cheb_jacobi(op, cheb_k, lmax, dinv, r, z, work);
    else if (precond == 3) orc_mg_vcycle(mg, 0, r, z);
    else                   orc_mg_vcycle_fp32(mg, r, z);          /* precond 4: mg holds the float-rounded levels */
}

/* c-9  preconditioned conjugate gradients, step by step (the pressure Poisson solve).
 * b: assembled, masked rhs; x: initial guess in, solution out (continuous, zero at masked nodes).
 * hist[0..hist_len): ||r_it|| for it = 0,1,...  Returns 0 converged, 1 maxit reached,
 * -5 breakdown (gamma <= 0 or not finite).  out3 = { iterations, ||r0||, ||r_final|| }.   */
static int pcg_core(const orc_op* op, int precond, int cheb_k, double lmax, const double* dinv, const orc_mg* mg,
            const double* b, double* x, double rtol, double atol, int maxit, int x0_is_zero,
            double* hist, int hist_len, double* out3)
{
    const int64_t n = op->n;
    double* r = (double*)malloc(sizeof(double) * (size_t)n * 9);
    double* z = r + n; double* p = r + 2 * n; double* q = r + 3 * n; double* tmp = r + 4 * n; double* work = r + 5 * n;
    int status = 1, it = 0;
    if (x0_is_zero) { for (int64_t l = 0; l < n; ++l) { x[l] = 0.0; r[l] = b[l]; } }
    else { orc_apply_A(op, x, q, tmp); for (int64_t l = 0; l < n; ++l) r[l] = b[l] - q[l]; }
    const double bnorm = sqrt(orc_dot(op, b, b));
    double rnorm = sqrt(orc_dot(op, r, r));
    const double target = fmax(rtol * bnorm, atol);
    out3[1] = rnorm;
    if (hist_len > 0) hist[0] = rnorm;
    double rho_old = 0.0;
    for (int64_t l = 0; l < n; ++l) p[l] = 0.0;
    if (rnorm <= target) status = 0;
    else for (it = 1; it <= maxit; ++it) {
        precond_apply(op, precond, cheb_k, lmax, dinv, mg, r, z, work);
        double rho_new = orc_dot(op, r, z);
        double beta = (it == 1) ? 0.0 : rho_new / rho_old;
        for (int64_t l = 0; l < n; ++l) p[l] = z[l] + beta * p[l];
        orc_apply_A(op, p, q, tmp);
        double gamma = orc_dot(op, p, q);
        if (!(gamma > 0.0) || !isfinite(gamma)) { status = -5; break; }
        double alpha = rho_new / gamma;
        for (int64_t l = 0; l < n; ++l) { x[l] += alpha * p[l]; r[l] -= alpha * q[l]; }
        rho_old = rho_new;
        rnorm = sqrt(orc_dot(op, r, r));
        if (it < hist_len) hist[it] = rnorm;
        if (rnorm <= target) { status = 0; break; }
    }
    if (it > maxit) it = maxit;
    out3[0] = (double)it; out3[2] = rnorm;
    free(r);
    return status;
}

int orc_pcg(const orc_op* op, int precond, int cheb_k, double lmax, const double* dinv,
            const double* b, double* x, double rtol, double atol, int maxit, int x0_is_zero,
            double* hist, int hist_len, double* out3)
{
    if (precond < 0 || precond > 2) return -1;
    return pcg_core(op, precond, cheb_k, lmax, dinv, NULL, b, x, rtol, atol, maxit, x0_is_zero, hist, hist_len, out3);
}
/* PCG on level 0 of mg with the V-cycle as preconditioner (f-1) */
int orc_pcg_mg(const orc_mg* mg, const double* b, double* x, double rtol, double atol, int maxit, int x0_is_zero,
               double* hist, int hist_len, double* out3)
{
    return pcg_core(&mg->lev[0].op, 3, 0, 0.0, mg->lev[0].dinv, mg, b, x, rtol, atol, maxit, x0_is_zero, hist, hist_len, out3);
}
/* the same with the FP32-storage V-cycle (R21): the outer PCG runs on op64 (fp64 operator), the preconditioner on mg32 */
int orc_pcg_mg_fp32(const orc_op* op64, const orc_mg* mg32, const double* b, double* x, double rtol, double atol, int maxit,
                    int x0_is_zero, double* hist, int hist_len, double* out3)
{
    return pcg_core(op64, 4, 0, 0.0, NULL, mg32, b, x, rtol, atol, maxit, x0_is_zero, hist, hist_len, out3);
}

/* c-10  Lanczos on D^-1/2 A D^-1/2 from the start vector v0 (continuous, masked; normalised here).
 * Writes the tridiagonal (alpha[m], beta[m]); the caller takes its largest eigenvalue x 1.1. */
int orc_lanczos(const orc_op* op, const double* dinv, const double* v0, int m, double* alpha, double* beta)
{
    const int64_t n = op->n;
    double* v = (double*)malloc(sizeof(double) * (size_t)n * 5);
    double* vold = v + n; double* w = v + 2 * n; double* t = v + 3 * n; double* tmp = v + 4 * n;
    double nrm = sqrt(orc_dot(op, v0, v0));
    for (int64_t l = 0; l < n; ++l) { v[l] = v0[l] / nrm; vold[l] = 0.0; }
    double bprev = 0.0; int steps = 0;
    for (int j = 0; j < m; ++j) {
        for (int64_t l = 0; l < n; ++l) t[l] = sqrt(dinv[l]) * v[l];
        orc_apply_A(op, t, w, tmp);
        for (int64_t l = 0; l < n; ++l) w[l] = sqrt(dinv[l]) * w[l] - bprev * vold[l];
        alpha[j] = orc_dot(op, w, v);
        for (int64_t l = 0; l < n; ++l) w[l] -= alpha[j] * v[l];
        beta[j] = sqrt(orc_dot(op, w, w));
        steps = j + 1;
        if (!(beta[j] > 0.0)) break;
        for (int64_t l = 0; l < n; ++l) { vold[l] = v[l]; v[l] = w[l] / beta[j]; }
        bprev = beta[j];
    }
    free(v);
    return steps;
}

/* ------------------------------------------------------------------------------------ */
/* c-11  in-situ consumer (the consumer of the zero-copy hand-off).
 * min, max over the n values; bin = min(nbins-1, floor((v-lo)*scale)), scale = nbins/(hi-lo),
 * values outside [lo,hi] go to the end bins.                                              */
void orc_minmax_hist(int64_t n, const double* v, int nbins, double lo, double hi, double* minmax, uint64_t* hist)
{
    double mn = INFINITY, mx = -INFINITY;
    const double scale = (double)nbins / (hi - lo);
    for (int b = 0; b < nbins; ++b) hist[b] = 0;
    for (int64_t l = 0; l < n; ++l) {
        if (v[l] < mn) mn = v[l];
        if (v[l] > mx) mx = v[l];
        double t = v[l] - lo;
        double s = t * scale;
        int64_t b = (s < 0.0) ? 0 : (int64_t)floor(s);
        if (b > nbins - 1) b = nbins - 1;
        hist[b] += 1;
    }
    minmax[0] = mn; minmax[1] = mx;
}

/* velocity magnitude, sqrt(fma(vz,vz,fma(vy,vy,vx*vx))) (reading R11) */
void orc_vmag(int64_t n, const double* vx, const double* vy, const double* vz, double* out)
{
    for (int64_t l = 0; l < n; ++l) out[l] = sqrt(fma(vz[l], vz[l], fma(vy[l], vy[l], vx[l] * vx[l])));
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
