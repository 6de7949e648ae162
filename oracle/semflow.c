/*
 * semflow.c -- CPU oracle of the operators that the Boussinesq time step needs besides the Helmholtz / Poisson solves
 * (Eqs. (1)-(3): du/dt + u.grad u = -grad p + T z^ + sqrt(Pr/Ra) lap u,
 * dT/dt + u.grad T = lap T / sqrt(Ra Pr), div u = 0).  The paper states the equations only; the discrete step is
 * DESIGN.md reading R25 and is assembled from these pieces in oracle/boussinesq.py.
 *
 * TEST INFRASTRUCTURE ONLY.  Plain C, fp64, the definitions written out; shares no code with csrc/.
 * Pins (tests/test_oracle_flow.py): closed-form metrics of a sheared affine mesh, exact gradients of polynomials, analytic integrals for
 * the weak divergence, grad(linear) exact on curved meshes, wdiv = grad^T, QQ^T wdiv o grad = A.  Parity unpinned: none.
 *
 *   metrics   J = d(x,y,z)/d(r,s,t) by applying D to the coordinates (as c-3); met[e][9][Np] = dr_a/dx_b,
 *             a = r,s,t (rows), b = x,y,z: the inverse of J, entry (a,b) at index 3a + b.
 *   grad      collocation gradient of a nodal field, element by element (discontinuous across elements):
 *             dphi/dx_b = sum_a (dr_a/dx_b) dphi/dr_a,  dphi/dr = sum_m D_im phi(m,j,k), ...
 *   wdiv      weak divergence (the transpose of grad in the GLL inner product), per element, unassembled:
 *             out_i = int grad(phi_i) . g = sum_a sum_m D_mi [ B (dr_a/dx . g) ](m, ...)     (B = W J from c-3)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#define IDX(i, j, k) ((k) * n1 * n1 + (j) * n1 + (i))

/* returns -1, or the first element with a non-positive Jacobian */
int64_t orc_metrics(int64_t E, int N, const double* x, const double* y, const double* z, const double* D, double* met)
{
    const int n1 = N + 1, Np = n1 * n1 * n1;
    int64_t bad = -1;
    for (int64_t e = 0; e < E; ++e) {
        const double *X = x + e * Np, *Y = y + e * Np, *Z = z + e * Np;
        double* m = met + e * 9 * (int64_t)Np;
        for (int k = 0; k < n1; ++k) for (int j = 0; j < n1; ++j) for (int i = 0; i < n1; ++i) {
            double xr = 0, xs = 0, xt = 0, yr = 0, ys = 0, yt = 0, zr = 0, zs = 0, zt = 0;
            for (int q = 0; q < n1; ++q) {
                xr += D[i * n1 + q] * X[IDX(q, j, k)]; xs += D[j * n1 + q] * X[IDX(i, q, k)]; xt += D[k * n1 + q] * X[IDX(i, j, q)];
                yr += D[i * n1 + q] * Y[IDX(q, j, k)]; ys += D[j * n1 + q] * Y[IDX(i, q, k)]; yt += D[k * n1 + q] * Y[IDX(i, j, q)];
                zr += D[i * n1 + q] * Z[IDX(q, j, k)]; zs += D[j * n1 + q] * Z[IDX(i, q, k)]; zt += D[k * n1 + q] * Z[IDX(i, j, q)];
            }
            const double J = xr * (ys * zt - yt * zs) - xs * (yr * zt - yt * zr) + xt * (yr * zs - ys * zr);
            if (!(J > 0.0) && bad < 0) bad = e;
            const int l = IDX(i, j, k);
            m[0 * Np + l] = (ys * zt - yt * zs) / J;  m[1 * Np + l] = -(xs * zt - xt * zs) / J; m[2 * Np + l] = (xs * yt - xt * ys) / J;
            m[3 * Np + l] = -(yr * zt - yt * zr) / J; m[4 * Np + l] = (xr * zt - xt * zr) / J;  m[5 * Np + l] = -(xr * yt - xt * yr) / J;
            m[6 * Np + l] = (yr * zs - ys * zr) / J;  m[7 * Np + l] = -(xr * zs - xs * zr) / J; m[8 * Np + l] = (xr * ys - xs * yr) / J;
        }
    }
    return bad;
}

void orc_grad(int64_t E, int N, const double* met, const double* D, const double* phi, double* gx, double* gy, double* gz)
{
    const int n1 = N + 1, Np = n1 * n1 * n1;
    for (int64_t e = 0; e < E; ++e) {
        const double* p = phi + e * Np; const double* m = met + e * 9 * (int64_t)Np;
        for (int k = 0; k < n1; ++k) for (int j = 0; j < n1; ++j) for (int i = 0; i < n1; ++i) {
            double pr = 0, ps = 0, pt = 0;
            for (int q = 0; q < n1; ++q) { pr += D[i * n1 + q] * p[IDX(q, j, k)]; ps += D[j * n1 + q] * p[IDX(i, q, k)]; pt += D[k * n1 + q] * p[IDX(i, j, q)]; }
            const int l = IDX(i, j, k);
            gx[e * Np + l] = m[0 * Np + l] * pr + m[3 * Np + l] * ps + m[6 * Np + l] * pt;
            gy[e * Np + l] = m[1 * Np + l] * pr + m[4 * Np + l] * ps + m[7 * Np + l] * pt;
            gz[e * Np + l] = m[2 * Np + l] * pr + m[5 * Np + l] * ps + m[8 * Np + l] * pt;
        }
    }
}

/* Bm [E][Np]: the mass factor W J (geo factor 7 of c-3) */
void orc_wdiv(int64_t E, int N, const double* met, const double* Bm, const double* D, const double* gx, const double* gy, const double* gz, double* out)
{
    const int n1 = N + 1, Np = n1 * n1 * n1;
    double* fr = (double*)malloc(sizeof(double) * 3 * (size_t)Np);
    double *fs = fr + Np, *ft = fs + Np;
    for (int64_t e = 0; e < E; ++e) {
        const double* m = met + e * 9 * (int64_t)Np;
        for (int l = 0; l < Np; ++l) {
            const double a = gx[e * Np + l], b = gy[e * Np + l], c = gz[e * Np + l], B = Bm[e * Np + l];
            fr[l] = B * (m[0 * Np + l] * a + m[1 * Np + l] * b + m[2 * Np + l] * c);
            fs[l] = B * (m[3 * Np + l] * a + m[4 * Np + l] * b + m[5 * Np + l] * c);
            ft[l] = B * (m[6 * Np + l] * a + m[7 * Np + l] * b + m[8 * Np + l] * c);
        }
        for (int k = 0; k < n1; ++k) for (int j = 0; j < n1; ++j) for (int i = 0; i < n1; ++i) {
            double s = 0.0;
            for (int q = 0; q < n1; ++q) s += D[q * n1 + i] * fr[IDX(q, j, k)] + D[q * n1 + j] * fs[IDX(i, q, k)] + D[q * n1 + k] * ft[IDX(i, j, q)];
            out[e * Np + IDX(i, j, k)] = s;
        }
    }
    free(fr);
}
