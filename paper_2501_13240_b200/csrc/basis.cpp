// GLL nodes, weights and derivative matrix on the host ("GLL quadrature", L100
// "(p+1)x(p+1) operator matrices ... identical for all elements").
//
// Nodes: roots of q(x) = P_{N+1}(x) - P_{N-1}(x) = (2N+1)/(N(N+1)) (x^2-1) P'_N(x), Newton with
// q'(x) = (2N+1) P_N(x), in long double, rounded once.  Weights rho_i = 2 / (N(N+1) P_N(xi_i)^2).
// D from barycentric weights, D_ij = (c_j / c_i) / (xi_i - xi_j), c_j = 1 / prod_{k != j}(xi_j - xi_k);
// the diagonal is minus the sum of the rounded off-diagonal row entries (reading R2), so that
// the operator annihilates constants to the rounding of the products only.
#include <cmath>

#include "semb_internal.h"

static void legendre3(int N, long double x, long double* Pm1, long double* P, long double* Pp1)
{
    long double p0 = 1.0L, p1 = x;          // P_0, P_1
    for (int n = 1; n < N; ++n) {           // -> p1 = P_N, p0 = P_{N-1}
        long double p2 = ((2 * n + 1) * x * p1 - n * p0) / (n + 1);
        p0 = p1; p1 = p2;
    }
    *Pm1 = p0; *P = p1;
    *Pp1 = ((2 * N + 1) * x * p1 - N * p0) / (N + 1);
}

void semb_basis_host(int N, double* xi, double* rho, double* D)
{
    const int n1 = N + 1;
    long double x[SEMB_MAXN1], w[SEMB_MAXN1];
    const long double pi = 3.141592653589793238462643383279502884L;
    x[0] = -1.0L; x[N] = 1.0L;
    for (int i = 1; i <= N / 2; ++i) {
        long double t = -cosl(pi * i / N);
        for (int it = 0; it < 60; ++it) {
            long double a, b, c;
            legendre3(N, t, &a, &b, &c);
            long double dt = (c - a) / ((2 * N + 1) * b);
            t -= dt;
            if (fabsl(dt) < 1e-20L) break;
        }
        x[i] = t; x[N - i] = -t;
    }
    if (N % 2 == 0) x[N / 2] = 0.0L;
    for (int i = 0; i < n1; ++i) {
        long double a, b, c;
        legendre3(N, x[i], &a, &b, &c);
        w[i] = 2.0L / (N * (N + 1.0L) * b * b);
    }
    if (xi)  for (int i = 0; i < n1; ++i) xi[i]  = (double)x[i];
    if (rho) for (int i = 0; i < n1; ++i) rho[i] = (double)w[i];
    if (!D) return;
    long double c[SEMB_MAXN1];
    for (int j = 0; j < n1; ++j) {
        long double p = 1.0L;
        for (int k = 0; k < n1; ++k) if (k != j) p *= (x[j] - x[k]);
        c[j] = 1.0L / p;
    }
    for (int i = 0; i < n1; ++i) {
        long double s = 0.0L;
        for (int j = 0; j < n1; ++j) {
            if (j == i) continue;
            double d = (double)((c[j] / c[i]) / (x[i] - x[j]));
            D[i * n1 + j] = d;
            s += d;
        }
        D[i * n1 + i] = (double)(-s);
    }
}
