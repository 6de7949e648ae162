"""Pins P1-P3, P16 of SURVEY.md §8(c): GLL rule, derivative matrix, geometric factors.

Every expected value here is a closed form, a textbook identity, or comes from an independent
library routine (numpy.polynomial.legendre) -- never from the oracle itself or the CUDA path.
"""
import numpy as np
import pytest
from numpy.polynomial import legendre as L

from paper_2501_13240_b200 import inputs as I


# ---------------------------------------------------------------- P1: GLL nodes and weights (c-1)
def test_gll_closed_forms(orc):
    xi, rho = orc.gll(1)
    assert np.array_equal(xi, [-1, 1]) and np.allclose(rho, [1, 1], rtol=0, atol=1e-15)
    xi, rho = orc.gll(2)
    assert np.array_equal(xi, [-1, 0, 1]) and np.allclose(rho, [1 / 3, 4 / 3, 1 / 3], rtol=0, atol=1e-15)
    xi, rho = orc.gll(3)
    assert np.allclose(xi, [-1, -1 / np.sqrt(5), 1 / np.sqrt(5), 1], rtol=0, atol=1e-15)
    assert np.allclose(rho, [1 / 6, 5 / 6, 5 / 6, 1 / 6], rtol=0, atol=1e-15)
    xi, rho = orc.gll(4)   # +-sqrt(3/7), weights 1/10, 49/90, 32/45
    assert np.allclose(xi, [-1, -np.sqrt(3 / 7), 0, np.sqrt(3 / 7), 1], atol=1e-15)
    assert np.allclose(rho, [0.1, 49 / 90, 32 / 45, 49 / 90, 0.1], atol=1e-15)


@pytest.mark.parametrize("N", range(1, 11))
def test_gll_against_numpy_legendre(orc, N):
    """interior nodes are the roots of P'_N (library root finder); rho_i = 2/(N(N+1)P_N(xi_i)^2)."""
    xi, rho = orc.gll(N)
    PN = L.Legendre.basis(N)
    roots = np.sort(np.real(PN.deriv().roots())) if N > 1 else np.array([])
    assert np.allclose(xi[1:-1], roots, rtol=0, atol=2e-14)
    assert np.allclose(rho, 2.0 / (N * (N + 1) * PN(xi) ** 2), rtol=1e-13)
    assert abs(rho.sum() - 2.0) < 1e-14
    assert np.array_equal(xi, -xi[::-1]) and np.array_equal(rho, rho[::-1])
    # exact for monomials up to degree 2N-1, inexact at 2N
    for k in range(0, 2 * N):
        exact = 2.0 / (k + 1) if k % 2 == 0 else 0.0
        assert abs(np.dot(rho, xi ** k) - exact) < 1e-14
    assert abs(np.dot(rho, xi ** (2 * N)) - 2.0 / (2 * N + 1)) > 1e-6 / N ** 3


# ---------------------------------------------------------------- P2: derivative matrix (c-2)
def test_dhat_closed_forms(orc):
    assert np.allclose(orc.dhat(1), [[-0.5, 0.5], [-0.5, 0.5]], atol=1e-15)
    assert np.allclose(orc.dhat(2), [[-1.5, 2, -0.5], [-0.5, 0, 0.5], [0.5, -2, 1.5]], atol=1e-15)


@pytest.mark.parametrize("N", range(1, 11))
def test_dhat_properties(orc, N):
    xi, _ = orc.gll(N)
    D = orc.dhat(N)
    assert abs(D[0, 0] + N * (N + 1) / 4) < 1e-12 and abs(D[N, N] - N * (N + 1) / 4) < 1e-12
    for i in range(1, N):
        assert abs(D[i, i]) < 1e-12                       # interior diagonal entries vanish
    for k in range(0, N + 1):                             # differentiates polynomials of degree <= N exactly
        d = k * xi ** (k - 1) if k > 0 else np.zeros(N + 1)
        assert np.allclose(D @ xi ** k, d, rtol=0, atol=5e-12)
    assert np.allclose(D[::-1, ::-1], -D, rtol=0, atol=1e-12)       # centro-antisymmetry
    # D[i,j] = l_j'(xi_i) from the library's Lagrange interpolant through the nodes
    for j in range(N + 1):
        c = np.zeros(N + 1); c[j] = 1.0
        lj = np.polynomial.polynomial.Polynomial.fit(xi, c, N, domain=[-1, 1], window=[-1, 1])
        assert np.allclose(D[:, j], lj.deriv()(xi), rtol=0, atol=2e-9 * (1 + N) ** 2)


# ---------------------------------------------------------------- P3 / P16: geometric factors (c-3)
def _one_element(N, xi, A, b):
    """nodes of the affine image x = A [r,s,t]^T + b of the reference cube, (k,j,i) i-fastest."""
    r = xi[None, None, :] + 0 * xi[:, None, None] + 0 * xi[None, :, None]
    s = xi[None, :, None] + 0 * r
    t = xi[:, None, None] + 0 * r
    R = np.stack([r.ravel(), s.ravel(), t.ravel()])
    X = A @ R + np.asarray(b)[:, None]
    return X[0].copy(), X[1].copy(), X[2].copy()


def test_geo_affine_brick(orc):
    N = 5
    xi, rho = orc.gll(N)
    hx, hy, hz = 0.7, 1.3, 0.4
    x, y, z = _one_element(N, xi, np.diag([hx / 2, hy / 2, hz / 2]), [1, 2, 3])
    g = orc.geo_factors(1, N, x, y, z)[0]
    W = (rho[:, None, None] * rho[None, :, None] * rho[None, None, :]).ravel()
    assert np.allclose(g[6], W * hx * hy * hz / 8, rtol=1e-13)
    assert np.allclose(g[0], W * hy * hz / (2 * hx), rtol=1e-13)
    assert np.allclose(g[3], W * hx * hz / (2 * hy), rtol=1e-13)
    assert np.allclose(g[5], W * hx * hy / (2 * hz), rtol=1e-13)
    for c in (1, 2, 4):
        assert np.abs(g[c]).max() < 1e-14
    assert abs(g[6].sum() - hx * hy * hz) < 1e-14


def test_geo_general_affine_map(orc):
    """x = A xi: G = W det(A) A^-1 A^-T (all six entries, catches sign/transposition slips)."""
    N = 4
    xi, rho = orc.gll(N)
    A = np.array([[1.0, 0.3, -0.2], [0.1, 0.8, 0.25], [-0.15, 0.2, 1.1]])
    assert np.linalg.det(A) > 0
    x, y, z = _one_element(N, xi, A, [0, 0, 0])
    g = orc.geo_factors(1, N, x, y, z)[0]
    W = (rho[:, None, None] * rho[None, :, None] * rho[None, None, :]).ravel()
    Ai = np.linalg.inv(A)
    M = np.linalg.det(A) * Ai @ Ai.T
    for idx, (a, b) in enumerate([(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]):
        assert np.allclose(g[idx], W * M[a, b], rtol=0, atol=1e-13), idx
    assert np.allclose(g[6], W * np.linalg.det(A), rtol=1e-13)


def test_geo_negative_jacobian_rejected(orc):
    N = 3
    xi, _ = orc.gll(N)
    x, y, z = _one_element(N, xi, np.diag([-1.0, 1.0, 1.0]), [0, 0, 0])
    with pytest.raises(ValueError):
        orc.geo_factors(1, N, x, y, z)


def test_volume_sums(orc, xi_of):
    m = I.box_mesh(3, 3, 3, 5, xi_of(5), deform=0.05)                 # deformation vanishes on the boundary
    assert abs(orc.geo_factors(m.E, m.N, m.x, m.y, m.z)[:, 6].sum() - 1.0) < 1e-13
    m = I.ogrid_mesh(4, 3, 3, 7, xi_of(7))                            # isoparametric cylinder, R = 0.5, H = 1
    assert abs(orc.geo_factors(m.E, m.N, m.x, m.y, m.z)[:, 6].sum() - np.pi / 4) < 1e-12
    m = I.box_mesh(2, 2, 4, 4, xi_of(4), zstretch=2.5)
    assert abs(orc.geo_factors(m.E, m.N, m.x, m.y, m.z)[:, 6].sum() - 1.0) < 1e-14


def test_table4_gridpoints_golden():
    """PAPER.md:L268, L274-285 (Table 4): gridpoints = N_e p^3 as printed; unique nodes of a periodic-xy box."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "table4_gridpoints.txt")
    rows = [l.split() for l in open(path) if not l.startswith("#") and l.strip()]
    assert len(rows) == 8
    for _, nx, ny, nz, p, printed, tol in rows:
        nx, ny, nz, p = int(nx), int(ny), int(nz), int(p)
        ne_p3 = nx * ny * nz * p ** 3
        assert abs(ne_p3 / 1e6 - float(printed)) <= float(tol)
        unique = (nx * p) * (ny * p) * (nz * p + 1)
        assert unique * nz * p == ne_p3 * (nz * p + 1)
