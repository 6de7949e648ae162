"""Pins of the Schwarz smoother of the oracle (oracle/schwarz.py; reading R26):
on tensor-product box meshes the fast-diagonalisation subdomain solve is the EXACT inverse of the assembled operator
restricted to the element's nodes (dense numpy inverse), the smoother is symmetric positive semi-definite, the fourth-kind
Chebyshev acceleration follows its closed-form polynomial, and the V-cycle with it needs fewer PCG iterations than with
Jacobi smoothing on the boundary-layer-stretched O-grid (the reason the paper uses it)."""
import numpy as np
import pytest

from paper_2501_13240_b200 import inputs as I
from test_oracle_operator import dense_matrix, make, to_global, to_local


@pytest.mark.parametrize("lam,tags,periodic", [(0.0, 0b10, (True, True, False)), (40.0, 0b110, (False, False, False)), (0.0, 0b10, (False, False, False))])
def test_subdomain_solve_is_the_exact_restricted_inverse_on_tensor_boxes(orc, xi_of, lam, tags, periodic):
    from oracle import schwarz as Sz
    N = 3
    m = I.box_mesh(3, 3, 3, N, xi_of(N), periodic=periodic, zstretch=1.8)       # non-uniform in z: lengths differ between neighbours
    P = make(orc, m, lam=lam, tags=tags)
    S = Sz.Schwarz(P, m.x, m.y, m.z)
    A = dense_matrix(P)
    free_g = to_global(P, P.mask) > 0
    rng = np.random.default_rng(3)
    Np = P.Np
    for e in (0, 4, 13, 22, 26):                                                  # corner, edge, centre and top-layer elements
        gids = P.gid[e * Np:(e + 1) * Np]
        assert np.unique(gids).size == Np                                         # 3 elements per periodic direction: no self-overlap
        v = rng.standard_normal(Np)
        fr = free_g[gids]
        v[~fr] = 0.0
        vloc = np.zeros(P.n); vloc[e * Np:(e + 1) * Np] = v
        got = S.local_solve(vloc)[e * Np:(e + 1) * Np]
        sub = gids[fr]
        expect = np.zeros(Np)
        expect[fr] = np.linalg.solve(A[np.ix_(sub, sub)], v[fr])
        assert np.abs(got - expect).max() <= 1e-11 * np.abs(expect).max(), (e, np.abs(got - expect).max())
        assert np.all(got[~fr] == 0.0)


def test_smoother_is_symmetric_positive_and_reduces_the_residual(orc, xi_of):
    from oracle import schwarz as Sz
    N = 3
    m = I.ogrid_mesh(2, 2, 3, N, xi_of(N))
    P = make(orc, m, tags=0b10)
    S = Sz.Schwarz(P, m.x, m.y, m.z)
    free = to_global(P, P.mask) > 0
    nu = P.n_unique
    Sd = np.zeros((nu, nu))
    for g in np.where(free)[0]:
        e = np.zeros(nu); e[g] = 1.0
        Sd[:, g] = to_global(P, S.apply(to_local(P, e)))
    Sf = Sd[np.ix_(free, free)]
    assert np.abs(Sf - Sf.T).max() <= 1e-12 * np.abs(Sf).max()
    ev = np.linalg.eigvalsh(0.5 * (Sf + Sf.T))
    assert ev[0] > 0.0
    assert np.all(Sd[~free] == 0) and np.all(Sd[:, ~free] == 0)
    # spectrum of S A: what the Lanczos estimate must bound, and far better conditioned than D^-1 A
    Af = dense_matrix(P)[np.ix_(free, free)]
    L = np.linalg.cholesky(Sf)
    sa = np.linalg.eigvalsh(L.T @ Af @ L)
    v0 = P.mask * orc.gs(P.gid, P.n_unique, I.uniform(3, P.n))
    lmax = Sz.lanczos_lmax(P, S, v0, 10)
    assert sa[-1] <= lmax <= 1.3 * sa[-1]
    da = np.linalg.eigvalsh(Af / np.sqrt(np.outer(np.diag(Af), np.diag(Af))))
    assert sa[-1] / sa[0] < 0.5 * da[-1] / da[0]


@pytest.mark.parametrize("k", [1, 2, 3])
def test_fourth_kind_chebyshev_schwarz_closed_form(orc, xi_of, k):
    """z = p_k(S A) S r with 1 - lam p_k(lam) = W_(k+1)(1 - 2 lam / lmax) / (2k + 3) on the dense spectrum of S^1/2 A S^1/2"""
    from oracle import schwarz as Sz
    N = 2
    m = I.box_mesh(2, 2, 2, N, xi_of(N), deform=0.05)
    P = make(orc, m, tags=0b10)
    S = Sz.Schwarz(P, m.x, m.y, m.z)
    free = to_global(P, P.mask) > 0
    nu = P.n_unique
    Sd = np.zeros((nu, nu))
    for g in np.where(free)[0]:
        e = np.zeros(nu); e[g] = 1.0
        Sd[:, g] = to_global(P, S.apply(to_local(P, e)))
    Sf = Sd[np.ix_(free, free)]; Sf = 0.5 * (Sf + Sf.T)
    Af = dense_matrix(P)[np.ix_(free, free)]
    L = np.linalg.cholesky(Sf)
    ev, V = np.linalg.eigh(L.T @ Af @ L)
    lmax = 1.07 * ev[-1]
    t = np.arccos(1.0 - 2.0 * ev / lmax)
    n = k + 1
    pk = (1.0 - np.sin((n + 0.5) * t) / np.sin(0.5 * t) / (2 * n + 1)) / ev
    rg = np.zeros(nu); rg[free] = np.random.default_rng(8).standard_normal(free.sum())
    z = Sz.cheb4(P, S, k, lmax, to_local(P, rg))
    expect = L @ ((V * pk) @ (V.T @ (L.T @ rg[free])))
    assert np.allclose(to_global(P, z)[free], expect, rtol=0, atol=1e-11 * np.abs(expect).max())


def test_schwarz_vcycle_beats_jacobi_smoothing_on_the_stretched_ogrid(orc, xi_of):
    from oracle import schwarz as Sz
    m, _ = I.config_mesh(2, xi_of, small=True)                                  # O-grid (4, 3, 4), N = 7, tanh-clustered layers
    mg = orc.Multigrid(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, 0.0, 0b10, [7, 3, 1], k_smooth=1, k_coarse=32, kind=4, coarse_frac=0.01)
    P = mg.levels[0]
    b = P.assemble_rhs(I.divergence_source(m, 5))
    rj = mg.pcg(b)
    ms = Sz.MultigridSchwarz(mg, k_smooth=1)
    rs = ms.pcg(b)
    res = b - P.apply_A(rs["x"])
    assert np.sqrt(P.dot(res, res)) <= 2e-10 * np.sqrt(P.dot(b, b))
    assert np.abs(rs["x"] - rj["x"]).max() <= 1e-8 * np.abs(rj["x"]).max()
    print("iterations: Chebyshev-Jacobi smoothing", rj["iters"], " Chebyshev-Schwarz smoothing", rs["iters"])
    assert rs["iters"] <= 0.7 * rj["iters"], (rs["iters"], rj["iters"])
