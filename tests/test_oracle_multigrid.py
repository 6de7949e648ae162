"""Pins of the p-multigrid V-cycle preconditioner of the oracle (reading R19).

Expected values never come from the oracle's own multigrid code: interpolation matrices are rebuilt from monomial
Vandermonde systems, the 3-D transfer from numpy.kron, the global prolongation from the numbering, the smoother
from the closed-form Chebyshev residual polynomial through a dense eigendecomposition, and the V-cycle from the
textbook error-propagation product  I - B A = (I - S A)(I - P B_c P^T A)(I - S A)  in dense algebra.
"""
import numpy as np
import pytest
from numpy.polynomial import chebyshev as Ch

from paper_2501_13240_b200 import inputs as I
from test_oracle_operator import dense_matrix, make, to_global, to_local


def vandermonde_interp(x_from, x_to):
    """Lagrange interpolation matrix through monomials: J = V(x_to) V(x_from)^-1 (independent of the product formula)."""
    n = len(x_from)
    return np.vander(x_to, n, increasing=True) @ np.linalg.inv(np.vander(x_from, n, increasing=True))


def test_interp_matrix_closed_forms(orc):
    J = orc.interp_matrix(1, 2)                                    # linear basis at -1, 0, 1
    assert np.array_equal(J, np.array([[1.0, 0.0], [0.5, 0.5], [0.0, 1.0]]))
    for Nc, Nf in [(1, 3), (3, 7), (1, 7), (5, 9), (2, 4), (7, 3), (9, 5)]:      # both directions (coordinates go fine -> coarse)
        xc, xf = orc.gll(Nc)[0], orc.gll(Nf)[0]
        J = orc.interp_matrix(Nc, Nf)
        assert J.shape == (Nf + 1, Nc + 1)
        assert np.allclose(J, vandermonde_interp(xc, xf), rtol=0, atol=1e-12)
        assert np.allclose(J.sum(axis=1), 1.0, rtol=0, atol=1e-14)                 # partition of unity
        for p in range(Nc + 1):                                                    # exact for degree <= N_from
            assert np.allclose(J @ xc ** p, xf ** p, rtol=0, atol=1e-13)
        assert np.array_equal(J[0], np.eye(Nc + 1)[0]) and np.array_equal(J[-1], np.eye(Nc + 1)[-1])   # end nodes coincide


def test_interp3_is_the_kronecker_product(orc):
    J = orc.interp_matrix(2, 4)
    E = 3
    v = I.uniform(3, E * 27)
    K = np.kron(J, np.kron(J, J))                                   # (k,j,i) ordering, i fastest
    out = orc.interp3(E, J, v)
    assert np.allclose(out.reshape(E, -1), v.reshape(E, -1) @ K.T, rtol=0, atol=1e-14)
    w = I.uniform(4, E * 125)
    outT = orc.interp3(E, J, w, transpose=True)
    assert np.allclose(outT.reshape(E, -1), w.reshape(E, -1) @ K, rtol=0, atol=1e-13)


def _mg(orc, m, lam, tags, orders, k=2, kc=2, lmax=None, kind=1, frac=0.1):
    return orc.Multigrid(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam, tags, orders, k_smooth=k, k_coarse=kc, lmax=lmax,
                         kind=kind, coarse_frac=frac)


def _cont(orc, P, seed):
    """continuous, masked random vector on the level problem P"""
    return P.mask * orc.gs(P.gid, P.n_unique, P.invmult * I.uniform(seed, P.n))


@pytest.mark.parametrize("kind", ["box", "ogrid"])
def test_transfer_continuity_mask_and_adjointness(orc, xi_of, kind):
    N = 4
    m = I.box_mesh(3, 2, 2, N, xi_of(N), deform=0.05, periodic=(True, False, False)) if kind == "box" \
        else I.ogrid_mesh(2, 2, 2, N, xi_of(N))
    mg = _mg(orc, m, 0.0, 0b10, [4, 2, 1], lmax=[1.0, 1.0, 1.0])
    for l in range(2):
        Pf, Pc = mg.levels[l], mg.levels[l + 1]
        # coarse coordinates are the fine interpolant at the coarse nodes: the coarse mesh has the same volume
        vc = _cont(orc, Pc, 11 + l)
        vf = mg.prolong(l, vc)
        assert np.allclose(orc.gs(Pf.gid, Pf.n_unique, vf * Pf.invmult), vf, rtol=0, atol=1e-14)    # continuous
        assert np.all(vf[Pf.mask == 0] == 0)
        rf = _cont(orc, Pf, 21 + l)
        rc = mg.restrict(l, rf)
        assert np.allclose(orc.gs(Pc.gid, Pc.n_unique, rc * Pc.invmult), rc, rtol=0, atol=1e-13)
        assert np.all(rc[Pc.mask == 0] == 0)
        lhs, rhs = Pf.dot(vf, rf), Pc.dot(vc, rc)                   # <P v, r>_f = <v, R r>_c on unique nodes
        assert abs(lhs - rhs) <= 1e-13 * max(abs(lhs), 1.0)
    # prolongation reproduces a field of degree <= N_c exactly: the coordinate x of an affine mesh (degree 1)
    if kind == "box":
        ma = I.box_mesh(3, 2, 2, N, xi_of(N))
        mga = _mg(orc, ma, 0.0, 0, [4, 2, 1], lmax=[1.0, 1.0, 1.0])
        for l in range(2):
            for c in range(3):
                assert np.allclose(orc.interp3(ma.E, mga.J[l], mga.coords[l + 1][c]), mga.coords[l][c], rtol=0, atol=1e-13)


def _global_prolongation(orc, Pf, Pc, Nf, Nc):
    """dense [n_unique_f, n_unique_c] from numpy's own interpolation matrix and the two numberings"""
    J = vandermonde_interp(orc.gll(Nc)[0], orc.gll(Nf)[0])
    K = np.kron(J, np.kron(J, J))
    Pg = np.zeros((Pf.n_unique, Pc.n_unique))
    gf = Pf.gid.reshape(Pf.E, -1); gc = Pc.gid.reshape(Pc.E, -1)
    for e in range(Pf.E):
        Pg[gf[e][:, None], gc[e][None, :]] = K                      # every copy of a fine node gives the same row
    return Pg


def _cheb_dense(Af, k, lmax, frac=0.1):
    Dm = np.diag(Af)
    ev, V = np.linalg.eigh(Af / np.sqrt(np.outer(Dm, Dm)))
    lmin = frac * lmax; theta = 0.5 * (lmax + lmin); delta = 0.5 * (lmax - lmin); sigma = theta / delta
    Tk1 = Ch.Chebyshev.basis(k + 1)
    pk = (1.0 - Tk1((theta - ev) / delta) / Tk1(sigma)) / ev
    return ((V * pk) @ V.T) / np.sqrt(np.outer(Dm, Dm))


@pytest.mark.parametrize("lam,tags,kc,frac", [(0.0, 0b10, 3, 0.1), (50.0, 0, 3, 0.1), (0.0, 0b10, 7, 0.02)])
def test_vcycle_equals_dense_composition_and_is_spd(orc, xi_of, lam, tags, kc, frac):
    N = 4
    m = I.box_mesh(2, 2, 2, N, xi_of(N), deform=0.05)
    orders = [4, 2, 1]
    mg0 = _mg(orc, m, lam, tags, orders, lmax=[1.0, 1.0, 1.0])
    A, free, lmax = [], [], []
    for P in mg0.levels:
        Ad = dense_matrix(P); fr = to_global(P, P.mask) > 0
        A.append(Ad[np.ix_(fr, fr)]); free.append(fr)
        Dm = np.diag(A[-1])
        lmax.append(1.1 * np.linalg.eigvalsh(A[-1] / np.sqrt(np.outer(Dm, Dm)))[-1])
    k = 2
    mg = _mg(orc, m, lam, tags, orders, k=k, kc=kc, lmax=lmax, frac=frac)
    B = _cheb_dense(A[2], kc, lmax[2], frac)                       # last level: interval [frac, 1] lmax
    for l in (1, 0):
        Pg = _global_prolongation(orc, mg.levels[l], mg.levels[l + 1], orders[l], orders[l + 1])[np.ix_(free[l], free[l + 1])]
        S = _cheb_dense(A[l], k, lmax[l]); Id = np.eye(A[l].shape[0])
        B = S + (Id - S @ A[l]) @ (S + Pg @ B @ Pg.T @ (Id - A[l] @ S))
    P0 = mg.levels[0]
    nf = int(free[0].sum())
    Bo = np.zeros((nf, nf))
    idx = np.flatnonzero(free[0])
    for c, g in enumerate(idx):
        e = np.zeros(P0.n_unique); e[g] = 1.0
        z = mg.vcycle(to_local(P0, e))
        assert np.all(z[P0.mask == 0] == 0)
        Bo[:, c] = to_global(P0, z)[free[0]]
    scale = np.abs(B).max()
    assert np.abs(Bo - B).max() <= 1e-11 * scale
    assert np.abs(Bo - Bo.T).max() <= 1e-12 * scale                 # symmetric
    assert np.linalg.eigvalsh(0.5 * (Bo + Bo.T))[0] > 0             # positive definite
    ev = np.linalg.eigvals(Bo @ A[0]).real
    # spectrum of M^-1 A: clustered below 1; it may exceed 1 slightly because the coarse operators are
    # re-discretisations, not Galerkin products (measured here: [0.85, 1.004])
    assert ev.min() > 0.3 and ev.max() < 1.2
    # the restriction alone: R = P^T on the free unique nodes
    rf = _cont(orc, P0, 9)
    rc = mg.restrict(0, rf)
    Pg = _global_prolongation(orc, mg.levels[0], mg.levels[1], orders[0], orders[1])[np.ix_(free[0], free[1])]
    assert np.allclose(to_global(mg.levels[1], rc)[free[1]], Pg.T @ to_global(P0, rf)[free[0]], rtol=0, atol=1e-13)


def test_pmg_pcg_solves_and_beats_chebyshev_jacobi(orc, xi_of):
    m, _ = I.config_mesh(2, xi_of, small=True)                      # reduced O-grid, N = 7
    mg = _mg(orc, m, 0.0, 0b10, [7, 3, 1], k=2, kc=4)
    P = mg.levels[0]
    b = P.assemble_rhs(I.divergence_source(m, 5))
    rm = mg.pcg(b, rtol=1e-10, hist_len=200)
    rj = P.pcg(b, precond=1)
    rc = P.pcg(b, precond=2, cheb_k=2, lmax=mg.lmax[0])
    assert rm["status"] == 0 and rj["status"] == 0
    assert rm["iters"] < 0.5 * rc["iters"] < 0.5 * rj["iters"]
    assert np.abs(rm["x"] - rj["x"]).max() <= 1e-8 * np.abs(rj["x"]).max()
    res = b - P.apply_A(rm["x"])
    assert np.sqrt(P.dot(res, res)) <= 2e-10 * np.sqrt(P.dot(b, b))
    assert np.all(np.diff(rm["hist"]) < 0) or rm["iters"] < 40     # residuals fall fast
    # Helmholtz with a large shift: the V-cycle must still be SPD (PCG converges) and cheap in iterations
    mgh = _mg(orc, m, 3000.0, 0b110, [7, 3, 1], k=2, kc=4)
    bh = mgh.levels[0].assemble_rhs(I.divergence_source(m, 6))
    rh = mgh.pcg(bh)
    assert rh["status"] == 0 and rh["iters"] <= mgh.levels[0].pcg(bh, precond=1)["iters"]


def test_estimated_bounds_cover_the_spectrum(orc, xi_of):
    """The per-level Chebyshev bound (1.1 x Lanczos-10 from the seeded rough vector) must lie above the true
    lambda_max(D^-1 A) of its level -- below it the smoother amplifies the top modes and the V-cycle is indefinite."""
    N = 4
    m = I.box_mesh(3, 3, 3, N, xi_of(N), deform=0.05)
    mg = _mg(orc, m, 0.0, 0b10, [4, 2, 1])
    for P, lm in zip(mg.levels, mg.lmax):
        Ad = dense_matrix(P); fr = to_global(P, P.mask) > 0
        Af = Ad[np.ix_(fr, fr)]; Dm = np.diag(Af)
        true = np.linalg.eigvalsh(Af / np.sqrt(np.outer(Dm, Dm)))[-1]
        assert true <= lm <= 1.35 * true, (true, lm)
    # the generator restated in the oracle is the recipe's (paper_2501_13240_b200/inputs.py)
    assert np.array_equal(orc._splitmix_uniform(orc.MG_LMAX_SEED, 1000), I.uniform(orc.MG_LMAX_SEED, 1000))


@pytest.mark.parametrize("k", [0, 1, 2, 4])
def test_fourth_kind_chebyshev_closed_form(orc, xi_of, k):
    """z = p_k(D^-1 A) D^-1 r with 1 - lam p_k(lam) = W_{k+1}(1 - 2 lam/lmax) / (2k + 3), W_n(cos t) = sin((n + 1/2) t) / sin(t/2)
    the Chebyshev polynomial of the fourth kind -- evaluated here through its trigonometric form on a dense spectrum."""
    N = 3
    m = I.ogrid_mesh(2, 2, 2, N, xi_of(N))
    P = make(orc, m, tags=0b10)
    A = dense_matrix(P); free = to_global(P, P.mask) > 0
    Af = A[np.ix_(free, free)]; Dm = np.diag(Af)
    ev, V = np.linalg.eigh(Af / np.sqrt(np.outer(Dm, Dm)))
    lmax = 1.07 * ev[-1]
    t = np.arccos(1.0 - 2.0 * ev / lmax)
    n = k + 1
    Wn = np.sin((n + 0.5) * t) / np.sin(0.5 * t)
    pk = (1.0 - Wn / (2 * n + 1)) / ev
    rg = np.zeros(P.n_unique); rg[free] = np.random.default_rng(8).standard_normal(free.sum())
    z = P.cheb4_jacobi(k, lmax, to_local(P, rg))
    expect = (V * pk) @ (V.T @ (rg[free] / np.sqrt(Dm))) / np.sqrt(Dm)
    assert np.allclose(to_global(P, z)[free], expect, rtol=0, atol=1e-12 * np.abs(expect).max())
    assert np.all(pk > 0)                                             # SPD smoother on (0, lmax]
    assert np.all(np.abs(Wn) <= 2 * n + 1 + 1e-9)


def test_fourth_kind_vcycle_converges_comparably(orc, xi_of):
    m, _ = I.config_mesh(2, xi_of, small=True)
    b = None; its = {}
    for kind in (1, 4):
        mg = _mg(orc, m, 0.0, 0b10, [7, 3, 1], k=2, kc=4, kind=kind)
        P = mg.levels[0]
        b = P.assemble_rhs(I.divergence_source(m, 5))
        r = mg.pcg(b)
        assert r["status"] == 0
        res = b - P.apply_A(r["x"])
        assert np.sqrt(P.dot(res, res)) <= 2e-10 * np.sqrt(P.dot(b, b))
        its[kind] = r["iters"]
    # measured: 37 (first kind on [0.1, 1] lmax) vs 40 (fourth kind, which needs no lower bound)
    assert its[4] <= 1.25 * its[1] and its[1] <= 1.25 * its[4], its


def test_fp32_storage_vcycle_is_a_small_perturbation(orc, xi_of):
    """R21: with FP32 storage of the levels the V-cycle differs from the fp64 one by float rounding only (each stored
    vector carries a relative error <= 2^-24, a few dozen stores per cycle), it leaves the fp64 V-cycle bit-for-bit
    untouched, and PCG around it reaches the same fp64 solution in the same number of iterations (+-1)."""
    m, _ = I.config_mesh(2, xi_of, small=True)
    kw = dict(k=1, kc=8, frac=0.05)
    mg64 = _mg(orc, m, 0.0, 0b10, [7, 3, 1], **kw)
    mg32 = orc.Multigrid(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, 0.0, 0b10, [7, 3, 1], k_smooth=1, k_coarse=8,
                         coarse_frac=0.05, lmax=mg64.lmax, fp32=True)
    P = mg64.levels[0]
    r = _cont(orc, P, 77)
    z64 = mg64.vcycle(r)
    z32 = mg32.vcycle(r)
    err = np.abs(z32 - z64).max() / np.abs(z64).max()
    assert 1e-9 < err < 5e-6, err                                   # rounding did happen, and only rounding
    assert np.array_equal(mg64.vcycle(r), z64)                      # the flag is off again outside the fp32 cycle
    assert np.array_equal(z32.astype(np.float32).astype(np.float64), z32)   # the result is a stored (float) vector
    assert np.all(z32[P.mask == 0] == 0)
    b = P.assemble_rhs(I.divergence_source(m, 5))
    r64, r32 = mg64.pcg(b), mg32.pcg(b)
    assert r64["status"] == 0 and r32["status"] == 0 and abs(r64["iters"] - r32["iters"]) <= 1
    assert np.abs(r32["x"] - r64["x"]).max() <= 1e-8 * np.abs(r64["x"]).max()
    res = b - P.apply_A(r32["x"])                                   # fp64 operator, fp64 residual
    assert np.sqrt(P.dot(res, res)) <= 2e-10 * np.sqrt(P.dot(b, b))
