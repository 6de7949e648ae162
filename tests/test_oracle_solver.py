"""Pins P10, P12, P13 of SURVEY.md §8(c) plus Lanczos and consumer pins: PCG, Chebyshev-Jacobi, export consumer.

Expected values: dense direct solves, scipy's CG (library routine), the closed-form Chebyshev
residual polynomial, the analytic manufactured solution, numpy reductions -- never the oracle itself.
"""
import numpy as np
import pytest
import scipy.sparse.linalg as spla
from numpy.polynomial import chebyshev as Ch

from paper_2501_13240_b200 import inputs as I
from test_oracle_operator import dense_matrix, make, to_global, to_local


def _free_system(P):
    A = dense_matrix(P)
    free = to_global(P, P.mask) > 0
    return A, free


# ---------------------------------------------------------------- P12: PCG vs dense direct solve / textbook CG
@pytest.mark.parametrize("precond", [0, 1, 2])
def test_pcg_matches_dense_solve(orc, xi_of, precond):
    N = 3
    m = I.box_mesh(2, 2, 3, N, xi_of(N), deform=0.05)
    P = make(orc, m, lam=0.0, tags=0b10)
    A, free = _free_system(P)
    f = I.uniform(21, m.n)
    b = P.assemble_rhs(orc.gs(P.gid, P.n_unique, f * P.invmult))          # continuous nodal f
    lmax = 0.0
    if precond == 2:
        Dm = np.diag(A)[free]
        lmax = 1.05 * np.linalg.eigvalsh(A[np.ix_(free, free)] / np.sqrt(np.outer(Dm, Dm)))[-1]
    r = P.pcg(b, precond=precond, cheb_k=2, lmax=lmax, rtol=1e-13, hist_len=400)
    assert r["status"] == 0
    xd = np.zeros(P.n_unique)
    xd[free] = np.linalg.solve(A[np.ix_(free, free)], to_global(P, b)[free])
    assert np.allclose(to_global(P, r["x"]), xd, rtol=0, atol=1e-10 * np.abs(xd).max())
    assert np.all(r["x"][P.mask == 0] == 0)
    # A-norm of the error decreases monotonically (CG optimality): check through the returned history
    # being finite and the final residual meeting the stopping rule on the unique-node 2-norm
    rb = to_global(P, b) - A @ to_global(P, r["x"])
    assert np.linalg.norm(rb) <= 1e-11 * np.linalg.norm(to_global(P, b))
    assert r["iters"] <= free.sum()                                        # finite termination


def test_unpreconditioned_pcg_is_textbook_cg(orc, xi_of):
    """precond 0 must reproduce scipy's CG iterate after the same number of steps (residual history)."""
    N = 3
    m = I.box_mesh(2, 2, 2, N, xi_of(N), deform=0.05)
    P = make(orc, m, lam=1.0, tags=0)
    A = dense_matrix(P)
    b = P.assemble_rhs(orc.gs(P.gid, P.n_unique, I.uniform(5, m.n) * P.invmult))
    bg = to_global(P, b)
    for its in (1, 3, 10):
        r = P.pcg(b, precond=0, rtol=0.0, maxit=its, hist_len=its + 1)
        assert r["status"] == 1 and r["iters"] == its
        xs, _ = spla.cg(A, bg, rtol=0.0, atol=0.0, maxiter=its)
        assert np.allclose(to_global(P, r["x"]), xs, rtol=0, atol=1e-11 * np.abs(xs).max())
        assert abs(r["hist"][its] - np.linalg.norm(bg - A @ xs)) <= 1e-9 * r["hist"][0]


def test_pcg_zero_rhs_and_initial_guess(orc, xi_of):
    N = 3
    m = I.box_mesh(2, 2, 2, N, xi_of(N))
    P = make(orc, m, lam=2.0, tags=0b10)
    r = P.pcg(np.zeros(P.n))
    assert r["iters"] == 0 and r["status"] == 0 and np.all(r["x"] == 0)
    b = P.assemble_rhs(orc.gs(P.gid, P.n_unique, I.uniform(9, m.n) * P.invmult))
    r1 = P.pcg(b, rtol=1e-12)
    r2 = P.pcg(b, x0=r1["x"], rtol=1e-8)                                   # already converged start
    assert r2["iters"] == 0 and np.array_equal(r2["x"], r1["x"])
    r3 = P.pcg(b, x0=0.5 * r1["x"], rtol=1e-12)
    assert np.allclose(r3["x"], r1["x"], rtol=0, atol=1e-10 * np.abs(r1["x"]).max())


# ---------------------------------------------------------------- P13: Chebyshev-Jacobi = closed-form polynomial
@pytest.mark.parametrize("k", [0, 1, 2, 3])
def test_chebyshev_jacobi_closed_form(orc, xi_of, k):
    """z = p_k(D^-1 A) D^-1 r with lam p_k(lam) = 1 - T_{k+1}((theta-lam)/delta) / T_{k+1}(sigma)."""
    N = 3
    m = I.ogrid_mesh(2, 2, 2, N, xi_of(N))
    P = make(orc, m, tags=0b10)
    A, free = _free_system(P)
    Af = A[np.ix_(free, free)]
    Dm = np.diag(Af)
    S = Af / np.sqrt(np.outer(Dm, Dm))                                     # D^-1/2 A D^-1/2
    ev, V = np.linalg.eigh(S)
    lmax = 1.1 * ev[-1]
    lmin = 0.1 * lmax; theta = 0.5 * (lmax + lmin); delta = 0.5 * (lmax - lmin); sigma = theta / delta
    Tk1 = Ch.Chebyshev.basis(k + 1)
    pk = (1.0 - Tk1((theta - ev) / delta) / Tk1(sigma)) / ev
    rg = np.zeros(P.n_unique); rg[free] = np.random.default_rng(4).standard_normal(free.sum())
    z = P.cheb_jacobi(k, lmax, to_local(P, rg))
    expect = (V * pk) @ (V.T @ (rg[free] / np.sqrt(Dm))) / np.sqrt(Dm)
    assert np.allclose(to_global(P, z)[free], expect, rtol=0, atol=1e-12 * np.abs(expect).max())
    assert np.all(pk > 0)                                                  # SPD preconditioner on (0, lmax]
    assert np.all(to_global(P, z)[~free] == 0)


def test_chebyshev_reduces_iterations_and_lanczos_bounds(orc, xi_of):
    m, _ = I.config_mesh(2, xi_of, small=True)
    P = make(orc, m, tags=0b10)
    v0 = P.mask * orc.gs(P.gid, P.n_unique, P.invmult * I.uniform(7, P.n))
    lmax = P.lanczos_lmax(v0, steps=10)
    b = P.assemble_rhs(I.divergence_source(m, 5))
    its = [P.pcg(b, precond=pc, cheb_k=k, lmax=lmax)["iters"] for pc, k in [(1, 0), (2, 1), (2, 2)]]
    assert its[0] > its[1] > its[2] and its[2] < 0.5 * its[0]
    x1 = P.pcg(b, precond=1)["x"]; x2 = P.pcg(b, precond=2, cheb_k=2, lmax=lmax)["x"]
    assert np.abs(x1 - x2).max() <= 1e-8 * np.abs(x1).max()
    # independent estimate of lambda_max(D^-1 A): power iteration written with numpy on the oracle's operator
    v = v0 / np.sqrt(P.dot(v0, v0))
    for _ in range(300):
        w = P.dinv * P.apply_A(v) * P.mask
        lam_pow = P.dot(v, P.apply_A(v)) / P.dot(v, v / P.dinv)
        v = w / np.sqrt(P.dot(w, w))
    assert lam_pow <= lmax <= 1.25 * lam_pow


@pytest.mark.parametrize("lam,tags", [(0.0, 0b10), (25.0, 0)])
def test_lanczos_ritz_values_are_the_rayleigh_ritz_values_of_the_krylov_space(orc, xi_of, lam, tags):
    """orc_lanczos pinned by the DEFINITION of its output: the eigenvalues of its tridiagonal matrix are the
    Rayleigh-Ritz values of S = D^-1/2 A D^-1/2 on the Krylov space span{v0, S v0, .., S^(m-1) v0}.  Here that space is
    built from the dense matrix by Arnoldi with full re-orthogonalisation in numpy (no three-term recurrence), on the
    unique free nodes, and all m Ritz values are compared."""
    import ctypes as C
    N, steps = 3, 10
    m = I.box_mesh(2, 2, 3, N, xi_of(N), deform=0.05)
    P = make(orc, m, lam=lam, tags=tags)
    A = dense_matrix(P)
    free = to_global(P, P.mask) > 0
    dg = to_global(P, 1.0 / P.dinv)[free]
    Sd = A[np.ix_(free, free)] / np.sqrt(np.outer(dg, dg))
    v0 = P.mask * orc.gs(P.gid, P.n_unique, P.invmult * I.uniform(11, P.n))
    a = np.zeros(steps); b = np.zeros(steps)
    k = orc.lib().orc_lanczos(C.byref(P._op), P.dinv.ctypes.data_as(C.c_void_p), v0.ctypes.data_as(C.c_void_p), C.c_int(steps),
                              a.ctypes.data_as(C.c_void_p), b.ctypes.data_as(C.c_void_p))
    assert k == steps
    T = np.diag(a) + np.diag(b[:-1], 1) + np.diag(b[:-1], -1)
    ritz = np.linalg.eigvalsh(T)
    Q = np.zeros((free.sum(), steps))
    q = to_global(P, v0)[free]
    for j in range(steps):
        for _ in range(2):
            q = q - Q[:, :j] @ (Q[:, :j].T @ q)
        Q[:, j] = q / np.linalg.norm(q)
        q = Sd @ Q[:, j]
    expect = np.linalg.eigvalsh(Q.T @ Sd @ Q)
    assert np.allclose(ritz, expect, rtol=1e-9, atol=0)
    top = np.linalg.eigvalsh(Sd)[-1]
    assert ritz[-1] <= top * (1 + 1e-12) and 1.1 * ritz[-1] >= top           # what lanczos_lmax relies on
    assert abs(P.lanczos_lmax(v0, steps) - 1.1 * expect[-1]) <= 1e-9 * top


# ---------------------------------------------------------------- P10: spectral convergence (reading R1 / SURVEY A1)
def test_spectral_convergence_dirichlet_cube(orc, xi_of):
    errs = []
    for N in range(2, 9):
        m = I.box_mesh(2, 2, 2, N, xi_of(N))
        P = make(orc, m, tags=0b110)                                      # Dirichlet on all six faces
        us, f = I.manufactured_sin(m)
        r = P.pcg(P.assemble_rhs(f), rtol=1e-13)
        assert r["status"] == 0
        errs.append(np.abs(r["x"] - us).max())
    errs = np.array(errs)
    assert np.all(errs[1:] < errs[:-1] / 5.0)                              # faster than any fixed algebraic rate
    assert errs[0] < 5e-2 and errs[3] < 5e-6 and errs[-1] < 5e-10
    # h-refinement at fixed N converges too (4^3 elements, N = 7: survey prototype 2.9e-12)
    m = I.box_mesh(4, 4, 4, 7, xi_of(7))
    P = make(orc, m, tags=0b110)
    us, f = I.manufactured_sin(m)
    assert np.abs(P.pcg(P.assemble_rhs(f), rtol=1e-13)["x"] - us).max() < 2e-11


def test_periodic_manufactured_solution(orc, xi_of):
    """configs[0] boundary conditions with a BC-compatible u* = sin(2 pi x) sin(2 pi y) sin(pi z)."""
    m, _ = I.config_mesh(0, xi_of)
    P = make(orc, m, tags=0b10)
    us, f = I.manufactured_sin(m, 2.0, 2.0, 1.0)
    r = P.pcg(P.assemble_rhs(f), rtol=1e-12)
    assert r["status"] == 0 and np.abs(r["x"] - us).max() < 1e-8


# ---------------------------------------------------------------- consumer (c-11)
def test_minmax_hist_and_vmag(orc):
    rng = np.random.default_rng(2)
    nb = 256
    bins = rng.integers(0, nb, 200000)
    v = (bins + 0.5) / nb                                                  # bin centres: no boundary ambiguity
    mn, mx, h = orc.minmax_hist(v, nb, 0.0, 1.0)
    assert mn == v.min() and mx == v.max()
    assert np.array_equal(h, np.bincount(bins, minlength=nb).astype(np.uint64))
    v = np.array([-3.0, 0.0, 0.999999, 1.0, 7.0, 0.5])                     # clamping to the end bins
    _, _, h = orc.minmax_hist(v, 4, 0.0, 1.0)
    assert list(h) == [2, 0, 1, 3]
    v = rng.uniform(0, 1, 100000)
    _, _, h = orc.minmax_hist(v, 64, 0.0, 1.0)
    hn, _ = np.histogram(v, bins=64, range=(0.0, 1.0))
    assert h.sum() == v.size and np.abs(h.astype(np.int64) - hn).sum() <= 4    # only edge-straddling values may differ
    a = np.array([3.0, 2.0, 1.0, 0.0]); b = np.array([4.0, 3.0, 4.0, 0.0]); c = np.array([12.0, 6.0, 8.0, 0.0])
    assert np.array_equal(orc.vmag(a, b, c), [13.0, 7.0, 9.0, 0.0])        # Pythagorean quadruples: exact
    x, y, z = rng.standard_normal((3, 1000))
    ref = np.sqrt(x.astype(np.longdouble) ** 2 + y.astype(np.longdouble) ** 2 + z.astype(np.longdouble) ** 2)
    assert np.all(np.abs(orc.vmag(x, y, z) - ref.astype(np.float64)) <= 2 * np.spacing(ref.astype(np.float64)))


# ---------------------------------------------------------------- R20: all-Neumann problem, zero-mean solution
@pytest.mark.parametrize("precond", [1, 2])
def test_null_mean_solution_is_the_pseudo_inverse_solution(orc, xi_of, precond):
    """lambda = 0 without Dirichlet nodes: A is singular with the constants as null space.  The solve of b - mean(b)
    returned with zero mean must equal numpy's pseudo-inverse (minimum-norm) solution on the unique nodes."""
    N = 3
    m = I.box_mesh(2, 3, 2, N, xi_of(N), deform=0.05)
    P = make(orc, m, lam=0.0, tags=0)
    A = dense_matrix(P)
    assert abs(np.linalg.eigvalsh(A)[0]) <= 1e-12 * np.linalg.eigvalsh(A)[-1]          # singular
    b = P.assemble_rhs(orc.gs(P.gid, P.n_unique, I.uniform(33, m.n) * P.invmult))       # NOT consistent: mean(b) != 0
    assert abs(P.mean(b)) > 1e-6
    lmax = 0.0
    if precond == 2:
        Dm = np.diag(A)
        lmax = 1.05 * np.linalg.eigvalsh(A / np.sqrt(np.outer(Dm, Dm)))[-1]
    r = P.pcg(b, precond=precond, cheb_k=2, lmax=lmax, rtol=1e-12, null_mean=True)
    assert r["status"] == 0
    xg = to_global(P, r["x"])
    bg = to_global(P, b)
    expect = np.linalg.pinv(A, hermitian=True) @ (bg - bg.mean())
    assert abs(xg.mean()) <= 1e-13 * np.abs(xg).max()
    assert np.allclose(xg, expect, rtol=0, atol=1e-9 * np.abs(expect).max())
