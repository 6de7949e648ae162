"""Pins P4-P9, P11, P14, P15 of SURVEY.md §8(c): axhelm, numbering, gather-scatter, mask, diagonal.

Expected values: closed forms, analytic integrals, brute force on tiny meshes, Kronecker-product
special case -- none produced by the oracle or the CUDA path.
"""
import numpy as np
import pytest

from paper_2501_13240_b200 import inputs as I


def make(orc, mesh, lam=0.0, tags=0):
    return orc.Problem(mesh.E, mesh.N, mesh.x, mesh.y, mesh.z, mesh.face_tag, mesh.period, lam=lam, dirichlet_tags=tags)


def to_local(P, vg):
    return vg[P.gid]


def to_global(P, vl):
    """one copy per global node (continuous vectors only)."""
    out = np.zeros(P.n_unique)
    out[P.gid] = vl
    return out


def dense_matrix(P):
    """assembled, masked operator as a dense [n_unique, n_unique] matrix, column by column."""
    A = np.zeros((P.n_unique, P.n_unique))
    for g in range(P.n_unique):
        e = np.zeros(P.n_unique); e[g] = 1.0
        A[:, g] = to_global(P, P.apply_A(to_local(P, e)))
    return A


# ---------------------------------------------------------------- P4, P5, P15
@pytest.mark.parametrize("kind", ["box", "ogrid"])
def test_const_nullspace_symmetry_and_local_pAp(orc, xi_of, kind):
    N = 5
    m = I.box_mesh(3, 2, 2, N, xi_of(N), deform=0.05) if kind == "box" else I.ogrid_mesh(2, 2, 2, N, xi_of(N))
    P = make(orc, m)
    # P4: A const = 0 for lambda = 0, unmasked
    w = P.apply_A(np.ones(P.n))
    assert np.abs(w).max() <= 1e-13 * np.abs(1.0 / P.dinv).max()
    # P5: x^T A y = y^T A x on random continuous vectors
    rng = np.random.default_rng(1)
    xg, yg = rng.standard_normal(P.n_unique), rng.standard_normal(P.n_unique)
    x, y = to_local(P, xg), to_local(P, yg)
    xAy, yAx = P.dot(x, P.apply_A(y)), P.dot(y, P.apply_A(x))
    assert abs(xAy - yAx) <= 1e-13 * max(abs(xAy), 1.0)
    # P15: p^T A p (assembled) = sum over local nodes of p_l (A_L p)_l, no weights
    loc = float(np.dot(x, orc.axhelm(m.E, N, P.geo, 0.0, x)))
    assert abs(loc - P.dot(x, P.apply_A(x))) <= 1e-13 * abs(loc)
    # Helmholtz term: A(lambda) - A(0) = lambda * assembled mass
    lam = 7.5
    P2 = make(orc, m, lam=lam)
    mass = orc.gs(P.gid, P.n_unique, P.geo[:, 6].ravel() * x)
    assert np.allclose(P2.apply_A(x) - P.apply_A(x), lam * mass, rtol=0, atol=1e-12 * np.abs(P2.apply_A(x)).max())


# ---------------------------------------------------------------- P6: exact weak Laplacian of monomials
def _mono_int(a, b, c, d, e, f):
    """int_[0,1]^3 grad(x^a y^b z^c) . grad(x^d y^e z^f)"""
    s = 0.0
    if a * d:
        s += a * d / ((a + d - 1) * (b + e + 1) * (c + f + 1))
    if b * e:
        s += b * e / ((a + d + 1) * (b + e - 1) * (c + f + 1))
    if c * f:
        s += c * f / ((a + d + 1) * (b + e + 1) * (c + f - 1))
    return s


def test_weak_laplacian_of_polynomials_affine(orc, xi_of):
    N = 4
    m = I.box_mesh(2, 3, 2, N, xi_of(N))
    P = make(orc, m)
    # GLL exactness needs deg_u + deg_v <= 2N-1 per variable (SURVEY P6 catch): deg u <= N, deg v <= N-1
    for (a, b, c), (d, e, f) in [((4, 4, 4), (3, 3, 3)), ((4, 0, 2), (1, 3, 2)), ((3, 2, 1), (3, 2, 1)), ((1, 1, 1), (1, 1, 1))]:
        u = m.x ** a * m.y ** b * m.z ** c
        v = m.x ** d * m.y ** e * m.z ** f
        got = P.dot(v, P.apply_A(u))
        assert abs(got - _mono_int(a, b, c, d, e, f)) < 2e-13, ((a, b, c), (d, e, f))
    # and it is NOT exact beyond the bound (guards against a vacuous test)
    u = m.x ** 4 * m.y ** 4
    assert abs(P.dot(u, P.apply_A(u)) - _mono_int(4, 4, 0, 4, 4, 0)) > 1e-9


def _mono_cross_int(p, q, a, b):
    """int_[0,1]^3 d_a(s^p) d_b(s^q) ds for monomials s^p = s1^p1 s2^p2 s3^p3 (a, b = directions 0..2)."""
    if p[a] == 0 or q[b] == 0:
        return 0.0
    v = float(p[a] * q[b])
    for d in range(3):
        e = p[d] + q[d] - (d == a) - (d == b)
        v /= (e + 1)
    return v


def test_weak_laplacian_of_polynomials_sheared_affine(orc, xi_of):
    """P6 on a SHEARED affine image X = A s of the unit cube: every element then has non-zero cross factors
    G_rs, G_rt, G_st, and  v^T A u = sum_ab C_ab int d_a p d_b q ds  with C = det(A) A^-1 A^-T in closed form --
    pins the use of the cross terms inside orc_axhelm analytically (a dropped, doubled or swapped cross term fails)."""
    N = 4
    m = I.box_mesh(2, 3, 2, N, xi_of(N))
    A = np.array([[1.0, 0.35, 0.2], [0.0, 0.9, 0.45], [0.15, 0.0, 1.2]])
    S = np.stack([m.x, m.y, m.z])                     # unit-cube coordinates s of every node
    X = A @ S
    P = orc.Problem(m.E, N, X[0], X[1], X[2], m.face_tag, [0, 0, 0])
    # the factors really are full: all three cross factors are of the size of the diagonal ones
    for c in (1, 2, 4):
        assert np.abs(P.geo[:, c]).max() > 0.05 * np.abs(P.geo[:, 0]).max()
    Ai = np.linalg.inv(A)
    Cm = np.linalg.det(A) * Ai @ Ai.T
    for pu, pv in [((4, 4, 4), (3, 3, 3)), ((4, 0, 2), (1, 3, 2)), ((3, 2, 1), (3, 2, 1)), ((1, 1, 0), (0, 1, 1)), ((2, 1, 3), (1, 3, 0))]:
        u = S[0] ** pu[0] * S[1] ** pu[1] * S[2] ** pu[2]
        v = S[0] ** pv[0] * S[1] ** pv[1] * S[2] ** pv[2]
        expect = sum(Cm[a, b] * _mono_cross_int(pu, pv, a, b) for a in range(3) for b in range(3))
        got = P.dot(v, P.apply_A(u))
        assert abs(got - expect) < 5e-13 * max(1.0, abs(expect)), (pu, pv, got, expect)
    # a pair whose value comes from the cross terms alone (u depends on s1 only, v on s2 only)
    u, v = S[0] ** 3, S[1] ** 2
    expect = Cm[0, 1] * _mono_cross_int((3, 0, 0), (0, 2, 0), 0, 1)
    assert abs(expect) > 0.1 and abs(P.dot(v, P.apply_A(u)) - expect) < 5e-13


def test_min_spacing_closed_form(orc, xi_of):
    """orc_min_spacing (sets the matching tolerance, R17): on an affine brick the smallest node spacing is
    (xi_1 - xi_0)/2 times the smallest element width -- closed form from the GLL points, which P1 pins."""
    for N, (nx, ny, nz) in [(3, (2, 3, 5)), (7, (4, 2, 3))]:
        m = I.box_mesh(nx, ny, nz, N, xi_of(N))
        xi = xi_of(N)
        expect = 0.5 * (xi[1] - xi[0]) * min(1.0 / nx, 1.0 / ny, 1.0 / nz)
        assert abs(orc.min_spacing(m.E, N, m.x, m.y, m.z) - expect) <= 1e-14


# ---------------------------------------------------------------- P7: Kronecker form on an affine structured box
def _assembled_1d(orc, ne, N, h):
    xi, rho = orc.gll(N)
    D = orc.dhat(N, xi)
    ng = ne * N + 1
    K = np.zeros((ng, ng)); M = np.zeros(ng)
    Ke = (2.0 / h) * D.T @ np.diag(rho) @ D
    for e in range(ne):
        s = slice(e * N, e * N + N + 1)
        K[s, s] += Ke
        M[s] += (h / 2.0) * rho
    return K, np.diag(M)


def test_kronecker_special_case(orc, xi_of):
    N = 3
    nx, ny, nz = 2, 3, 2
    m = I.box_mesh(nx, ny, nz, N, xi_of(N))
    lam = 2.0
    P = make(orc, m, lam=lam)
    A = dense_matrix(P)
    Kx, Mx = _assembled_1d(orc, nx, N, 1 / nx); Ky, My = _assembled_1d(orc, ny, N, 1 / ny); Kz, Mz = _assembled_1d(orc, nz, N, 1 / nz)
    # lattice index of every global node (gx fastest) from the coordinates
    gx = np.rint(to_global(P, m.x) * 0 + np.searchsorted(np.unique(np.round(m.x, 12)), np.round(to_global(P, m.x), 12))).astype(int)
    gy = np.searchsorted(np.unique(np.round(m.y, 12)), np.round(to_global(P, m.y), 12))
    gz = np.searchsorted(np.unique(np.round(m.z, 12)), np.round(to_global(P, m.z), 12))
    lin = (gz * (ny * N + 1) + gy) * (nx * N + 1) + gx
    T = np.kron(Mz, np.kron(My, Kx)) + np.kron(Mz, np.kron(Ky, Mx)) + np.kron(Kz, np.kron(My, Mx)) \
        + lam * np.kron(Mz, np.kron(My, Mx))
    assert np.allclose(A, T[np.ix_(lin, lin)], rtol=0, atol=1e-13 * np.abs(T).max())


# ---------------------------------------------------------------- P8: definiteness by dense eigenvalues
def test_definiteness_tiny(orc, xi_of):
    N = 3
    m = I.box_mesh(2, 2, 2, N, xi_of(N), deform=0.05)
    ev = np.linalg.eigvalsh(dense_matrix(make(orc, m)))
    assert abs(ev[0]) < 1e-12 * ev[-1] and ev[1] > 1e-6 * ev[-1]          # exactly one zero mode (constants)
    P = make(orc, m, tags=0b10)                                            # Dirichlet on z = 0,1
    A = dense_matrix(P)
    free = to_global(P, P.mask) > 0
    assert np.all(A[~free] == 0) and np.all(A[:, ~free] == 0)
    assert np.linalg.eigvalsh(A[np.ix_(free, free)])[0] > 1e-6 * ev[-1]
    assert np.linalg.eigvalsh(dense_matrix(make(orc, m, lam=3.0)))[0] > 0


# ---------------------------------------------------------------- P9: numbering
def _brute_partition(m, tol):
    """O(n^2) definition: same node iff coordinates agree within tol after periodic wrapping."""
    C = np.stack([m.x, m.y, m.z], 1)
    label = np.arange(m.n)
    for l in range(m.n):
        d = np.abs(C - C[l])
        for k in range(3):
            if m.period[k] > 0:
                d[:, k] = np.minimum(d[:, k], np.abs(d[:, k] - m.period[k]))
        label[l] = np.flatnonzero(np.all(d <= tol, 1))[0]
    return label


@pytest.mark.parametrize("kind", ["box_periodic", "box_deformed", "ogrid"])
def test_numbering_matches_bruteforce_first_touch(orc, xi_of, kind):
    N = 3
    if kind == "box_periodic":
        m = I.box_mesh(3, 2, 2, N, xi_of(N), periodic=(True, True, False))
    elif kind == "box_deformed":
        m = I.box_mesh(2, 2, 3, N, xi_of(N), deform=0.05)
    else:
        m = I.ogrid_mesh(2, 2, 2, N, xi_of(N))
    tol = 1e-8 * orc.min_spacing(m.E, m.N, m.x, m.y, m.z)
    gid, nu = orc.numbering(m.E, m.N, m.x, m.y, m.z, m.period)
    label = _brute_partition(m, tol)
    firsts = np.flatnonzero(label == np.arange(m.n))                     # class representatives, ascending
    assert nu == firsts.size
    expect = np.searchsorted(firsts, label).astype(np.int32)             # rank of the smallest member
    assert np.array_equal(gid, expect)


def test_numbering_counts(orc, xi_of):
    m, _ = I.config_mesh(0, xi_of)                                        # 4^3, N=7, periodic x,y
    gid, nu = orc.numbering(m.E, m.N, m.x, m.y, m.z, m.period)
    assert nu == 28 * 28 * 29 == 22736
    mult = np.bincount(gid)[gid]
    assert np.array_equal(np.bincount(mult, minlength=9)[[1, 2, 4, 8]], [14976, 13440, 3968, 384])
    assert abs(np.sum(1.0 / mult) - nu) < 1e-9
    m = I.box_mesh(3, 4, 2, 5, xi_of(5), periodic=(True, True, False))   # Table-4 style (nx p)(ny p)(nz p + 1)
    assert orc.numbering(m.E, m.N, m.x, m.y, m.z, m.period)[1] == 15 * 20 * 11
    m = I.box_mesh(3, 3, 3, 4, xi_of(4), deform=0.05)
    assert orc.numbering(m.E, m.N, m.x, m.y, m.z, m.period)[1] == 13 ** 3
    m = I.ogrid_mesh(4, 3, 4, 7, xi_of(7))
    gid, nu = orc.numbering(m.E, m.N, m.x, m.y, m.z, m.period)
    assert nu == I.ogrid_unique_nodes(4, 3, 4, 7) == 92597
    assert set(np.unique(np.bincount(gid))) == {1, 2, 3, 4, 6, 8}        # 3 elements meet at the inner-square corners


def test_numbering_structured_lattice_formula(orc, xi_of):
    N, nx, ny, nz = 4, 3, 2, 2
    m = I.box_mesh(nx, ny, nz, N, xi_of(N), periodic=(True, False, False))
    gid, nu = orc.numbering(m.E, m.N, m.x, m.y, m.z, m.period)
    e = np.arange(m.n) // m.Np; loc = np.arange(m.n) % m.Np
    i, j, k = loc % (N + 1), (loc // (N + 1)) % (N + 1), loc // (N + 1) ** 2
    ex, ey, ez = e % nx, (e // nx) % ny, e // (nx * ny)
    ix = (ex * N + i) % (nx * N); iy = ey * N + j; iz = ez * N + k
    lattice = (iz * (ny * N + 1) + iy) * (nx * N) + ix
    # same partition: lattice id <-> gid is a bijection
    pairs = np.unique(np.stack([lattice, gid], 1), axis=0)
    assert pairs.shape[0] == nu == np.unique(lattice).size


# ---------------------------------------------------------------- P14: gather-scatter
def test_gs_integers_bitwise_and_mult(orc, xi_of):
    m = I.ogrid_mesh(2, 2, 2, 4, xi_of(4))
    gid, nu = orc.numbering(m.E, m.N, m.x, m.y, m.z, m.period)
    rng = np.random.default_rng(3)
    v = rng.integers(-(1 << 19), 1 << 19, m.n).astype(np.float64)
    s = np.zeros(nu); np.add.at(s, gid, v)
    assert np.array_equal(orc.gs(gid, nu, v), s[gid])
    assert np.array_equal(orc.gs(gid, nu, np.ones(m.n)), np.bincount(gid)[gid].astype(float))   # QQ^T 1 = mult


def test_mask_counts_and_class_or(orc, xi_of):
    m, _ = I.config_mesh(0, xi_of)
    P = make(orc, m, tags=0b10)
    assert int((P.mask == 0).sum()) == 2 * 16 * 64                       # z=0 and z=1 faces of 4x4 elements
    assert np.all(m.z[P.mask == 0] * (1 - m.z[P.mask == 0]) == 0) and np.all((m.z[P.mask == 1] > 0) & (m.z[P.mask == 1] < 1))
    m = I.box_mesh(2, 2, 2, 3, xi_of(3))
    P = make(orc, m, tags=0b100)                                         # side walls only (tag 2)
    on_wall = (m.x == 0) | (m.x == 1) | (m.y == 0) | (m.y == 1)
    assert np.array_equal(P.mask == 0, on_wall)                          # includes copies in elements whose own face is interior
    assert np.all(make(orc, m, tags=0).mask == 1)


# ---------------------------------------------------------------- P11: diagonal by brute force
def test_diagonal_bruteforce(orc, xi_of):
    N = 3
    m = I.box_mesh(2, 2, 2, N, xi_of(N), deform=0.08)
    for lam in (0.0, 11.0):
        P = make(orc, m, lam=lam)
        A = dense_matrix(P)
        got = to_global(P, 1.0 / P.dinv)
        assert np.allclose(got, np.diag(A), rtol=1e-13)
    P = make(orc, m, tags=0b10)
    assert np.all(P.dinv[P.mask == 0] == 1.0)
    # the edge/corner cross terms matter on non-orthogonal elements: dropping them must be visible
    m = I.ogrid_mesh(2, 2, 1, N, xi_of(N))
    P = make(orc, m)
    d = orc.diag_local(m.E, N, P.geo, 0.0)
    l = 4 * m.Np                                                         # corner node of the first east-block element
    e0 = np.zeros(m.n); e0[l] = 1.0
    assert abs(orc.axhelm(m.E, N, P.geo, 0.0, e0)[l] - d[l]) < 1e-14 * abs(d[l])
    D = orc.dhat(N)
    cross = 2 * (D[0, 0] ** 2) * (P.geo[4, 1, 0] + P.geo[4, 2, 0] + P.geo[4, 4, 0])
    assert abs(cross) > 1e-3 * abs(d[l])


def test_axhelm_variable_coefficients(orc, xi_of):
    """lam0/lam1 fields (reading R3): constant fields reduce to scaled scalar operator."""
    N = 4
    m = I.box_mesh(2, 2, 2, N, xi_of(N), deform=0.05)
    P = make(orc, m)
    u = I.uniform(11, m.n)
    w = orc.axhelm(m.E, N, P.geo, 0.0, u, lam0=np.full(m.n, 2.5), lam1=np.full(m.n, 3.0))
    ref = 2.5 * orc.axhelm(m.E, N, P.geo, 0.0, u) + 3.0 * P.geo[:, 6].ravel() * u
    assert np.allclose(w, ref, rtol=0, atol=1e-13 * np.abs(ref).max())
