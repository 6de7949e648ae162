"""Pins of the flow operators and of the Boussinesq step of the oracle (oracle/semflow.c, oracle/boussinesq.py;
SURVEY.md §8 f-2; reading R25): closed-form metrics, exact differentiation of polynomials, analytic integrals for
the weak divergence, the conduction state as a fixed point, and second-order convergence in time on a manufactured solution
whose forcing sympy derives from PAPER.md Eqs. (1)-(3)."""
import numpy as np
import pytest

from paper_2501_13240_b200 import inputs as I


def sheared_box(orc, nx, ny, nz, N):
    m = I.box_mesh(nx, ny, nz, N, orc.gll(N)[0])
    A = np.array([[1.0, 0.35, 0.2], [0.0, 0.9, 0.45], [0.15, 0.0, 1.2]])
    S = np.stack([m.x, m.y, m.z])
    X = A @ S
    P = orc.Problem(m.E, N, X[0], X[1], X[2], m.face_tag, [0, 0, 0])
    return m, A, S, X, P


def test_metrics_grad_and_wdiv_on_a_sheared_affine_mesh(orc):
    from oracle import boussinesq as Bq
    N, (nx, ny, nz) = 4, (2, 3, 2)
    m, A, S, X, P = sheared_box(orc, nx, ny, nz, N)
    ops = Bq.FlowOps(P, X[0], X[1], X[2])
    # metrics: x = A s, s = s0 + h (r + 1) / 2 per direction  =>  dr_a/dx_b = (2 / h_a) (A^-1)_ab, constant
    Ai = np.linalg.inv(A)
    h = np.array([1.0 / nx, 1.0 / ny, 1.0 / nz])
    for a in range(3):
        for b in range(3):
            assert np.abs(ops.met[:, 3 * a + b] - 2.0 / h[a] * Ai[a, b]).max() < 1e-11
    # gradient of polynomials in the PHYSICAL coordinates of degree <= N per reference direction: exact
    for pw in [(4, 0, 0), (1, 2, 1), (0, 3, 1), (2, 2, 0)]:
        s1, s2, s3 = S
        f = s1 ** pw[0] * s2 ** pw[1] * s3 ** pw[2]
        ds = [pw[0] * s1 ** max(pw[0] - 1, 0) * s2 ** pw[1] * s3 ** pw[2] if pw[0] else 0 * s1,
              pw[1] * s1 ** pw[0] * s2 ** max(pw[1] - 1, 0) * s3 ** pw[2] if pw[1] else 0 * s1,
              pw[2] * s1 ** pw[0] * s2 ** pw[1] * s3 ** max(pw[2] - 1, 0) if pw[2] else 0 * s1]
        g = ops.grad(f)
        for b in range(3):                                           # df/dx_b = sum_a df/ds_a (A^-1)_ab
            expect = sum(ds[a] * Ai[a, b] for a in range(3))
            assert np.abs(g[b] - expect).max() < 2e-12, (pw, b)
    # weak divergence: v^T wdiv(g) = int grad v . g dX analytically (monomials in s, degrees within the GLL exactness)
    detA = np.linalg.det(A)

    def mono_int(p):
        return 1.0 / ((p[0] + 1) * (p[1] + 1) * (p[2] + 1))
    v = S[0] ** 2 * S[1] * S[2] ** 3
    dv = [(2, (1, 1, 3)), (1, (2, 0, 3)), (3, (2, 1, 2))]           # (coefficient, exponents) of dv/ds_a
    gq = [(1, 0, 2), (0, 2, 1), (3, 1, 0)]                           # g_b = s^gq[b]
    gvec = [S[0] ** q[0] * S[1] ** q[1] * S[2] ** q[2] for q in gq]
    expect = 0.0
    for b in range(3):
        for a in range(3):
            c, pe = dv[a]
            expect += detA * Ai[a, b] * c * mono_int(tuple(pe[d] + gq[b][d] for d in range(3)))
    got = float(np.dot(v, ops.wdiv(*gvec)))
    assert abs(got - expect) < 1e-13 * max(1.0, abs(expect))


@pytest.mark.parametrize("kind", ["box_deformed", "ogrid"])
def test_grad_of_linear_functions_is_exact_on_curved_meshes_and_wdiv_is_its_transpose(orc, xi_of, kind):
    from oracle import boussinesq as Bq
    m = I.box_mesh(2, 2, 2, 5, xi_of(5), deform=0.05) if kind == "box_deformed" else I.config_mesh(2, xi_of, small=True)[0]
    P = orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period)
    ops = Bq.FlowOps(P, m.x, m.y, m.z)
    f = 0.7 * m.x - 1.3 * m.y + 0.4 * m.z + 2.0                     # isoparametric: J^-T (J^T a) = a on any element
    g = ops.grad(f)
    scale = np.abs(ops.met).max() * np.abs(f).max()
    for b, a in enumerate((0.7, -1.3, 0.4)):
        assert np.abs(g[b] - a).max() < 1e-13 * scale
    # transpose identity: sum_l v_l wdiv(g)_l = sum_l B_l grad v_l . g_l  for arbitrary nodal data
    v = I.uniform(1, m.n); gv = [I.uniform(2 + c, m.n) for c in range(3)]
    gr = ops.grad(v)
    lhs = float(np.dot(v, ops.wdiv(*gv)))
    rhs = float(np.sum(ops.B.ravel() * (gr[0] * gv[0] + gr[1] * gv[1] + gr[2] * gv[2])))
    assert abs(lhs - rhs) < 1e-12 * np.sum(np.abs(ops.B.ravel() * (gr[0] * gv[0])))
    # and the assembled Laplacian is wdiv o grad:  QQ^T wdiv(grad v) = A v for continuous v
    vg = I.uniform(9, P.n_unique)[P.gid]
    lap = orc.gs(P.gid, P.n_unique, ops.wdiv(*ops.grad(vg)))
    ref = P.apply_A(vg)
    assert np.abs(lap - ref).max() < 1e-11 * np.abs(ref).max()


def test_conduction_state_is_a_fixed_point(orc, xi_of):
    """zero velocity and T = 1 - z.  Buoyancy (1 - z) z^ is the gradient of z - z^2/2, which lies in the
    pressure space, so the discrete step keeps u = 0, theta = 0 to the solver tolerance."""
    from oracle import boussinesq as Bq
    N = 4
    m = I.box_mesh(2, 2, 3, N, xi_of(N), periodic=(True, True, False), zstretch=1.5)
    P = orc.Problem(m.E, N, m.x, m.y, m.z, m.face_tag, m.period)
    S = Bq.Boussinesq(P, m.x, m.y, m.z, Ra=1e4, Pr=0.7, dt=0.01, tags_u=0b10, tags_T=0b10, rtol=1e-12)
    for _ in range(3):
        S.step()
    assert max(np.abs(c).max() for c in S.u) < 1e-9 and np.abs(S.th).max() < 1e-9
    # the pressure is the hydrostatic one up to a constant: grad p = (0, 0, 1 - z)
    gp = S.ops.grad(S.p)
    assert np.abs(gp[2] - (1.0 - m.z)).max() < 1e-8 and np.abs(gp[0]).max() < 1e-8


def _manufactured():
    import sympy as sp
    x, y, z, t, nu, ka = sp.symbols("x y z t nu kappa")
    gt = sp.Rational(1, 10) * sp.cos(t)
    ux = gt * sp.pi * sp.sin(2 * sp.pi * x) * sp.sin(2 * sp.pi * z)
    uy = sp.Integer(0) * x
    uz = -2 * sp.pi * gt * sp.cos(2 * sp.pi * x) * sp.sin(sp.pi * z) ** 2
    th = sp.Rational(1, 5) * sp.sin(t + 1) * sp.sin(2 * sp.pi * x) * sp.sin(sp.pi * z)
    p = sp.cos(2 * sp.pi * x) * sp.cos(sp.pi * z) * sp.sin(t)
    T = th + 1 - z
    U = [ux, uy, uz]
    assert sp.simplify(sum(sp.diff(U[c], v) for c, v in enumerate((x, y, z)))) == 0
    lap = lambda q: sum(sp.diff(q, v, 2) for v in (x, y, z))
    adv = lambda q: sum(U[c] * sp.diff(q, v) for c, v in enumerate((x, y, z)))
    f = [sp.diff(U[c], t) + adv(U[c]) + sp.diff(p, v) - nu * lap(U[c]) - (T if c == 2 else 0) for c, v in enumerate((x, y, z))]
    fT = sp.diff(th, t) + adv(T) - ka * lap(th)
    L = lambda e: sp.lambdify((x, y, z, t, nu, ka), e, "numpy")
    return [L(e) for e in U], L(th), [L(e) for e in f] + [L(fT)]


def test_second_order_in_time_on_a_manufactured_solution(orc, xi_of):
    """Forcing derived by sympy from PAPER.md Eqs. (1)-(3); periodic x, y, no-slip isothermal plates.  Halving dt divides
    the velocity and temperature errors at t = 0.2 by about 4 (BDF2 / EXT2 with the curl-curl pressure boundary term)."""
    from oracle import boussinesq as Bq
    N = 8
    m = I.box_mesh(2, 1, 2, N, xi_of(N), periodic=(True, True, False))
    P = orc.Problem(m.E, N, m.x, m.y, m.z, m.face_tag, m.period)
    U, TH, F = _manufactured()
    Ra, Pr = 400.0, 1.0
    nu, ka = np.sqrt(Pr / Ra), 1.0 / np.sqrt(Ra * Pr)
    ev = lambda fn, t: np.broadcast_to(np.asarray(fn(m.x, m.y, m.z, t, nu, ka), dtype=np.float64), m.x.shape).copy()
    errs = []
    for dt in (0.02, 0.01, 0.005):
        S = Bq.Boussinesq(P, m.x, m.y, m.z, Ra=Ra, Pr=Pr, dt=dt, tags_u=0b10, tags_T=0b10, rtol=1e-12)
        S.u = [ev(c, 0.0) for c in U]; S.th = ev(TH, 0.0)
        nsteps = int(round(0.2 / dt))
        for s in range(nsteps):
            S.step(f=[ev(c, s * dt) for c in F])
        t1 = nsteps * dt
        eu = max(np.abs(S.u[c] - ev(U[c], t1)).max() for c in range(3))
        et = np.abs(S.th - ev(TH, t1)).max()
        errs.append((eu, et))
    (eu0, et0), (eu1, et1), (eu2, et2) = errs
    assert eu2 < 2e-4 and et2 < 2e-4
    assert 3.0 < eu1 / eu2 < 5.5 and 3.0 < et1 / et2 < 5.5, errs
