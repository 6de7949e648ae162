"""GPU parity of the geometry representations of axhelm (reading R23): float-stored factors,
affine elements (7 constants per element), trilinear elements (24 coefficients per element, factors rebuilt per node).

The operator is the SAME one, so the oracle does not change: modes 2 and 3 are compared with the oracle's axhelm on the
oracle's own factors within max(1e-12, eps * kappa) (two evaluations of G from the same coordinates, reading R22: on these
meshes that is 1e-12), mode 1 with the oracle's axhelm applied to the float-rounded factors at 1e-12 (widening is exact).
"""
import numpy as np
import pytest

from paper_2501_13240_b200 import inputs as I

pytestmark = pytest.mark.gpu
TOL = 1e-12


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (there is no CPU fallback)")
    return torch


@pytest.fixture(scope="module")
def semb():
    from paper_2501_13240_b200 import semb as S
    S.lib()
    return S


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def normwise(a, ref):
    return np.abs(a - ref).max() / max(np.abs(ref).max(), 1e-300)


def r22_bound(orc, m):
    xi = orc.gll(m.N)[0]
    D = orc.dhat(m.N)
    cmax = max(np.abs(m.x).max(), np.abs(m.y).max(), np.abs(m.z).max())
    kappa = np.abs(D).sum(axis=1).max() * cmax * (xi[1] - xi[0]) / orc.min_spacing(m.E, m.N, m.x, m.y, m.z)
    return max(TOL, np.finfo(np.float64).eps * kappa)


def sheared(m):
    A = np.array([[1.0, 0.35, 0.2], [0.0, 0.9, 0.45], [0.15, 0.0, 1.2]])
    X = A @ np.stack([m.x, m.y, m.z])
    return I.Mesh(m.E, m.N, X[0].copy(), X[1].copy(), X[2].copy(), m.face_tag, m.period, m.name + "_sheared", m.meta)


MESHES = {
    # name: (builder, class)   class: "affine" | "trilinear" | "curved"
    "brick_stretched_N7": (lambda xi: I.box_mesh(4, 3, 5, 7, xi(7), periodic=(True, True, False), zstretch=2.5), "affine"),
    "sheared_N5":         (lambda xi: sheared(I.box_mesh(3, 4, 3, 5, xi(5))), "affine"),
    "brick_N3_ragged":    (lambda xi: I.box_mesh(3, 3, 3, 3, xi(3)), "affine"),
    "brick_N9":           (lambda xi: I.box_mesh(2, 3, 2, 9, xi(9), zstretch=2.0), "affine"),
    "jitter_N7":          (lambda xi: I.trilinear_box_mesh(4, 4, 3, 7, xi(7), jitter=0.2), "trilinear"),
    "jitter_N5_stretch":  (lambda xi: I.trilinear_box_mesh(3, 3, 6, 5, xi(5), jitter=0.15, zstretch=2.0), "trilinear"),
    "jitter_N9":          (lambda xi: I.trilinear_box_mesh(2, 2, 3, 9, xi(9), jitter=0.2), "trilinear"),
    "jitter_N2":          (lambda xi: I.trilinear_box_mesh(5, 3, 5, 2, xi(2), jitter=0.2), "trilinear"),
    "deformed_N7":        (lambda xi: I.box_mesh(3, 3, 3, 7, xi(7), deform=0.05), "curved"),
    "ogrid_N7":           (lambda xi: I.config_mesh(2, xi, small=True)[0], "curved"),
}


@pytest.mark.parametrize("name", list(MESHES))
def test_geometry_modes_apply_the_same_operator(torch_cuda, semb, orc, xi_of, name):
    torch = torch_cuda
    build, cls = MESHES[name]
    m = build(xi_of)
    P = orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam=0.0, dirichlet_tags=0)
    G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    try:
        u = I.uniform(I.seed_for(3, 1), m.n)
        ud = dev(torch, u); wd = torch.empty_like(ud)
        bound = r22_bound(orc, m)
        allowed = {"affine": (1, 2, 3), "trilinear": (1, 3), "curved": (1,)}[cls]
        for mode in (1, 2, 3):
            if mode not in allowed:
                with pytest.raises(semb.SembError) as ei:
                    G.set_geometry_mode(mode)
                assert ei.value.code == -4                                   # SEMB_EGEOM, mode unchanged:
                G.apply_axhelm(ud, wd, lam=0.0)
                assert normwise(wd.cpu().numpy(), orc.axhelm(m.E, m.N, P.geo, 0.0, u)) <= TOL
                continue
            dtri, daff = G.set_geometry_mode(mode)
            if mode >= 2:
                assert (daff if mode == 2 else dtri) <= 16 * np.finfo(np.float64).eps
            # mode 1: the LIBRARY's fp64 factors rounded to float (a double at a float rounding boundary would otherwise flip
            # with the 1e-13 difference between the two evaluations of G, reading R22, and show as 6e-8 in that factor)
            geo_ref = P.geo if mode >= 2 else np.ascontiguousarray(G.geo_host().astype(np.float32).astype(np.float64))
            for lam in (0.0, 1e3):
                G.apply_axhelm(ud, wd, lam=lam)
                ref = orc.axhelm(m.E, m.N, geo_ref, lam, u)
                err = normwise(wd.cpu().numpy(), ref)
                assert err <= (bound if mode >= 2 else TOL), (name, mode, lam, err)
            # batched fields go through the same kernels
            U3 = I.uniform(5, 3 * m.n); U3d = dev(torch, U3); W3d = torch.empty_like(U3d)
            G.apply_axhelm(U3d, W3d, lam=2.0, nfields=3)
            W3 = W3d.cpu().numpy()
            for f in range(3):
                assert normwise(W3[f * m.n:(f + 1) * m.n], orc.axhelm(m.E, m.N, geo_ref, 2.0, U3[f * m.n:(f + 1) * m.n])) <= (bound if mode >= 2 else TOL)
            G.set_geometry_mode(0)
        if cls == "trilinear":
            assert G.set_geometry_mode(3)[1] > 1e-3                           # measurably not affine
            G.set_geometry_mode(0)
        # coefficient fields need the stored factors
        G.set_geometry_mode(1)
        with pytest.raises(semb.SembError):
            G.apply_axhelm(ud, wd, lam0=ud)
        G.set_geometry_mode(0)
    finally:
        G.close()


@pytest.mark.parametrize("name,mode", [("brick_stretched_N7", 2), ("brick_stretched_N7", 3), ("jitter_N7", 3), ("deformed_N7", 1), ("jitter_N9", 3), ("brick_N9", 2)])
@pytest.mark.parametrize("precond", [1, 2, 3])
def test_solves_in_every_geometry_mode(torch_cuda, semb, orc, xi_of, name, mode, precond):
    """The solver's fused operator launches read the selected representation too: same iteration counts (+-1) and the same
    solution as the oracle's solve with its stored fp64 factors; mode 1 perturbs the operator by 6e-8, so its solution is
    compared with the oracle's solve on the float-rounded factors."""
    torch = torch_cuda
    m = MESHES[name][0](xi_of)
    lam = 0.0 if precond != 2 else 30.0
    P = orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam=lam, dirichlet_tags=0b10)
    G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    if mode == 1:
        P.geo[...] = G.geo_host().astype(np.float32).astype(np.float64)
        P.set_operator(lam, 0b10)
    try:
        G.set_geometry_mode(mode)
        b = P.assemble_rhs(I.divergence_source(m, 5))
        x = torch.zeros(m.n, dtype=torch.float64, device="cuda")
        if precond == 3:
            rg = G.pcg_solve(dev(torch, b), x, lam=lam, tags=0b10, precond=3, rtol=1e-10)
            ro = P.pcg(b, precond=1, rtol=1e-10)
            assert rg["status"] == 0 and rg["iters"] < ro["iters"]
            tol_x = 2e-7 if mode == 1 else 1e-8        # mode 1: the levels' diagonal comes from the unrounded factors (a preconditioner detail)
        else:
            lmax = P.lanczos_lmax(b, 10) if precond == 2 else 0.0
            rg = G.pcg_solve(dev(torch, b), x, lam=lam, tags=0b10, precond=precond, cheb_degree=2, cheb_lmax=lmax, rtol=1e-10)
            ro = P.pcg(b, precond=precond, cheb_k=2, lmax=lmax, rtol=1e-10)
            assert rg["status"] == 0 and abs(rg["iters"] - ro["iters"]) <= 1, (rg["iters"], ro["iters"])
            tol_x = 1e-8 if mode != 1 else 1e-6        # mode 1: dinv is built from the unrounded factors, the oracle's from the rounded ones
        assert normwise(x.cpu().numpy(), ro["x"]) <= tol_x
        r = b - P.apply_A(x.cpu().numpy())
        assert np.sqrt(P.dot(r, r)) <= 2e-10 * np.sqrt(P.dot(b, b))           # oracle-verified true residual
    finally:
        G.close()


def test_fullsize_affine_and_trilinear_boxes(torch_cuda, semb, orc, xi_of):
    """64^3 elements, N = 7 (the bench configuration of the geometry-mode section): sampled elements against the oracle."""
    torch = torch_cuda
    ne, N, Np = 64, 7, 512
    for kind, mode in (("affine", 2), ("affine", 3), ("trilinear", 3)):
        m = (I.box_mesh(ne, ne, ne, N, semb.gll(N)[0], zstretch=2.0) if kind == "affine"
             else I.trilinear_box_mesh(ne, ne, ne, N, semb.gll(N)[0], jitter=0.2, zstretch=2.0))
        G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
        try:
            G.set_geometry_mode(mode)
            u = I.uniform(I.seed_for(3, 1), m.n)
            ud = dev(torch, u); wd = torch.empty_like(ud)
            rng = np.random.default_rng(11)
            sample = np.unique(np.concatenate([[0, 1, ne - 1, m.E // 2, m.E - 1], rng.integers(0, m.E, 40)]))
            idx = (sample[:, None] * Np + np.arange(Np)[None, :]).reshape(-1)
            geo_s = orc.geo_factors(len(sample), N, m.x[idx], m.y[idx], m.z[idx])
            ms = I.Mesh(len(sample), N, m.x[idx], m.y[idx], m.z[idx], None, [0, 0, 0], "sample")
            bound = r22_bound(orc, ms)
            for lam in (0.0, 1e4):
                G.apply_axhelm(ud, wd, lam=lam)
                w = wd.cpu().numpy()
                err = normwise(w[idx], orc.axhelm(len(sample), N, geo_s, lam, u[idx]))
                print(f"fullsize {kind} mode {mode} lam {lam}: {err:.2e} (bound {bound:.1e})")
                assert err <= bound and np.isfinite(w).all()
        finally:
            G.close()
        del m


def test_geometry_modes_on_the_smallest_meshes(torch_cuda, semb, orc, xi_of):
    """Degenerate sizes: one element, order 1 (8 nodes) and order 2, every representation, ragged packed blocks (32 / 14 elements per block)."""
    torch = torch_cuda
    for N, ne in ((1, (1, 1, 1)), (1, (5, 3, 7)), (2, (1, 1, 1)), (2, (3, 5, 3))):
        m = I.box_mesh(*ne, N, xi_of(N), zstretch=1.5)
        P = orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period)
        G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
        try:
            u = I.uniform(9, m.n); ud = dev(torch, u); wd = torch.empty_like(ud)
            for mode in (0, 1, 2, 3):
                G.set_geometry_mode(mode)
                geo_ref = P.geo if mode != 1 else np.ascontiguousarray(G.geo_host().astype(np.float32).astype(np.float64))
                for lam in (0.0, 7.0):
                    G.apply_axhelm(ud, wd, lam=lam)
                    assert normwise(wd.cpu().numpy(), orc.axhelm(m.E, m.N, geo_ref, lam, u)) <= TOL, (N, ne, mode, lam)
        finally:
            G.close()
