"""GPU parity of the Schwarz smoother and of the p-multigrid V-cycle that uses it (csrc/schwarz.cu, mg.cu; SURVEY.md §8 f-1;
PAPER.md:L102; reading R26) against oracle/schwarz.py.  The subdomain eigenproblems are solved by Jacobi rotations
on the device and by LAPACK in the oracle: S r agrees to 1e-11; the V-cycle and the solves follow."""
import numpy as np
import pytest

from paper_2501_13240_b200 import inputs as I

pytestmark = pytest.mark.gpu


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


MESHES = {
    "box_per_str_N5": (lambda xi: I.box_mesh(3, 3, 4, 5, xi(5), periodic=(True, True, False), zstretch=2.0), 0.0, 0b10),
    "box_def_N3":     (lambda xi: I.box_mesh(3, 2, 3, 3, xi(3), deform=0.05), 25.0, 0b110),
    "ogrid_N7":       (lambda xi: I.config_mesh(2, xi, small=True)[0], 0.0, 0b10),
    "ogrid_N9_helm":  (lambda xi: I.config_mesh(4, xi, small=True)[0], 3000.0, 0b110),
    "N2":             (lambda xi: I.box_mesh(4, 3, 3, 2, xi(2), deform=0.04), 0.0, 0b10),
    "N10":            (lambda xi: I.box_mesh(2, 2, 2, 10, xi(10), zstretch=1.5), 0.0, 0b10),
}


@pytest.mark.parametrize("name", list(MESHES))
def test_schwarz_apply(torch_cuda, semb, orc, xi_of, name):
    from oracle import schwarz as Sz
    torch = torch_cuda
    build, lam, tags = MESHES[name]
    m = build(xi_of)
    P = orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam=lam, dirichlet_tags=tags)
    S = Sz.Schwarz(P, m.x, m.y, m.z)
    G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    try:
        r = P.mask * orc.gs(P.gid, P.n_unique, P.invmult * I.uniform(4, m.n))
        out = torch.empty(m.n, dtype=torch.float64, device="cuda")
        G.schwarz_apply(dev(torch, r), out, lam=lam, tags=tags)
        ref = S.apply(r)
        assert normwise(out.cpu().numpy(), ref) <= 1e-11, name
    finally:
        G.close()


@pytest.mark.parametrize("name,orders", [("ogrid_N7", [7, 3, 1]), ("box_per_str_N5", [5, 2, 1])])
def test_vcycle_and_solve_with_schwarz_smoothing(torch_cuda, semb, orc, xi_of, name, orders):
    from oracle import schwarz as Sz
    torch = torch_cuda
    build, lam, tags = MESHES[name]
    m = build(xi_of)
    mg = orc.Multigrid(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam, tags, orders, k_smooth=1, k_coarse=16, kind=4)
    P = mg.levels[0]
    ms = Sz.MultigridSchwarz(mg, k_smooth=1)
    G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    try:
        r = P.mask * orc.gs(P.gid, P.n_unique, P.invmult * I.uniform(6, m.n))
        z = torch.empty(m.n, dtype=torch.float64, device="cuda")
        kw = dict(lam=lam, tags=tags, mg_orders=orders, mg_smooth=1, mg_coarse=16, mg_lmax=mg.lmax, mg_kind=4, mg_schwarz=True)
        G.mg_vcycle(dev(torch, r), z, **kw)
        ref = ms.vcycle(r)
        assert normwise(z.cpu().numpy(), ref) <= 1e-7, name              # lambda_max(S A) is estimated independently on both sides
        b = P.assemble_rhs(I.divergence_source(m, 5))
        ro = ms.pcg(b)
        rj = mg.pcg(b)
        x = torch.zeros(m.n, dtype=torch.float64, device="cuda")
        rg = G.pcg_solve(dev(torch, b), x, precond=3, rtol=1e-10, **kw)
        assert rg["status"] == 0 and abs(rg["iters"] - ro["iters"]) <= 1, (rg["iters"], ro["iters"])
        assert normwise(x.cpu().numpy(), ro["x"]) <= 1e-8
        res = b - P.apply_A(x.cpu().numpy())
        assert np.sqrt(P.dot(res, res)) <= 2e-10 * np.sqrt(P.dot(b, b))
        assert ro["iters"] < rj["iters"]                                  # fewer iterations than Chebyshev-Jacobi smoothing
        print(f"{name}: Chebyshev-Jacobi smoothing {rj['iters']} iterations, Chebyshev-Schwarz {ro['iters']} (GPU {rg['iters']})")
        # FP32-storage levels (R21): same count +- 2, fp64 true residual
        x.zero_()
        rf = G.pcg_solve(dev(torch, b), x, precond=3, rtol=1e-10, mg_fp32=True, **kw)
        assert rf["status"] == 0 and abs(rf["iters"] - ro["iters"]) <= 2, (rf["iters"], ro["iters"])
        res = b - P.apply_A(x.cpu().numpy())
        assert np.sqrt(P.dot(res, res)) <= 2e-10 * np.sqrt(P.dot(b, b))
    finally:
        G.close()
