"""GPU parity of the p-multigrid V-cycle preconditioner (reading R19) against the oracle:
level sizes and numbering, transfer operators, one V-cycle, and full PCG solves, on the reduced members of the
box and O-grid families.  The Chebyshev bounds of every level are the oracle's (the estimator is compared
separately), so both sides apply the same polynomial."""
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


CASES = {
    "box5":   (lambda xi: I.box_mesh(3, 3, 4, 5, xi(5), deform=0.05, periodic=(True, False, False)), [5, 3, 1], 0.0, 0b10),
    "ogrid7": (lambda xi: I.config_mesh(2, xi, small=True)[0], [7, 3, 1], 0.0, 0b10),
    "ogrid9": (lambda xi: I.config_mesh(4, xi, small=True)[0], [9, 5, 3, 1], 0.0, 0b10),
    "box4_2": (lambda xi: I.box_mesh(2, 3, 2, 4, xi(4), deform=0.05), [4, 1], 10.0, 0),
}


@pytest.fixture(scope="module")
def cases(torch_cuda, semb, orc, xi_of):
    cache = {}

    def get(name):
        if name not in cache:
            mk, orders, lam, tags = CASES[name]
            m = mk(xi_of)
            mg = orc.Multigrid(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam, tags, orders, k_smooth=2, k_coarse=4)
            G = semb.Mesh(m.E, m.N, dev(torch_cuda, m.x), dev(torch_cuda, m.y), dev(torch_cuda, m.z), m.face_tag, m.period)
            cache[name] = (m, mg, G, orders, lam, tags)
        return cache[name]
    yield get
    for c in cache.values():
        c[2].close()


def cont(orc, P, seed):
    return P.mask * orc.gs(P.gid, P.n_unique, P.invmult * I.uniform(seed, P.n))


@pytest.mark.parametrize("name", list(CASES))
def test_levels_and_transfer(torch_cuda, cases, orc, name):
    torch = torch_cuda
    m, mg, G, orders, lam, tags = cases(name)
    for l, P in enumerate(mg.levels):
        assert G.mg_level_size(l, lam, tags, orders) == P.n
    for l in range(len(orders) - 1):
        Pf, Pc = mg.levels[l], mg.levels[l + 1]
        vc = cont(orc, Pc, 40 + l)
        out = torch.empty(Pf.n, dtype=torch.float64, device="cuda")
        G.mg_transfer(l, False, dev(torch, vc), out, lam, tags, orders)
        assert normwise(out.cpu().numpy(), mg.prolong(l, vc)) <= 1e-13
        rf = cont(orc, Pf, 50 + l)
        outc = torch.empty(Pc.n, dtype=torch.float64, device="cuda")
        G.mg_transfer(l, True, dev(torch, rf), outc, lam, tags, orders)
        assert normwise(outc.cpu().numpy(), mg.restrict(l, rf)) <= 1e-13


@pytest.mark.parametrize("name", list(CASES))
def test_vcycle(torch_cuda, cases, orc, name):
    torch = torch_cuda
    m, mg, G, orders, lam, tags = cases(name)
    P = mg.levels[0]
    r = cont(orc, P, 60)
    z = torch.empty(P.n, dtype=torch.float64, device="cuda")
    used = G.mg_vcycle(dev(torch, r), z, lam, tags, orders, 2, 4, mg.lmax, mg_coarse_frac=0.1)
    assert np.allclose(used, mg.lmax, rtol=0, atol=0)
    ref = mg.vcycle(r)
    assert normwise(z.cpu().numpy(), ref) <= 1e-11
    assert np.all(z.cpu().numpy()[P.mask == 0] == 0)
    # the library's own estimate of the bounds: same estimator, same start vector.  On a level with a few dozen
    # unknowns the 10-step Krylov space is nearly exhausted and the last Ritz value is rounding-sensitive (1e-4).
    used2 = G.mg_vcycle(dev(torch, r), z, lam, tags, orders, 2, 4, None, mg_coarse_frac=0.1)
    assert np.allclose(used2, mg.lmax, rtol=1e-3, atol=0)
    assert np.allclose(used2[0], mg.lmax[0], rtol=1e-6, atol=0)


@pytest.mark.parametrize("name", list(CASES))
def test_pmg_pcg(torch_cuda, cases, orc, name):
    torch = torch_cuda
    m, mg, G, orders, lam, tags = cases(name)
    P = mg.levels[0]
    b = P.assemble_rhs(I.divergence_source(m, I.seed_for(2, 70)))
    ro = mg.pcg(b, rtol=1e-10, hist_len=300)
    x = torch.zeros(P.n, dtype=torch.float64, device="cuda")
    rg = G.pcg_solve(dev(torch, b), x, lam=lam, tags=tags, precond=3, rtol=1e-10, hist_len=300, check_every=3,
                     mg_orders=orders, mg_smooth=2, mg_coarse=4, mg_lmax=mg.lmax, mg_coarse_frac=0.1)
    assert ro["status"] == 0 and rg["status"] == 0
    assert abs(rg["iters"] - ro["iters"]) <= 1, (rg["iters"], ro["iters"])
    xg = x.cpu().numpy()
    assert normwise(xg, ro["x"]) <= 1e-8
    res = b - P.apply_A(xg)
    assert np.sqrt(P.dot(res, res)) <= 2e-10 * np.sqrt(P.dot(b, b))
    k = min(10, len(ro["hist"]), len(rg["hist"]))
    assert np.allclose(rg["hist"][:k], ro["hist"][:k], rtol=1e-8, atol=0)
    # far fewer iterations than Jacobi on the same system
    xj = torch.zeros_like(x)
    rj = G.pcg_solve(dev(torch, b), xj, lam=lam, tags=tags, precond=1, rtol=1e-10)
    assert rg["iters"] < rj["iters"]
    assert normwise(xg, xj.cpu().numpy()) <= 1e-7


def test_default_hierarchy_and_bad_orders(torch_cuda, cases, orc):
    torch = torch_cuda
    m, mg, G, orders, lam, tags = cases("ogrid7")
    P = mg.levels[0]
    b = P.assemble_rhs(I.divergence_source(m, 3))
    x = torch.zeros(P.n, dtype=torch.float64, device="cuda")
    rg = G.pcg_solve(dev(torch, b), x, lam=lam, tags=tags, precond=3)           # defaults: 7, 3, 1; degrees 1 and 32 on [0.01, 1]; estimated bounds
    assert rg["status"] == 0
    res = b - P.apply_A(x.cpu().numpy())
    assert np.sqrt(P.dot(res, res)) <= 2e-10 * np.sqrt(P.dot(b, b))
    with pytest.raises(Exception):
        G.pcg_solve(dev(torch, b), x, lam=lam, tags=tags, precond=3, mg_orders=[7, 7, 1])
    with pytest.raises(Exception):
        G.pcg_solve(dev(torch, b), x, lam=lam, tags=tags, precond=3, mg_orders=[5, 3, 1])


def test_fourth_kind_smoother(torch_cuda, cases, orc):
    """mg_smoother_kind = 4: the fourth-kind Chebyshev polynomial of PAPER.md:L102 in every smoother of the cycle."""
    torch = torch_cuda
    m, mg1, G, orders, lam, tags = cases("ogrid7")
    mg = orc.Multigrid(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam, tags, orders, k_smooth=2, k_coarse=4,
                       lmax=mg1.lmax, kind=4)
    P = mg.levels[0]
    r = cont(orc, P, 61)
    z = torch.empty(P.n, dtype=torch.float64, device="cuda")
    G.mg_vcycle(dev(torch, r), z, lam, tags, orders, 2, 4, mg.lmax, mg_kind=4, mg_coarse_frac=0.1)
    assert normwise(z.cpu().numpy(), mg.vcycle(r)) <= 1e-11
    assert normwise(z.cpu().numpy(), mg1.vcycle(r)) > 1e-3           # and it is a different polynomial than the first kind
    b = P.assemble_rhs(I.divergence_source(m, I.seed_for(2, 71)))
    ro = mg.pcg(b, rtol=1e-10)
    x = torch.zeros(P.n, dtype=torch.float64, device="cuda")
    rg = G.pcg_solve(dev(torch, b), x, lam=lam, tags=tags, precond=3, rtol=1e-10, mg_orders=orders, mg_smooth=2, mg_coarse=4,
                     mg_lmax=mg.lmax, mg_kind=4, mg_coarse_frac=0.1)
    assert ro["status"] == 0 and rg["status"] == 0 and abs(rg["iters"] - ro["iters"]) <= 1
    assert normwise(x.cpu().numpy(), ro["x"]) <= 1e-8


def test_coarse_level_as_chebyshev_solver(torch_cuda, cases, orc):
    """mg_coarse_lmin_frac / a high mg_coarse_degree: the last level's first-kind polynomial on [frac, 1] lmax."""
    torch = torch_cuda
    m, mg1, G, orders, lam, tags = cases("box5")
    mg = orc.Multigrid(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam, tags, orders, k_smooth=1, k_coarse=24,
                       lmax=mg1.lmax, coarse_frac=0.01)
    P = mg.levels[0]
    r = cont(orc, P, 62)
    z = torch.empty(P.n, dtype=torch.float64, device="cuda")
    G.mg_vcycle(dev(torch, r), z, lam, tags, orders, 1, 24, mg.lmax, mg_coarse_frac=0.01)
    assert normwise(z.cpu().numpy(), mg.vcycle(r)) <= 1e-11
    b = P.assemble_rhs(I.divergence_source(m, I.seed_for(2, 72)))
    ro = mg.pcg(b, rtol=1e-10)
    x = torch.zeros(P.n, dtype=torch.float64, device="cuda")
    rg = G.pcg_solve(dev(torch, b), x, lam=lam, tags=tags, precond=3, rtol=1e-10, mg_orders=orders, mg_smooth=1, mg_coarse=24,
                     mg_lmax=mg.lmax, mg_coarse_frac=0.01)
    assert ro["status"] == 0 and rg["status"] == 0 and abs(rg["iters"] - ro["iters"]) <= 1
    assert normwise(x.cpu().numpy(), ro["x"]) <= 1e-8
    with pytest.raises(Exception):
        G.pcg_solve(dev(torch, b), x, lam=lam, tags=tags, precond=3, mg_orders=orders, mg_coarse=65)


@pytest.mark.parametrize("precond", [1, 3])
def test_all_neumann_pressure_zero_mean(torch_cuda, semb, orc, xi_of, precond):
    """null_mean (R20): lambda = 0, no Dirichlet node -- the closed-cell pressure problem (PAPER.md:L238, L266:
    no-slip walls all around).  Inconsistent right-hand side in, zero-mean solution of A x = b - mean(b) out."""
    torch = torch_cuda
    m = I.box_mesh(4, 3, 3, 5, xi_of(5), deform=0.05, zstretch=2.0)
    orders = [5, 3, 1]
    mg = orc.Multigrid(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, 0.0, 0, orders, k_smooth=1, k_coarse=8, coarse_frac=0.05)
    P = mg.levels[0]
    b = P.assemble_rhs(I.divergence_source(m, 9) + 0.3)
    assert abs(P.mean(b)) > 1e-6
    G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    try:
        x = torch.zeros(P.n, dtype=torch.float64, device="cuda")
        if precond == 1:
            ro = P.pcg(b, precond=1, rtol=1e-10, null_mean=True)
            rg = G.pcg_solve(dev(torch, b), x, lam=0.0, tags=0, precond=1, rtol=1e-10, null_mean=True)
        else:
            ro = mg.pcg(b, rtol=1e-10, null_mean=True)
            rg = G.pcg_solve(dev(torch, b), x, lam=0.0, tags=0, precond=3, rtol=1e-10, null_mean=True, mg_orders=orders,
                             mg_smooth=1, mg_coarse=8, mg_coarse_frac=0.05, mg_lmax=mg.lmax)
        assert ro["status"] == 0 and rg["status"] == 0 and abs(rg["iters"] - ro["iters"]) <= 1, (rg["iters"], ro["iters"])
        xg = x.cpu().numpy()
        assert normwise(xg, ro["x"]) <= 1e-8
        assert abs(P.mean(xg)) <= 1e-13 * np.abs(xg).max()
        res = (b - P.mean(b)) - P.apply_A(xg)
        assert np.sqrt(P.dot(res, res)) <= 2e-10 * np.sqrt(P.dot(b - P.mean(b), b - P.mean(b)))
        with pytest.raises(Exception):                      # Dirichlet nodes and null_mean exclude each other
            G.pcg_solve(dev(torch, b), x, lam=0.0, tags=0b10, precond=1, null_mean=True)
    finally:
        G.close()


@pytest.mark.parametrize("name", ["ogrid7", "box5"])
def test_fp32_storage_levels(torch_cuda, cases, orc, name):
    """mg_fp32 (R21): vectors and geometric factors of the levels stored in float, arithmetic in fp64.  The
    oracle rounds every vector of the cycle where it is stored; kernels that fuse two of the oracle's steps round once
    where the oracle rounds twice and the streaming kernels add in float, so the two cycles agree to a few float roundings
    (bar 2e-6 normwise, derived in DESIGN.md R21), while the PCG around the cycle stays fp64: same iteration count +-1, true
    residual below 2e-10.  The two PRECONDITIONERS differ at 1e-7, so the iterates part ways and the converged solutions
    agree only as well as two solves to rtol 1e-10 do: kappa(A) * 2 rtol ~ 1e-7 (bar 2e-7), not the 1e-8 of the fp64 path."""
    torch = torch_cuda
    m, mg64, G, orders, lam, tags = cases(name)
    mg32 = orc.Multigrid(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam, tags, orders, k_smooth=1, k_coarse=8,
                         coarse_frac=0.05, lmax=mg64.lmax, fp32=True)
    P = mg32.levels[0]
    r = cont(orc, P, 63)
    z = torch.empty(P.n, dtype=torch.float64, device="cuda")
    G.mg_vcycle(dev(torch, r), z, lam, tags, orders, 1, 8, mg32.lmax, mg_coarse_frac=0.05, mg_fp32=True)
    zg = z.cpu().numpy()
    assert normwise(zg, mg32.vcycle(r)) <= 2e-6
    assert np.array_equal(zg.astype(np.float32).astype(np.float64), zg)          # a stored float vector, widened
    assert np.all(zg[P.mask == 0] == 0)
    z64 = torch.empty_like(z)
    G.mg_vcycle(dev(torch, r), z64, lam, tags, orders, 1, 8, mg32.lmax, mg_coarse_frac=0.05)
    assert 1e-9 < normwise(zg, z64.cpu().numpy()) < 5e-6                          # it really ran in float storage
    b = P.assemble_rhs(I.divergence_source(m, I.seed_for(2, 73)))
    ro = mg32.pcg(b, rtol=1e-10)
    x = torch.zeros(P.n, dtype=torch.float64, device="cuda")
    rg = G.pcg_solve(dev(torch, b), x, lam=lam, tags=tags, precond=3, rtol=1e-10, mg_orders=orders, mg_smooth=1, mg_coarse=8,
                     mg_lmax=mg32.lmax, mg_coarse_frac=0.05, mg_fp32=True)
    assert ro["status"] == 0 and rg["status"] == 0 and abs(rg["iters"] - ro["iters"]) <= 1
    xg = x.cpu().numpy()
    assert normwise(xg, ro["x"]) <= 2e-7
    res = b - P.apply_A(xg)
    assert np.sqrt(P.dot(res, res)) <= 2e-10 * np.sqrt(P.dot(b, b))


@pytest.mark.parametrize("name", list(CASES))
def test_last_level_assembled_operator_against_matrix_free(torch_cuda, cases, orc, name):
    """csrc/coarse.cu: the order-1 last level works on its assembled operator (one launch per Chebyshev step).  The element matrices
    come from the level's own operator kernel, so the two forms are the same operator up to the order of the sums: V-cycles agree
    to rounding (fp64 levels 1e-12; FP32 levels: both within the 2e-6 of reading R21 of the oracle, and 2e-6 of each other), also
    after the Dirichlet tag set changes on the same hierarchy.  SEMB_MG_COARSE_ASSEMBLED=0 keeps the matrix-free form."""
    import os
    torch = torch_cuda
    m, mg, G, orders, lam, tags = cases(name)
    P = mg.levels[0]
    r = dev(torch, cont(orc, P, 61))
    out = {}
    for fp32 in (False, True):
        for env in ("0", "1"):
            os.environ["SEMB_MG_COARSE_ASSEMBLED"] = env
            try:
                z = torch.empty(P.n, dtype=torch.float64, device="cuda")
                G.mg_vcycle(r, z, lam, tags, orders, 2, 32, mg.lmax, mg_coarse_frac=0.02, mg_fp32=fp32)
                out[(fp32, env)] = z.cpu().numpy()
            finally:
                os.environ.pop("SEMB_MG_COARSE_ASSEMBLED", None)
    assert normwise(out[(False, "1")], out[(False, "0")]) <= 1e-12
    assert normwise(out[(True, "1")], out[(True, "0")]) <= 2e-6
    assert normwise(out[(True, "1")], out[(False, "1")]) <= 2e-6
    # another tag set on the same hierarchy (the level's free-node flags are rebuilt), then the first one again
    other = 0b110 if name.startswith("ogrid") else (0b10 if tags == 0 else 0)
    if other == 0 and lam == 0.0:
        return                                              # all-Neumann Poisson is singular: covered by the null_mean tests
    Po = orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam=lam, dirichlet_tags=other)
    ro = dev(torch, cont(orc, Po, 62))
    zz = {}
    for env in ("0", "1"):
        os.environ["SEMB_MG_COARSE_ASSEMBLED"] = env
        try:
            z = torch.empty(P.n, dtype=torch.float64, device="cuda")
            G.mg_vcycle(ro, z, lam, other, orders, 2, 32, None, mg_coarse_frac=0.02)
            zz[env] = z.cpu().numpy()
        finally:
            os.environ.pop("SEMB_MG_COARSE_ASSEMBLED", None)
    assert normwise(zz["1"], zz["0"]) <= 1e-12 and np.all(zz["1"][Po.mask == 0] == 0)
    z = torch.empty(P.n, dtype=torch.float64, device="cuda")
    G.mg_vcycle(r, z, lam, tags, orders, 2, 32, mg.lmax, mg_coarse_frac=0.02)
    assert np.array_equal(z.cpu().numpy(), out[(False, "1")])
