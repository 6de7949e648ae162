"""Small meshes: the whole Jacobi-PCG solve as ONE persistent cooperative kernel (csrc/pcg_persist.cu) against the
launch-per-phase loop of csrc/pcg.cu (k_iter_small: two launches per iteration) and against the CPU oracle.

The two GPU paths add their partial sums in different (each fixed) orders, so they agree like two correct PCG runs do: the same
iteration count +-1, residual histories to 1e-9 relative while the residual is well above rounding, solutions to the bar of
test_pcg_mesh_families (1e-8 normwise).  SEMB_PCG_PERSIST=0 in the environment selects the loop (read at every solve)."""
import os

import numpy as np
import pytest

from paper_2501_13240_b200 import inputs as I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.fixture(scope="module")
def semb(torch_cuda):
    from paper_2501_13240_b200 import semb as S
    S.lib()
    return S


def normwise(a, ref):
    return np.abs(a - ref).max() / max(np.abs(ref).max(), 1e-300)


MESHES = {
    "cfg0":        lambda xi: I.config_mesh(0, xi)[0],                                                     # 64 elements, N = 7
    "box_per_str": lambda xi: I.box_mesh(3, 3, 4, 5, xi(5), periodic=(True, True, False), zstretch=2.5),   # periodic classes
    "ogrid7":      lambda xi: I.config_mesh(2, xi, small=True)[0],                                         # 3- and 5-valent edges
    "N3":          lambda xi: I.box_mesh(4, 3, 5, 3, xi(3), deform=0.05),                                  # 16 threads per block
    "N9":          lambda xi: I.box_mesh(2, 3, 2, 9, xi(9), deform=0.04),                                  # permuted line layout
}
CASES = [  # mesh, lambda, tags, precond, null_mean
    ("cfg0", 0.0, 0b10, 1, False), ("cfg0", 0.0, 0b10, 0, False), ("cfg0", 250.0, 0b10, 1, False),
    ("box_per_str", 0.0, 0b10, 1, False), ("box_per_str", 30.0, 0, 1, False), ("box_per_str", 0.0, 0, 1, True),
    ("ogrid7", 0.0, 0b10, 1, False), ("ogrid7", 100.0, 0b110, 1, False),
    ("N3", 0.0, 0b10, 1, False), ("N9", 0.0, 0b10, 1, False),
]


def solve(G, b, x, persist, **kw):
    os.environ["SEMB_PCG_PERSIST"] = "1" if persist else "0"
    try:
        return G.pcg_solve(b, x, **kw)
    finally:
        os.environ.pop("SEMB_PCG_PERSIST", None)


@pytest.fixture(scope="module")
def problems(torch_cuda, semb, orc, xi_of):
    cache = {}

    def get(name):
        if name not in cache:
            m = MESHES[name](xi_of)
            dev = lambda a: torch_cuda.from_numpy(np.ascontiguousarray(a)).cuda()
            cache[name] = (m, semb.Mesh(m.E, m.N, dev(m.x), dev(m.y), dev(m.z), m.face_tag, m.period))
        return cache[name]
    return get


@pytest.mark.parametrize("name,lam,tags,precond,null_mean", CASES)
def test_persistent_solve_against_loop_and_oracle(torch_cuda, orc, problems, name, lam, tags, precond, null_mean):
    torch = torch_cuda
    m, G = problems(name)
    P = orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam=lam, dirichlet_tags=tags)
    f = I.uniform(I.seed_for(8, 1), m.n)
    if null_mean:
        f = f - (f * P.geo[:, 6].ravel()).sum() / P.geo[:, 6].sum()               # compatible right-hand side
    b_ref = P.assemble_rhs(f)
    b = torch.from_numpy(b_ref).cuda()
    kw = dict(lam=lam, tags=tags, precond=precond, rtol=1e-10, maxit=3000, hist_len=64, null_mean=null_mean)
    out = {}
    for persist in (False, True):
        x = torch.zeros_like(b)
        st = solve(G, b, x, persist, **kw)
        assert st["status"] == 0
        out[persist] = (st, x.cpu().numpy())
    (s0, x0), (s1, x1) = out[False], out[True]
    assert s1["launches"] <= 6 and s0["launches"] >= 2 * s0["iters"]             # one launch for all iterations / two per iteration
    assert abs(s1["iters"] - s0["iters"]) <= 1
    assert normwise(x1, x0) <= 1e-8
    k = min(len(s0["hist"]), len(s1["hist"]), 20)
    assert np.allclose(s1["hist"][:k], s0["hist"][:k], rtol=1e-9, atol=0.0)
    ro = P.pcg(b_ref, precond=precond, rtol=1e-10, maxit=3000, null_mean=null_mean)   # the CPU oracle, as test_pcg_mesh_families does
    assert ro["status"] == 0 and abs(s1["iters"] - ro["iters"]) <= 1
    assert normwise(x1, ro["x"]) <= 1e-8
    # reproducible run to run: fixed summation orders
    x = torch.zeros_like(b)
    s2 = solve(G, b, x, True, **kw)
    assert s2["iters"] == s1["iters"] and np.array_equal(x.cpu().numpy(), x1) and np.array_equal(s2["hist"], s1["hist"])


def test_persistent_stop_rules_and_warm_start(torch_cuda, orc, problems):
    torch = torch_cuda
    m, G = problems("cfg0")
    P = orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam=0.0, dirichlet_tags=0b10)
    b_ref = P.assemble_rhs(I.uniform(I.seed_for(8, 2), m.n))
    b = torch.from_numpy(b_ref).cuda()
    res = {}
    for persist in (False, True):                                                 # maxit reached: status 1, exactly 7 iterations
        x = torch.zeros_like(b)
        st = solve(G, b, x, persist, tags=0b10, precond=1, rtol=1e-10, maxit=7)
        assert st["status"] == 1 and st["iters"] == 7
        res[persist] = (st["r_norm"], x.cpu().numpy())
    assert abs(res[True][0] - res[False][0]) <= 1e-10 * res[False][0] and normwise(res[True][1], res[False][1]) <= 1e-10
    ro = P.pcg(b_ref, precond=1, rtol=1e-10, maxit=7)
    assert normwise(res[True][1], ro["x"]) <= 1e-10
    # warm start from a continuous, masked guess: both paths take the same number of iterations to the same solution
    x_start = ro["x"]
    its = {}
    for persist in (False, True):
        x = torch.from_numpy(x_start.copy()).cuda()
        st = solve(G, b, x, persist, tags=0b10, precond=1, rtol=1e-10, maxit=3000, x0_is_zero=False)
        assert st["status"] == 0
        its[persist] = (st["iters"], x.cpu().numpy())
    assert abs(its[True][0] - its[False][0]) <= 1 and normwise(its[True][1], its[False][1]) <= 1e-8
    # zero right-hand side: converged before the first iteration, nothing launched that iterates
    x = torch.zeros_like(b)
    st = solve(G, torch.zeros_like(b), x, True, tags=0b10, precond=1, rtol=1e-10, maxit=50)
    assert st["status"] == 0 and st["iters"] == 0 and float(x.abs().max()) == 0.0


def test_persistent_breakdown_is_reported(torch_cuda, semb, problems):
    torch = torch_cuda
    m, G = problems("cfg0")
    b = torch.from_numpy(I.uniform(I.seed_for(8, 3), m.n)).cuda()
    G.gather_scatter(b); G.apply_mask(b, 0b10)
    for persist in (False, True):                                                 # indefinite operator: p.Ap <= 0
        x = torch.zeros_like(b)
        with pytest.raises(semb.SembError) as ei:
            solve(G, b, x, persist, lam=-1e6, tags=0b10, precond=0, rtol=1e-10, maxit=200)
        assert ei.value.code == -5
