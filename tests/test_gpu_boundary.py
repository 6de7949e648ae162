"""GPU tests of the boundary's less-travelled paths (include/semb200.h): the semb_allocator callback, the error
returns SEMB_EBREAKDOWN and SEMB_EMATCH, strided fields in the consumer, the p.Ap block reduction at block sizes that
are not a multiple of the warp size, and the bounded Jacobi-diagonal cache.
"""
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


def test_allocator_callback_owns_every_library_buffer(torch_cuda, semb, orc, xi_of):
    """semb_allocator (include/semb200.h): with a torch-backed allocator the library allocates NOTHING outside torch's
    pool -- the device's free memory moves only by what torch reserved -- and every buffer is returned at destroy."""
    torch = torch_cuda
    m, prm = I.config_mesh(2, xi_of, small=True)
    x, y, z = dev(torch, m.x), dev(torch, m.y), dev(torch, m.z)
    P = orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam=0.0, dirichlet_tags=0b10)
    b = P.assemble_rhs(I.divergence_source(m, 5))
    bd = dev(torch, b)
    # first a handle WITHOUT the callback: loads the library's kernels (module memory) and shows the counter-case
    G0 = semb.Mesh(m.E, m.N, x, y, z, m.face_tag, m.period)
    xs = torch.zeros(m.n, dtype=torch.float64, device="cuda")
    G0.pcg_solve(bd, xs, tags=0b10, precond=3, mg_fp32=True, maxit=3)
    G0.pcg_solve(bd, xs, tags=0b10, precond=2, maxit=3)
    G0.close()
    torch.cuda.synchronize()
    A = semb.TorchAllocator()
    free0, res0 = torch.cuda.mem_get_info()[0], torch.cuda.memory_reserved()
    G = semb.Mesh(m.E, m.N, x, y, z, m.face_tag, m.period, allocator=A)
    assert A.calls > 10 and len(A.live) > 5
    for kw in (dict(precond=1), dict(precond=2), dict(precond=3), dict(precond=3, mg_fp32=True)):
        xs.zero_()
        r = G.pcg_solve(bd, xs, tags=0b10, rtol=1e-10, **kw)
        assert r["status"] == 0
    ro = P.pcg(b, precond=1, rtol=1e-10)
    assert normwise(xs.cpu().numpy(), ro["x"]) <= 2e-7
    torch.cuda.synchronize()
    free1, res1 = torch.cuda.mem_get_info()[0], torch.cuda.memory_reserved()
    assert res1 > res0                                              # the library's memory sits in torch's pool ...
    assert free0 - free1 == res1 - res0, (free0 - free1, res1 - res0)   # ... and nowhere else
    peak = A.peak_bytes
    G.close()
    assert len(A.live) == 0 and peak > 7 * 8 * m.n                  # everything returned; at least the factors were ours


def test_breakdown_is_reported(torch_cuda, semb, xi_of):
    """SEMB_EBREAKDOWN: lambda < 0 large enough makes D^T G D + lambda B indefinite, p.Ap <= 0 in the first iteration."""
    torch = torch_cuda
    m = I.box_mesh(3, 3, 3, 4, xi_of(4))
    G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    try:
        f = dev(torch, I.uniform(3, m.n))
        b = torch.empty_like(f)
        G.assemble_rhs(f, b, 0)
        x = torch.zeros_like(b)
        with pytest.raises(semb.SembError) as ei:
            G.pcg_solve(b, x, lam=-1e6, tags=0, precond=0, rtol=1e-10, maxit=50)
        assert ei.value.code == -5
        r = G.pcg_solve(b, x, lam=+1e6, tags=0, precond=0, rtol=1e-10, maxit=500)      # the handle stays usable
        assert r["status"] == 0
    finally:
        G.close()


def test_matching_that_is_not_an_equivalence_is_reported(torch_cuda, semb, orc, xi_of):
    """SEMB_EMATCH (reading R17): three copies of a node at 0, +0.7 tol, +1.4 tol match pairwise in a chain but the
    outer two do not -- neither the oracle nor the library may number that silently."""
    torch = torch_cuda
    N = 2
    m = I.box_mesh(2, 2, 1, N, xi_of(N))
    tol = 1e-8 * orc.min_spacing(m.E, N, m.x, m.y, m.z)
    x = m.x.copy()
    Np = (N + 1) ** 3
    centre = np.isclose(m.x, 0.5) & np.isclose(m.y, 0.5)             # the edge shared by all four elements
    for e, shift in ((1, 0.7 * tol), (2, 1.4 * tol)):
        sel = np.zeros(m.n, dtype=bool); sel[e * Np:(e + 1) * Np] = True
        x[sel & centre] += shift
    with pytest.raises(ValueError):
        orc.numbering(m.E, N, x, m.y, m.z, m.period, tol=tol)
    with pytest.raises(semb.SembError) as ei:
        semb.Mesh(m.E, N, dev(torch, x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    assert ei.value.code == -6
    G = semb.Mesh(m.E, N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)   # unperturbed: fine
    G.close()


def test_consumer_with_strided_field(torch_cuda, semb, orc):
    """semb_field_minmax_hist on a descriptor with stride != 1 (sub-fields are handed over as base
    pointer + offset / stride): element i is ptr[i * stride]."""
    torch = torch_cuda
    n, stride = 100003, 3
    v = I.uniform(77, n * stride)
    vd = dev(torch, v)
    d = semb.FieldDesc(b"strided", vd.data_ptr() + 8, 1, 1, n - 1, stride, 0, 0.0)      # starts at element 1
    mm = torch.zeros(2, dtype=torch.float64, device="cuda"); hist = torch.zeros(100, dtype=torch.int64, device="cuda")
    ref = v[1::stride][:n - 1]
    for lo, hi in ((-1.0, 1.0), (0.0, 0.0)):
        semb.field_minmax_hist(d, 100, lo, hi, mm, hist)
        mn, mx, h = orc.minmax_hist(ref, 100, lo if lo < hi else ref.min(), hi if lo < hi else ref.max())
        assert mm[0].item() == mn and mm[1].item() == mx
        assert np.array_equal(hist.cpu().numpy().astype(np.uint64), h)


@pytest.mark.parametrize("N", [2, 4, 5, 6, 8, 9, 10])
def test_fused_pAp_at_ragged_block_sizes(torch_cuda, semb, orc, xi_of, N):
    """k_axhelm_line runs with blockDim = (N+1)^2 x elements-per-block: 25, 36, 49, 81, 100, 121 threads are not a
    multiple of the warp size, so the block sum of p.Ap must not read lanes that were never launched.
    After exactly ONE PCG iteration from x0 = 0, x = alpha z0 with alpha = rho / p.Ap: x pins p.Ap to 1e-12."""
    torch = torch_cuda
    m = I.box_mesh(3, 2, 3, N, xi_of(N), deform=0.05)
    P = orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam=0.0, dirichlet_tags=0b10)
    G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    try:
        for lam in (0.0, 50.0):
            P.set_operator(lam, 0b10)
            b = P.assemble_rhs(I.uniform(5 + N, m.n))
            x = torch.zeros(m.n, dtype=torch.float64, device="cuda")
            rg = G.pcg_solve(dev(torch, b), x, lam=lam, tags=0b10, precond=1, rtol=0.0, maxit=1, hist_len=2)
            ro = P.pcg(b, precond=1, rtol=0.0, maxit=1, hist_len=2)
            assert rg["iters"] == ro["iters"] == 1
            z0 = P.dinv * b
            alpha_g = float(np.dot(x.cpu().numpy(), z0) / np.dot(z0, z0))
            alpha_o = float(np.dot(ro["x"], z0) / np.dot(z0, z0))
            assert abs(alpha_g - alpha_o) <= 1e-12 * abs(alpha_o), (N, lam, alpha_g, alpha_o)
            assert normwise(x.cpu().numpy(), ro["x"]) <= 1e-12
            assert abs(rg["hist"][1] - ro["hist"][1]) <= 1e-12 * ro["hist"][0]
    finally:
        G.close()


def test_jacobi_diagonal_cache_is_bounded(torch_cuda, semb, orc, xi_of):
    """A variable time step changes lambda = c / dt every step: the handle keeps the lambda-independent
    parts of the diagonal once and only the 8 most recently used (tags, lambda) diagonals, so device memory stops
    growing; every diagonal, fresh or recomputed after eviction, matches the oracle to 1e-12."""
    torch = torch_cuda
    m = I.box_mesh(6, 6, 6, 5, xi_of(5), deform=0.05)
    P = orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam=0.0, dirichlet_tags=0b10)
    G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    try:
        d = torch.empty(m.n, dtype=torch.float64, device="cuda")
        lams = [1.5 / (5e-4 * (1.0 + 0.01 * s)) for s in range(40)]
        free = []
        for lam in lams:
            G.jacobi_diag(d, lam, 0b10)
            torch.cuda.synchronize()
            free.append(torch.cuda.mem_get_info()[0])
        assert free[-1] == free[12], "device memory still growing after the cache filled"
        for lam in (lams[0], lams[-1], 0.0):                         # lams[0] was evicted long ago
            G.jacobi_diag(d, lam, 0b10)
            P.set_operator(lam, 0b10)
            assert normwise(d.cpu().numpy(), P.dinv) <= 1e-12
    finally:
        G.close()
