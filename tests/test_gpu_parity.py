"""GPU parity: every C-ABI call of libsemb200.so against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json:north_star): integer connectivity and numbering bit-exact;
axhelm / gather-scatter / diagonal within 1e-12 normwise (max|gpu - ref| <= 1e-12 max|ref|); full solves
within +-1 iteration, final relative residual <= 1e-10, solution within 1e-8 normwise.
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


def gpu_mesh(torch, semb, m):
    return semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)


def oracle_problem(orc, m, lam=0.0, tags=0):
    return orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period, lam=lam, dirichlet_tags=tags)


def normwise(a, ref):
    return np.abs(a - ref).max() / max(np.abs(ref).max(), 1e-300)


MESHES = {
    "cfg0":        lambda xi: I.config_mesh(0, xi)[0],
    "box_def":     lambda xi: I.box_mesh(5, 4, 3, 7, xi(7), deform=0.05),
    "box_per_str": lambda xi: I.box_mesh(3, 3, 4, 5, xi(5), periodic=(True, True, False), zstretch=2.5),
    "ogrid7":      lambda xi: I.config_mesh(2, xi, small=True)[0],
    "ogrid9":      lambda xi: I.config_mesh(4, xi, small=True)[0],
    "one_elem":    lambda xi: I.box_mesh(1, 1, 1, 4, xi(4)),
    "N1":          lambda xi: I.box_mesh(3, 2, 2, 1, xi(1), deform=0.05),
    "N10":         lambda xi: I.box_mesh(2, 2, 2, 10, xi(10), deform=0.05),
    # small orders pack several elements into one block (32 / 14 / 8): element counts that leave a ragged last block
    "N1_ragged":   lambda xi: I.box_mesh(5, 3, 5, 1, xi(1), deform=0.05),
    "N2_ragged":   lambda xi: I.box_mesh(3, 5, 3, 2, xi(2), deform=0.05),
    "N3_ragged":   lambda xi: I.box_mesh(3, 3, 3, 3, xi(3), deform=0.05),
}


@pytest.fixture(scope="module")
def cases(torch_cuda, semb, orc, xi_of):
    cache = {}

    def get(name):
        if name not in cache:
            m = MESHES[name](xi_of)
            cache[name] = (m, oracle_problem(orc, m), gpu_mesh(torch_cuda, semb, m))
        return cache[name]
    yield get
    for _, _, g in cache.values():
        g.close()


# ------------------------------------------------------------------------------------------ setup
@pytest.mark.parametrize("name", list(MESHES))
def test_numbering_bit_exact(cases, name):
    m, P, G = cases(name)
    assert G.n_unique == P.n_unique
    assert np.array_equal(G.gid_host(), P.gid)                       # canonical first-touch ids, bit for bit
    # gather lists: classes with >= 2 copies, by gid, members ascending in l -- rebuilt here from the oracle's gid
    order = np.argsort(P.gid, kind="stable")
    counts = np.bincount(P.gid, minlength=P.n_unique)
    keep = counts[P.gid[order]] >= 2
    ids_ref = order[keep].astype(np.int32)
    off_ref = np.concatenate([[0], np.cumsum(counts[counts >= 2])]).astype(np.int32)
    off, ids = G.gs_lists_host()
    assert G.n_shared == ids_ref.size and G.n_gs == off_ref.size - 1
    assert np.array_equal(ids, ids_ref) and np.array_equal(off, off_ref)
    assert np.array_equal(G.invmult_host(), P.invmult)
    assert abs(G.info.tol - 1e-8 * __import__("oracle.semoracle", fromlist=["x"]).min_spacing(m.E, m.N, m.x, m.y, m.z)) <= 1e-20


@pytest.mark.parametrize("name", ["cfg0", "box_def", "ogrid7", "ogrid9", "N10"])
def test_geometric_factors(cases, name):
    m, P, G = cases(name)
    geo = G.geo_host()
    # the six G factors are one symmetric tensor: errors are measured against its largest entry (on affine
    # meshes the cross terms are pure rounding noise around 0, so a per-factor norm would compare noise with noise)
    scale = np.abs(P.geo[:, :6]).max()
    for g in range(6):
        assert np.abs(geo[:, g] - P.geo[:, g]).max() <= TOL * scale, f"factor {g}"
    assert normwise(geo[:, 6], P.geo[:, 6]) <= TOL


def test_caller_supplied_gid(torch_cuda, semb, orc, xi_of):
    m = I.box_mesh(3, 3, 2, 4, xi_of(4), periodic=(True, False, False), deform=0.03)
    P = oracle_problem(orc, m)
    labels = (P.gid.astype(np.int64) * 7919 % 1000003).astype(np.int32)      # arbitrary injective relabelling
    assert np.unique(labels).size == P.n_unique
    G = semb.Mesh(m.E, m.N, dev(torch_cuda, m.x), dev(torch_cuda, m.y), dev(torch_cuda, m.z), m.face_tag, m.period,
                  gid=dev(torch_cuda, labels))
    assert np.array_equal(G.gid_host(), P.gid)
    G.close()


def test_negative_jacobian_is_reported(torch_cuda, semb, xi_of):
    m = I.box_mesh(2, 2, 2, 3, xi_of(3))
    x = m.x.copy(); x[64:128] = -x[64:128]                                  # mirror element 1 -> J < 0
    with pytest.raises(semb.SembError) as ei:
        semb.Mesh(m.E, m.N, dev(torch_cuda, x), dev(torch_cuda, m.y), dev(torch_cuda, m.z), m.face_tag, m.period)
    assert ei.value.code == -4 and "element 1" in str(ei.value)


# ------------------------------------------------------------------------------------------ axhelm
@pytest.mark.parametrize("name", list(MESHES))
@pytest.mark.parametrize("lam", [0.0, 1e4])
def test_axhelm(torch_cuda, cases, orc, name, lam):
    m, P, G = cases(name)
    u = I.uniform(I.seed_for(0, 1), m.n)
    ref = orc.axhelm(m.E, m.N, P.geo, lam, u)
    w = torch_cuda.full((m.n,), np.nan, dtype=torch_cuda.float64, device="cuda")
    G.apply_axhelm(dev(torch_cuda, u), w, lam=lam)
    w = w.cpu().numpy()
    assert normwise(w, ref) <= TOL
    per_elem = np.abs((w - ref).reshape(m.E, -1)).max(1) / np.abs(ref.reshape(m.E, -1)).max(1)
    assert per_elem.max() <= TOL


@pytest.mark.parametrize("name", ["box_def", "N1_ragged", "N2_ragged", "N3_ragged"])
def test_axhelm_batched_and_variable_coefficients(torch_cuda, cases, orc, name):
    m, P, G = cases(name)
    U = np.stack([I.uniform(I.seed_for(1, 10 + f), m.n) for f in range(3)])
    W = torch_cuda.zeros((3, m.n), dtype=torch_cuda.float64, device="cuda")
    G.apply_axhelm(dev(torch_cuda, U), W, lam=1e4, nfields=3)
    for f in range(3):
        assert normwise(W[f].cpu().numpy(), orc.axhelm(m.E, m.N, P.geo, 1e4, U[f])) <= TOL
    lam0 = 1.0 + 0.5 * np.sin(2 * np.pi * m.x) * np.sin(2 * np.pi * m.y) * np.sin(2 * np.pi * m.z)
    lam1 = np.full(m.n, 1e4)
    w = torch_cuda.zeros(m.n, dtype=torch_cuda.float64, device="cuda")
    G.apply_axhelm(dev(torch_cuda, U[0]), w, lam=0.0, lam0=dev(torch_cuda, lam0), lam1=dev(torch_cuda, lam1))
    assert normwise(w.cpu().numpy(), orc.axhelm(m.E, m.N, P.geo, 0.0, U[0], lam0=lam0, lam1=lam1)) <= TOL


def test_axhelm_order9_persistent_blocks(torch_cuda, semb, orc, xi_of):
    """N = 9 stand-alone launches (and N = 7 launches on several fields) run k_axhelm_stage: persistent blocks (3 per SM on B200 = 444
    at N = 9) that walk over the elements blockIdx.x + i * gridDim.x, apply each to all fields, with the factors of their next element in
    flight (TMA into shared memory).  9 x 8 x 7 = 504 elements: a full round and a ragged one; then a single element (one block, no
    next element)."""
    for dims, nf, N in (((9, 8, 7), 2, 9), ((1, 1, 1), 1, 9), ((10, 10, 10), 3, 7), ((1, 1, 1), 2, 7)):
        # N = 7: several fields only (888 resident blocks: 1000 elements = one full round and a ragged one, all 3 fields per element)
        m = I.box_mesh(*dims, N, xi_of(N), deform=0.04)
        P, G = oracle_problem(orc, m), gpu_mesh(torch_cuda, semb, m)
        U = np.stack([I.uniform(I.seed_for(1, 40 + f), m.n) for f in range(nf)])
        for lam in (0.0, 1e4):
            W = torch_cuda.full((nf, m.n), np.nan, dtype=torch_cuda.float64, device="cuda")
            G.apply_axhelm(dev(torch_cuda, U), W, lam=lam, nfields=nf)
            for f in range(nf):
                ref = orc.axhelm(m.E, m.N, P.geo, lam, U[f])
                w = W[f].cpu().numpy()
                assert normwise(w, ref) <= TOL
                per_elem = np.abs((w - ref).reshape(m.E, -1)).max(1) / np.abs(ref.reshape(m.E, -1)).max(1)
                assert per_elem.max() <= TOL
        G.close()


def test_axhelm_host_entry_point(torch_cuda, cases, orc):
    m, P, G = cases("cfg0")
    u = I.uniform(3, m.n); w = np.zeros(m.n)
    G.apply_axhelm_host(u, w, lam=2.0)
    assert normwise(w, orc.axhelm(m.E, m.N, P.geo, 2.0, u)) <= TOL


# ------------------------------------------------------------------------------------------ gather-scatter, mask
@pytest.mark.parametrize("name", ["cfg0", "box_def", "box_per_str", "ogrid7", "ogrid9", "one_elem"])
def test_gather_scatter(torch_cuda, cases, orc, name):
    m, P, G = cases(name)
    vi = np.floor(I.uniform(7, m.n, -2.0 ** 19, 2.0 ** 19))                # integers sum exactly: bitwise parity
    w = dev(torch_cuda, vi)
    G.gather_scatter(w)
    assert np.array_equal(w.cpu().numpy(), orc.gs(P.gid, P.n_unique, vi))
    v = np.stack([I.uniform(8, m.n), I.uniform(9, m.n)])
    w = dev(torch_cuda, v)
    G.gather_scatter(w, nfields=2)
    for f in range(2):
        assert normwise(w[f].cpu().numpy(), orc.gs(P.gid, P.n_unique, v[f])) <= TOL
    ones = torch_cuda.ones(m.n, dtype=torch_cuda.float64, device="cuda")
    G.gather_scatter(ones)                                                 # QQ^T 1 = multiplicity
    assert np.array_equal(1.0 / ones.cpu().numpy(), P.invmult)


@pytest.mark.parametrize("name,tags", [("cfg0", 0b10), ("ogrid7", 0b10), ("ogrid7", 0b110), ("ogrid7", 0b100), ("box_def", 0)])
def test_mask_rhs_operator_diag(torch_cuda, cases, orc, name, tags):
    m, P0, G = cases(name)
    lam = 3000.0
    P = oracle_problem(orc, m, lam=lam, tags=tags)
    v = I.uniform(11, m.n)
    w = dev(torch_cuda, v)
    G.apply_mask(w, tags)
    assert np.array_equal(w.cpu().numpy(), v * P.mask)
    f = I.uniform(12, m.n)
    b = torch_cuda.zeros(m.n, dtype=torch_cuda.float64, device="cuda")
    G.assemble_rhs(dev(torch_cuda, f), b, tags)
    assert normwise(b.cpu().numpy(), P.assemble_rhs(f)) <= TOL
    vc = orc.gs(P.gid, P.n_unique, v * P.invmult)                          # continuous vector
    out = torch_cuda.zeros(m.n, dtype=torch_cuda.float64, device="cuda")
    G.apply_operator(dev(torch_cuda, vc), out, lam, tags)
    assert normwise(out.cpu().numpy(), P.apply_A(vc)) <= TOL
    dinv = torch_cuda.zeros(m.n, dtype=torch_cuda.float64, device="cuda")
    G.jacobi_diag(dinv, lam, tags)
    assert normwise(dinv.cpu().numpy(), P.dinv) <= TOL


# ------------------------------------------------------------------------------------------ solves
def _solve_both(torch_cuda, orc, m, G, lam, tags, precond, f, cheb_k=2, rtol=1e-10, x0=None, check_every=0):
    P = oracle_problem(orc, m, lam=lam, tags=tags)
    b = P.assemble_rhs(f)
    lmax = 0.0
    if precond == 2:
        lmax = P.lanczos_lmax(b, 10)
    ro = P.pcg(b, x0=x0, precond=precond, cheb_k=cheb_k, lmax=lmax, rtol=rtol, hist_len=4000)
    x = torch_cuda.zeros(m.n, dtype=torch_cuda.float64, device="cuda") if x0 is None else dev(torch_cuda, x0)
    rg = G.pcg_solve(dev(torch_cuda, b), x, lam=lam, tags=tags, precond=precond, cheb_degree=cheb_k, cheb_lmax=lmax,
                     rtol=rtol, x0_is_zero=x0 is None, hist_len=4000, check_every=check_every)
    xg = x.cpu().numpy()
    assert ro["status"] == 0 and rg["status"] == 0
    assert abs(rg["iters"] - ro["iters"]) <= 1
    assert normwise(xg, ro["x"]) <= 1e-8
    assert np.all(xg[P.mask == 0] == 0)
    # oracle-verified true residual of the GPU solution
    res = b - P.apply_A(xg)
    assert np.sqrt(P.dot(res, res)) <= 2e-10 * np.sqrt(P.dot(b, b))
    k = min(20, len(ro["hist"]), len(rg["hist"]))
    assert np.allclose(rg["hist"][:k], ro["hist"][:k], rtol=1e-9, atol=0)
    assert abs(rg["b_norm"] - np.sqrt(P.dot(b, b))) <= 1e-12 * rg["b_norm"]
    return ro, rg


@pytest.mark.parametrize("precond", [0, 1, 2])
def test_pcg_cfg0(torch_cuda, cases, orc, precond):
    """configs[0]: 4^3 affine cube, periodic x,y, Dirichlet z, f = 3 pi^2 sin sin sin, rtol 1e-10."""
    m, _, G = cases("cfg0")
    _, f = I.manufactured_sin(m)
    _solve_both(torch_cuda, orc, m, G, 0.0, 0b10, precond, f)


@pytest.mark.parametrize("name,lam,tags,precond", [
    ("N1_ragged", 0.0, 0b10, 1), ("N2_ragged", 5.0, 0b10, 2), ("N3_ragged", 0.0, 0b110, 1),
    ("box_def", 0.0, 0b110, 1), ("box_def", 1e4, 0, 1), ("ogrid7", 0.0, 0b10, 2), ("ogrid7", 0.0, 0b10, 1),
    ("ogrid9", 3000.0, 0b110, 1), ("ogrid9", 0.0, 0b10, 1), ("box_per_str", 0.0, 0b10, 2)])
def test_pcg_mesh_families(torch_cuda, cases, orc, name, lam, tags, precond):
    m, _, G = cases(name)
    f = I.divergence_source(m, I.seed_for(2, 20))
    _solve_both(torch_cuda, orc, m, G, lam, tags, precond, f, check_every=5)


def test_pcg_initial_guess_and_maxit(torch_cuda, cases, orc):
    m, _, G = cases("box_def")
    f = I.divergence_source(m, 77)
    ro, rg = _solve_both(torch_cuda, orc, m, G, 10.0, 0b10, 1, f)
    x0 = ro["x"] * (1.0 + 1e-3)                                            # continuous, masked start
    ro2, rg2 = _solve_both(torch_cuda, orc, m, G, 10.0, 0b10, 1, f, x0=x0)
    assert rg2["iters"] < rg["iters"]
    P = oracle_problem(orc, m, lam=10.0, tags=0b10)
    b = P.assemble_rhs(f)
    x = torch_cuda.zeros(m.n, dtype=torch_cuda.float64, device="cuda")
    r = G.pcg_solve(dev(torch_cuda, b), x, lam=10.0, tags=0b10, precond=1, maxit=7, hist_len=16, check_every=3)
    o = P.pcg(b, precond=1, maxit=7, hist_len=16)
    assert r["status"] == 1 and r["iters"] == 7 and o["iters"] == 7
    assert normwise(x.cpu().numpy(), o["x"]) <= 1e-10
    # zero right-hand side: converged at iteration 0
    x = torch_cuda.ones(m.n, dtype=torch_cuda.float64, device="cuda")
    r = G.pcg_solve(torch_cuda.zeros(m.n, dtype=torch_cuda.float64, device="cuda"), x, lam=10.0, tags=0b10)
    assert r["status"] == 0 and r["iters"] == 0 and float(x.abs().max()) == 0.0


def test_step_driver_cfg4_recipe(torch_cuda, cases, orc):
    """configs[4] on the reduced N = 9 O-grid (R12): per step one pressure Poisson solve (Dirichlet {1}) and
    three velocity ({1,2}) plus one temperature ({1}) Helmholtz solves with lambda = 1.5/dt = 3000, through ONE
    semb_step_solve call; right-hand sides b(s) = M QQ^T B(f + 0.1 rms(f) eta(s)); steps >= 2 start from the previous
    step's solution.  Every solve is compared with the oracle run on the same inputs (its own warm starts)."""
    torch = torch_cuda
    m, _, G = cases("ogrid9")
    lam_h = 3000.0
    kinds = [(0.0, 0b10), (lam_h, 0b110), (lam_h, 0b110), (lam_h, 0b110), (lam_h, 0b10)]
    probs = [oracle_problem(orc, m, lam=l, tags=t) for l, t in kinds]
    f0 = [I.divergence_source(m, I.seed_for(4, 30 + i)) for i in range(5)]
    xg = [torch.zeros(m.n, dtype=torch.float64, device="cuda") for _ in range(5)]
    xo = [None] * 5
    for step in range(3):
        bs = []
        for i, P in enumerate(probs):
            eta = I.uniform(I.seed_for(4, 100 * (step + 1) + i), m.n)
            f = f0[i] + 0.1 * np.sqrt(np.mean(f0[i] ** 2)) * eta
            bs.append(P.assemble_rhs(f))
        solves = [dict(b=dev(torch, bs[i]), x=xg[i], lam=kinds[i][0], tags=kinds[i][1], precond=1, rtol=1e-10,
                       x0_is_zero=(step == 0), check_every=7) for i in range(5)]
        rc, stats = G.step_solve(solves)
        assert rc == 0 and len(stats) == 5
        for i, P in enumerate(probs):
            ro = P.pcg(bs[i], x0=xo[i], precond=1, rtol=1e-10)
            xo[i] = ro["x"]
            assert ro["status"] == 0 and stats[i]["status"] == 0
            assert abs(stats[i]["iters"] - ro["iters"]) <= 1, (step, i, stats[i]["iters"], ro["iters"])
            assert normwise(xg[i].cpu().numpy(), ro["x"]) <= 1e-8
            assert stats[i]["r_norm"] <= 1e-10 * stats[i]["b_norm"]
    # an invalid item stops the sequence with its error
    bad = [dict(b=dev(torch, bs[0]), x=xg[0], precond=7)]
    with pytest.raises(Exception):
        G.step_solve(bad)


def test_cheb_jacobi_and_lmax(torch_cuda, cases, orc):
    m, _, G = cases("ogrid7")
    P = oracle_problem(orc, m, lam=0.0, tags=0b10)
    v0 = P.assemble_rhs(I.divergence_source(m, 5))
    lo = P.lanczos_lmax(v0, 10)
    lg = G.estimate_lmax(dev(torch_cuda, v0), 0.0, 0b10, steps=10)
    assert abs(lg - lo) <= 1e-6 * lo
    r = v0
    for k in (0, 1, 2, 3):
        z = torch_cuda.zeros(m.n, dtype=torch_cuda.float64, device="cuda")
        G.cheb_jacobi(dev(torch_cuda, r), z, 0.0, 0b10, k, lo)
        assert normwise(z.cpu().numpy(), P.cheb_jacobi(k, lo, r)) <= TOL


def test_pcg_estimates_lmax_itself(torch_cuda, cases, orc):
    m, _, G = cases("ogrid7")
    P = oracle_problem(orc, m, lam=0.0, tags=0b10)
    b = P.assemble_rhs(I.divergence_source(m, 6))
    x = torch_cuda.zeros(m.n, dtype=torch_cuda.float64, device="cuda")
    r = G.pcg_solve(dev(torch_cuda, b), x, tags=0b10, precond=2, cheb_degree=2, cheb_lmax=0.0)
    assert r["status"] == 0 and abs(r["lmax_used"] - P.lanczos_lmax(b, 10)) <= 1e-6 * r["lmax_used"]
    rj = G.pcg_solve(dev(torch_cuda, b), torch_cuda.zeros_like(x), tags=0b10, precond=1)
    assert r["iters"] < rj["iters"]                                        # Chebyshev cuts the iteration count


# ------------------------------------------------------------------------------------------ export
def test_export_is_zero_copy_and_consumer_is_exact(torch_cuda, semb, cases, orc):
    torch = torch_cuda
    m, _, G = cases("box_def")
    T = (1.0 - m.z) + 0.05 * I.uniform(31, m.n)
    v = [I.uniform(32 + c, m.n) for c in range(3)]
    dT = dev(torch, T); dv = [dev(torch, c) for c in v]
    G.publish_field("temperature", dT)
    for name, t in zip(("velocity_x", "velocity_y", "velocity_z"), dv):
        G.publish_field(name, t)
    G.export_field("velocity_magnitude")             # a consumer asks for the derived field: publish_state keeps it current from now on
    # one untimed pass first: the driver loads kernel images lazily and grows the context's local-memory pool on the first launch
    # of a kernel with a stack frame -- context growth, not an allocation of the call
    warm_mm = torch.zeros(2, dtype=torch.float64, device="cuda"); warm_h = torch.zeros(256, dtype=torch.int64, device="cuda")
    G.publish_state(0, 0.0)
    semb.field_minmax_hist(G.export_field("temperature"), 256, 0.0, 1.0, warm_mm, warm_h)
    semb.field_minmax_hist(G.export_field("temperature"), 256, 0.0, 0.0, warm_mm, warm_h)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    G.publish_state(17, 0.25)
    d = G.export_field("temperature")
    assert d.ptr == dT.data_ptr() and d.count == m.n and d.stride == 1          # pointer identity: no copy
    assert d.memspace == 1 and d.dtype == 1 and d.cycle == 17 and d.time == 0.25
    dm = G.export_field("velocity_magnitude")
    mm = torch.zeros(2, dtype=torch.float64, device="cuda"); hist = torch.zeros(256, dtype=torch.int64, device="cuda")
    semb.field_minmax_hist(d, 256, 0.0, 1.0, mm, hist)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                               # nothing allocated by publish/export/consume
    mn, mx, h = orc.minmax_hist(T, 256, 0.0, 1.0)
    assert mm[0].item() == mn and mm[1].item() == mx
    assert np.array_equal(hist.cpu().numpy().astype(np.uint64), h)
    vm_ref = orc.vmag(*v)
    semb.field_minmax_hist(dm, 64, 0.0, 0.0, mm, hist[:64])                    # range = [min, max] found on the device
    mn, mx, h = orc.minmax_hist(vm_ref, 64, vm_ref.min(), vm_ref.max())
    assert mm[0].item() == mn and mm[1].item() == mx
    assert np.array_equal(hist[:64].cpu().numpy().astype(np.uint64), h)
    # the same statistics from the three components, |v| computed on the fly (nothing written): one pass with a given range,
    # two when the range is to be found; both exactly the oracle's counts
    dx, dy, dz = (G.export_field(nm) for nm in ("velocity_x", "velocity_y", "velocity_z"))
    for lo, hi in ((0.0, 1.8), (0.0, 0.0)):
        semb.vector_magnitude_minmax_hist(dx, dy, dz, 64, lo, hi, mm, hist[:64])
        mn, mx, h = orc.minmax_hist(vm_ref, 64, lo if lo < hi else vm_ref.min(), hi if lo < hi else vm_ref.max())
        assert mm[0].item() == mn and mm[1].item() == mx
        assert np.array_equal(hist[:64].cpu().numpy().astype(np.uint64), h)
    with pytest.raises(semb.SembError):
        G.export_field("no_such_field")
