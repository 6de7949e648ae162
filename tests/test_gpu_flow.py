"""GPU parity of the flow operators and of the Boussinesq step (csrc/flow.cu) against the oracle (oracle/semflow.c,
oracle/boussinesq.py, reading R25): gradient / weak divergence / explicit terms at 1e-12
normwise, the full step through its five solves within the solver tolerance."""
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


MESHES = {
    "box_per_str_N5": lambda xi: I.box_mesh(3, 3, 4, 5, xi(5), periodic=(True, True, False), zstretch=2.0),
    "box_def_N7":     lambda xi: I.box_mesh(3, 2, 3, 7, xi(7), deform=0.05),
    "ogrid_N7":       lambda xi: I.config_mesh(2, xi, small=True)[0],
    "ogrid_N9":       lambda xi: I.config_mesh(4, xi, small=True)[0],
    "N2":             lambda xi: I.box_mesh(4, 3, 5, 2, xi(2), deform=0.04),
    "N10":            lambda xi: I.box_mesh(2, 2, 2, 10, xi(10), deform=0.05),
}


@pytest.mark.parametrize("name", list(MESHES))
def test_gradient_wdiv_and_explicit_terms(torch_cuda, semb, orc, xi_of, name):
    from oracle import boussinesq as Bq
    torch = torch_cuda
    m = MESHES[name](xi_of)
    P = orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period)
    ops = Bq.FlowOps(P, m.x, m.y, m.z)
    G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    try:
        z = lambda k=1: torch.empty(k * m.n, dtype=torch.float64, device="cuda")
        phi = np.sin(2 * m.x + 0.3) * np.cos(3 * m.y) + m.z ** 2 + 0.1 * I.uniform(3, m.n)
        g = [z(), z(), z()]
        G.gradient(dev(torch, phi), *g)
        ref = ops.grad(phi)
        scale = max(np.abs(r).max() for r in ref)
        for b in range(3):
            assert np.abs(g[b].cpu().numpy() - ref[b]).max() <= TOL * scale, (name, b)
        gv = [I.uniform(10 + c, m.n) for c in range(3)]
        out = z()
        G.weak_divergence(*[dev(torch, c) for c in gv], out)
        assert normwise(out.cpu().numpy(), ops.wdiv(*gv)) <= TOL
        # explicit terms with and without forcing; the vorticity comes back mass-averaged
        gidv = lambda seed: I.uniform(seed, P.n_unique)[P.gid]                # continuous fields
        u = [0.3 * gidv(20 + c) + np.sin(2 * np.pi * m.x + c) * m.z * (1 - m.z) for c in range(3)]
        th = 0.2 * gidv(30) * m.z * (1 - m.z)
        f = [I.uniform(40 + c, m.n) for c in range(4)]
        S = Bq.Boussinesq(P, m.x, m.y, m.z, Ra=1e4, Pr=0.7, dt=0.01, tags_u=0b10, tags_T=0b10)
        for forcing in (None, f):
            N4, om3 = z(4), z(3)
            G.flow_explicit_terms(*[dev(torch, c) for c in u], dev(torch, th), N4, om3, forcing=[dev(torch, c) for c in forcing] if forcing else None)
            Nref, om = S.explicit_terms(u, th, forcing)
            N4h, om3h = N4.cpu().numpy().reshape(4, m.n), om3.cpu().numpy().reshape(3, m.n)
            ns = max(np.abs(r).max() for r in Nref)
            for c in range(4):
                assert np.abs(N4h[c] - Nref[c]).max() <= TOL * ns, (name, "N", c)
            omb = [ops.average(c) for c in om]
            os_ = max(np.abs(r).max() for r in omb)
            for c in range(3):
                assert np.abs(om3h[c] - omb[c]).max() <= TOL * os_, (name, "omega", c)
    finally:
        G.close()


@pytest.mark.parametrize("name,tags_u", [("box_per_str_N5", 0b10), ("ogrid_N7", 0b110)])
def test_boussinesq_steps_match_the_oracle(torch_cuda, semb, orc, xi_of, name, tags_u):
    """Three steps (order 1, then BDF2/EXT2 twice) from a perturbed conduction state with the same preconditioners on both
    sides (Jacobi-PCG everywhere): iteration counts +-1 per solve, fields to 1e-8 of the velocity / temperature scale."""
    from oracle import boussinesq as Bq
    torch = torch_cuda
    m = MESHES[name](xi_of)
    P = orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period)
    Ra, Pr, dt = 2e4, 0.7, 5e-3
    S = Bq.Boussinesq(P, m.x, m.y, m.z, Ra=Ra, Pr=Pr, dt=dt, tags_u=tags_u, tags_T=0b10, rtol=1e-10)
    th0 = 0.05 * I.uniform(7, P.n_unique)[P.gid] * np.sin(np.pi * m.z)
    P.set_operator(0.0, 0b10)
    th0 = th0 * P.mask
    S.th = th0.copy()
    G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    try:
        st = semb.FlowState(m.n)
        st.theta.copy_(dev(torch, th0))
        for step in range(3):
            S.iters = []
            S.step()
            rc, its = G.boussinesq_step(st, Ra, Pr, dt, tags_u, 0b10, rtol=1e-10, precond_p=1, precond_u=1)
            assert rc == 0
            assert all(abs(a - b) <= 1 for a, b in zip(its, S.iters)), (step, its, S.iters)
            us = max(np.abs(c).max() for c in S.u)
            for c in range(3):
                assert np.abs(st.u[c].cpu().numpy() - S.u[c]).max() <= 1e-8 * us, (step, c)
            assert normwise(st.theta.cpu().numpy(), S.th) <= 1e-8
            pg, po = st.p.cpu().numpy(), S.p
            assert np.abs(pg - po).max() <= 1e-7 * np.abs(po).max()
        assert us > 1e-6                                                # the perturbation did set the fluid in motion
        assert int(st.c.step_index) == 3
    finally:
        G.close()


def test_boussinesq_with_multigrid_pressure_and_conduction_fixed_point(torch_cuda, semb, orc, xi_of):
    """Library defaults (p-multigrid on FP32 levels for the pressure): the conduction state u = 0, T = 1 - z stays put
    (PAPER.md:L272), and a perturbed run agrees with the oracle's Jacobi-PCG run to the solver tolerance."""
    from oracle import boussinesq as Bq
    torch = torch_cuda
    m = MESHES["box_per_str_N5"](xi_of)
    G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    try:
        st = semb.FlowState(m.n)
        for _ in range(3):
            rc, its = G.boussinesq_step(st, 1e5, 0.7, 1e-2, 0b10, 0b10, rtol=1e-11, mg_fp32=True)
            assert rc == 0
        assert max(float(c.abs().max()) for c in st.u) < 1e-8 and float(st.theta.abs().max()) < 1e-8
        gp = [torch.empty(m.n, dtype=torch.float64, device="cuda") for _ in range(3)]
        G.gradient(st.p, *gp)
        assert np.abs(gp[2].cpu().numpy() - (1.0 - m.z)).max() < 1e-7          # hydrostatic pressure
        P = orc.Problem(m.E, m.N, m.x, m.y, m.z, m.face_tag, m.period)
        S = Bq.Boussinesq(P, m.x, m.y, m.z, Ra=1e5, Pr=0.7, dt=1e-2, tags_u=0b10, tags_T=0b10, rtol=1e-11)
        P.set_operator(0.0, 0b10)
        th0 = 0.05 * I.uniform(7, P.n_unique)[P.gid] * np.sin(np.pi * m.z) * P.mask
        S.th = th0.copy()
        st = semb.FlowState(m.n); st.theta.copy_(dev(torch, th0))
        for _ in range(4):
            S.step()
            rc, its = G.boussinesq_step(st, 1e5, 0.7, 1e-2, 0b10, 0b10, rtol=1e-11, mg_fp32=True)
            assert rc == 0 and its[0] < 40
        us = max(np.abs(c).max() for c in S.u)
        for c in range(3):
            assert np.abs(st.u[c].cpu().numpy() - S.u[c]).max() <= 1e-7 * us
        assert normwise(st.theta.cpu().numpy(), S.th) <= 1e-7
    finally:
        G.close()
