"""CPU oracle of one Boussinesq time step (Eqs. (1)-(3); boundary and initial
conditions PAPER.md:L238 "top and bottom plates are isothermal and no-slip", L272 "zero velocity field and a linear
temperature profile, T = 1 - z").

TEST INFRASTRUCTURE ONLY (see semoracle.c): imported by tests/ and bench.py's cpu_baseline leg, never by the product.

The paper gives the equations, not the time discretisation (NekRS: BDF/EXT with a pressure Poisson equation
"the pressure Poisson solve ... the stiffest sub-step").  DESIGN.md reading R25 fixes the step below; every line is one of
the oracle's primitives (semflow.c: grad, wdiv; semoracle.c: gs, mask, PCG), in the order written here.

    nu = sqrt(Pr / Ra), kappa = 1 / sqrt(Ra Pr);   theta = T - (1 - z)  (homogeneous Dirichlet on the plates)
    order 1 on the first step (beta0 = 1, b = [1], a = [1]), then BDF2 / EXT2 (beta0 = 3/2, b = [2, -1/2], a = [2, -1])
    (i)   N_c     = -(u . grad) u_c + delta_cz T + f_c,   N_theta = -(u . grad) theta + u_z + f_theta       (collocation)
          omega   = curl u (collocation);  omega_bar = QQ^T(B omega) / QQ^T(B);  C = curl omega_bar
    (ii)  u~_c    = sum_k b_k u_c^(n+1-k) + dt sum_k a_k N_c^(n+1-k)
          g_c     = u~_c / dt - nu sum_k a_k C_c^(n+1-k)          (curl-curl form of the viscous term in the pressure equation)
          b_p     = QQ^T wdiv(g);   A p = b_p  (all Neumann: null_mean, R20), started from p^n
    (iii) u^_c    = u~_c - dt dp/dx_c (collocation);   (A + beta0/(nu dt) B) u_c^(n+1) = M QQ^T (B u^_c) / (nu dt),  start u_c^n
          theta~  = sum_k b_k theta^(n+1-k) + dt sum_k a_k N_theta^(n+1-k)
          (A + beta0/(kappa dt) B) theta^(n+1) = M QQ^T (B theta~) / (kappa dt),  start theta^n

Pins (tests/test_oracle_flow.py): the conduction state is a fixed point; second order in time on a manufactured solution whose
forcing sympy derives from Eqs. (1)-(3).  Parity unpinned: none.
"""
import ctypes as C

import numpy as np

from . import semoracle as O


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


class FlowOps:
    """metrics + collocation gradient + weak divergence on one mesh (semflow.c)"""

    def __init__(self, P, x, y, z):
        self.P = P
        self.E, self.N, self.n = P.E, P.N, P.n
        self.met = np.zeros((P.E, 9, P.Np))
        bad = O.lib().orc_metrics(C.c_int64(P.E), C.c_int(P.N), _p(O._f64(x)), _p(O._f64(y)), _p(O._f64(z)), _p(P.D), _p(self.met))
        if bad >= 0:
            raise ValueError(f"non-positive Jacobian in element {bad}")
        self.B = np.ascontiguousarray(P.geo[:, 6])                      # mass factor W J, [E, Np]
        self.Bassembled = O.gs(P.gid, P.n_unique, self.B.ravel())

    def grad(self, phi):
        g = [np.zeros(self.n) for _ in range(3)]
        O.lib().orc_grad(C.c_int64(self.E), C.c_int(self.N), _p(self.met), _p(self.P.D), _p(O._f64(phi)), _p(g[0]), _p(g[1]), _p(g[2]))
        return g

    def wdiv(self, gx, gy, gz):
        out = np.zeros(self.n)
        O.lib().orc_wdiv(C.c_int64(self.E), C.c_int(self.N), _p(self.met), _p(self.B), _p(self.P.D), _p(O._f64(gx)), _p(O._f64(gy)),
                         _p(O._f64(gz)), _p(out))
        return out

    def curl(self, vx, vy, vz):
        gx, gy, gz = self.grad(vx), self.grad(vy), self.grad(vz)
        return [gz[1] - gy[2], gx[2] - gz[0], gy[0] - gx[1]]

    def average(self, v):
        """mass-weighted average of a discontinuous field: QQ^T(B v) / QQ^T(B)"""
        return O.gs(self.P.gid, self.P.n_unique, self.B.ravel() * v) / self.Bassembled


class Boussinesq:
    def __init__(self, P, x, y, z, Ra, Pr, dt, tags_u, tags_T, rtol=1e-10, solver=None):
        """P: semoracle.Problem of the mesh.  solver(P, lam, tags, b, x0, null_mean) -> x replaces the oracle's Jacobi-PCG
        (tests pass a p-multigrid PCG for larger meshes)."""
        self.P, self.ops = P, FlowOps(P, x, y, z)
        self.z = O._f64(z)
        self.nu, self.kappa, self.dt = float(np.sqrt(Pr / Ra)), float(1.0 / np.sqrt(Ra * Pr)), float(dt)
        self.tags_u, self.tags_T, self.rtol = int(tags_u), int(tags_T), float(rtol)
        self.solver = solver or self._pcg
        n = P.n
        self.u = [np.zeros(n) for _ in range(3)]; self.th = np.zeros(n); self.p = np.zeros(n)
        self.u1 = [np.zeros(n) for _ in range(3)]; self.th1 = np.zeros(n)           # level n-1
        self.N0 = [np.zeros(n) for _ in range(4)]; self.N1 = [np.zeros(n) for _ in range(4)]   # N at n, n-1 (x, y, z, theta)
        self.C0 = [np.zeros(n) for _ in range(3)]; self.C1 = [np.zeros(n) for _ in range(3)]   # curl curl at n, n-1
        self.step_index = 0
        self.iters = []

    def _pcg(self, P, lam, tags, b, x0, null_mean):
        P.set_operator(lam, tags)
        r = P.pcg(b, x0=x0, precond=1, rtol=self.rtol, maxit=20000, null_mean=null_mean)
        assert r["status"] == 0, r["status"]
        self.iters.append(r["iters"])
        return r["x"]

    def explicit_terms(self, u, th, f=None):
        """(N_x, N_y, N_z, N_theta), omega  -- step (i) without the averaging"""
        ops = self.ops
        g = [ops.grad(c) for c in u]; gt = ops.grad(th)
        T = th + (1.0 - self.z)
        N = [-(u[0] * g[c][0] + u[1] * g[c][1] + u[2] * g[c][2]) for c in range(3)]
        N[2] = N[2] + T
        Nt = -(u[0] * gt[0] + u[1] * gt[1] + u[2] * gt[2]) + u[2]
        if f is not None:
            N = [N[c] + f[c] for c in range(3)]; Nt = Nt + f[3]
        om = [g[2][1] - g[1][2], g[0][2] - g[2][0], g[1][0] - g[0][1]]
        return N + [Nt], om

    def step(self, f=None):
        P, ops, dt, nu, ka = self.P, self.ops, self.dt, self.nu, self.kappa
        first = self.step_index == 0
        beta0, b, a = (1.0, [1.0, 0.0], [1.0, 0.0]) if first else (1.5, [2.0, -0.5], [2.0, -1.0])
        # (i)
        N, om = self.explicit_terms(self.u, self.th, f)
        omb = [ops.average(c) for c in om]
        Cc = ops.curl(*omb)
        # (ii)
        ut = [b[0] * self.u[c] + b[1] * self.u1[c] + dt * (a[0] * N[c] + a[1] * self.N1[c]) for c in range(3)]
        g = [ut[c] / dt - nu * (a[0] * Cc[c] + a[1] * self.C1[c]) for c in range(3)]
        bp = O.gs(P.gid, P.n_unique, ops.wdiv(*g))
        self.p = self.solver(P, 0.0, 0, bp, self.p, True)          # started from the previous step's pressure (zero on the first step)
        # (iii)
        gp = ops.grad(self.p)
        un = []
        P.set_operator(beta0 / (nu * dt), self.tags_u)
        for c in range(3):
            uh = ut[c] - dt * gp[c]
            rhs = P.assemble_rhs(uh / (nu * dt))
            un.append(self.solver(P, beta0 / (nu * dt), self.tags_u, rhs, self.u[c], False))
        tt = b[0] * self.th + b[1] * self.th1 + dt * (a[0] * N[3] + a[1] * self.N1[3])
        P.set_operator(beta0 / (ka * dt), self.tags_T)
        thn = self.solver(P, beta0 / (ka * dt), self.tags_T, P.assemble_rhs(tt / (ka * dt)), self.th, False)
        # rotate
        self.u1, self.th1, self.N1, self.C1 = self.u, self.th, N, Cc
        self.u, self.th = un, thn
        self.step_index += 1
        return self
