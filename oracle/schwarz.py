"""CPU oracle of the overlapping Schwarz smoother of the p-multigrid preconditioner (§2.2:
"p-multigrid that uses 4th-kind Chebyshev-acceleration of overlapping Schwarz smoothers").  The paper names the method
and gives no formulas; reading R26 fixes them.

TEST INFRASTRUCTURE ONLY: imported by tests/ (and bench.py's cpu_baseline leg), never by the product.

Subdomains = the element closures (the (N+1)^3 nodes of one element; neighbouring subdomains overlap in their shared
faces, edges and corners).  The subdomain operator is the separable ("fast diagonalisation") approximation

    A~_e = B_t x B_s x A_r + B_t x A_s x B_r + A_t x B_s x B_r + lambda B_t x B_s x B_r

of the assembled operator restricted to the element's nodes with homogeneous Dirichlet values on every other node:
per direction d the element is a 1-D GLL element of length l_d (mean of its four straight edges), A_d = (2/l_d) K^,
B_d = (l_d/2) diag(rho), K^ = D^T diag(rho) D; at an end node shared with a neighbour of length l' across that face the
neighbour's end entries (2/l') K^_NN and (l'/2) rho_N are added (the restriction of the assembled 1-D operator); an end
node on a Dirichlet face is removed; a Neumann boundary face adds nothing.  The neighbour's length travels through a
gather-scatter of the interior nodes of each face (two copies each, whatever the neighbour's orientation).  On an affine box mesh whose operator IS separable, A~_e is
exactly the assembled operator restricted to the element's nodes (the pin).

Smoother:  S r = M QQ^T [ w o A~_e^-1 ( w o r ) ],  w = sqrt(1 / multiplicity)  -- symmetric positive semi-definite.
A~_e^-1 = (S_t x S_s x S_r) [Lam_r (+) Lam_s (+) Lam_t + lambda]^-1 (S_t x S_s x S_r)^T with A_d S_d = B_d S_d Lam_d,
S_d^T B_d S_d = I (numpy.linalg.eigh on B^-1/2 A B^-1/2: a library primitive as one step).

Pins (tests/test_oracle_schwarz.py): exact restricted inverse on tensor boxes, dense symmetric positive S, closed-form fourth-kind
polynomial in S A, Lanczos bound.  Parity unpinned: none.
"""
import numpy as np

from . import semoracle as O


def edge_lengths(P, x, y, z):
    """l[e, d], d = r, s, t: mean straight length of the four edges of element e in direction d"""
    n1 = P.N + 1
    X = np.stack([O._f64(x), O._f64(y), O._f64(z)], -1).reshape(P.E, n1, n1, n1, 3)      # [e, k, j, i, c]
    N = P.N
    l = np.zeros((P.E, 3))
    for a in (0, N):
        for b in (0, N):
            l[:, 0] += np.linalg.norm(X[:, a, b, N] - X[:, a, b, 0], axis=-1)            # r: i varies, (k, j) = (a, b)
            l[:, 1] += np.linalg.norm(X[:, a, N, b] - X[:, a, 0, b], axis=-1)            # s: j varies, (k, i) = (a, b)
            l[:, 2] += np.linalg.norm(X[:, N, a, b] - X[:, 0, a, b], axis=-1)            # t: k varies, (j, i) = (a, b)
    return 0.25 * l


def probe_index(N, face):
    """local node index (within an element) of the probe node of face r-, r+, s-, s+, t-, t+ : (i, j, k) with the face's own
    coordinate at its end and the two others equal to 1"""
    n1 = N + 1
    i, j, k = [(0, 1, 1), (N, 1, 1), (1, 0, 1), (1, N, 1), (1, 1, 0), (1, 1, N)][face]
    return k * n1 * n1 + j * n1 + i


class Schwarz:
    def __init__(self, P, x, y, z):
        """P: semoracle.Problem with its operator (lam, Dirichlet tags) set; N >= 2."""
        assert P.N >= 2
        self.P = P
        N, n1, E, Np = P.N, P.N + 1, P.E, P.Np
        rho = P.rho
        K = P.D.T @ np.diag(rho) @ P.D
        self.len = edge_lengths(P, x, y, z)
        # neighbour lengths through the gather-scatter of the face probes
        # every INTERIOR node of a face carries the element's length normal to that face: such a node has exactly two copies
        # (this element's and the neighbour's) wherever the neighbour's local axes point, so the sum is l_own + l_neighbour
        F4 = np.zeros((E, n1, n1, n1))                                            # [e, k, j, i]
        inn = slice(1, N)
        F4[:, inn, inn, 0] = self.len[:, 0, None, None]; F4[:, inn, inn, N] = self.len[:, 0, None, None]
        F4[:, inn, 0, inn] = self.len[:, 1, None, None]; F4[:, inn, N, inn] = self.len[:, 1, None, None]
        F4[:, 0, inn, inn] = self.len[:, 2, None, None]; F4[:, N, inn, inn] = self.len[:, 2, None, None]
        F = F4.reshape(E, Np)
        Gs = O.gs(P.gid, P.n_unique, F.ravel()).reshape(E, Np)
        mult = 1.0 / P.invmult.reshape(E, Np)
        ft = P.face_tag.reshape(E, 6)
        self.S = np.zeros((E, 3, n1, n1)); self.lam = np.ones((E, 3, n1))
        for e in range(E):
            for d in range(3):
                l = self.len[e, d]
                A = (2.0 / l) * K.copy(); B = (l / 2.0) * rho.copy()
                free = np.ones(n1, dtype=bool)
                for side, node in ((0, 0), (1, N)):
                    f = 2 * d + side
                    pi = probe_index(N, f)
                    tag = int(ft[e, f])
                    if tag > 0 and (P.tags >> tag) & 1:
                        free[node] = False                                   # Dirichlet face: the end node is not an unknown
                    elif mult[e, pi] > 1.5:
                        ln = Gs[e, pi] - l                                   # the neighbour's length normal to the shared face
                        A[node, node] += (2.0 / ln) * K[N, N]
                        B[node] += (ln / 2.0) * rho[N]
                idx = np.where(free)[0]
                bh = 1.0 / np.sqrt(B[idx])
                lam, Y = np.linalg.eigh(bh[:, None] * A[np.ix_(idx, idx)] * bh[None, :])
                self.S[e, d][np.ix_(idx, np.arange(idx.size))] = bh[:, None] * Y
                self.lam[e, d, :idx.size] = lam
                self.nfree = getattr(self, "nfree", np.zeros((E, 3), dtype=np.int64))
                self.nfree[e, d] = idx.size
        self.w = np.sqrt(P.invmult).reshape(E, n1, n1, n1)

    def local_solve(self, v):
        """A~_e^-1 v element by element; v, result [n] (local, no weights, no assembly)"""
        P = self.P
        n1, E = P.N + 1, P.E
        V = O._f64(v).reshape(E, n1, n1, n1)                                 # [e, k, j, i]
        Sr, Ss, St = self.S[:, 0], self.S[:, 1], self.S[:, 2]
        t = np.einsum("eia,ejb,ekc,ekji->ecba", Sr, Ss, St, V)                # (S_t x S_s x S_r)^T v
        den = self.lam[:, 2][:, :, None, None] + self.lam[:, 1][:, None, :, None] + self.lam[:, 0][:, None, None, :] + P.lam
        # dummy modes of removed (Dirichlet) nodes have zero eigenvector columns: they contribute nothing
        big = np.abs(den).max(axis=(1, 2, 3), keepdims=True)
        inv = np.where(den > 1e-12 * big, 1.0 / np.where(den > 1e-12 * big, den, 1.0), 0.0)   # pseudo-inverse on a singular block
        t = t * inv
        out = np.einsum("eia,ejb,ekc,ecba->ekji", Sr, Ss, St, t)
        return out.reshape(-1)

    def apply(self, r):
        """S r = M QQ^T [ w o A~^-1 (w o r) ]"""
        P = self.P
        w = self.w.ravel()
        z = w * self.local_solve(w * O._f64(r))
        return P.mask * O.gs(P.gid, P.n_unique, z)


def lanczos_lmax(P, S, v0, steps=10):
    """1.1 x the largest Ritz value of S A after `steps` steps of the conjugate-gradient (Lanczos) recurrence for A with the
    preconditioner S from the continuous, masked start vector v0: T_jj = 1/alpha_j + beta_(j-1)/alpha_(j-1),
    T_(j,j+1) = sqrt(beta_j)/alpha_j."""
    r = O._f64(v0).copy()
    z = S.apply(r)
    rho = P.dot(r, z)
    p = z.copy()
    al, be = [], []
    for j in range(steps):
        q = P.apply_A(p)
        a = rho / P.dot(p, q)
        r = r - a * q
        z = S.apply(r)
        rho_new = P.dot(r, z)
        b = rho_new / rho
        al.append(a); be.append(b)
        if not (rho_new > 1e-28 * abs(rho)):
            break
        p = z + b * p
        rho = rho_new
    m = len(al)
    T = np.zeros((m, m))
    for j in range(m):
        T[j, j] = 1.0 / al[j] + (be[j - 1] / al[j - 1] if j > 0 else 0.0)
        if j + 1 < m:
            T[j, j + 1] = T[j + 1, j] = np.sqrt(be[j]) / al[j]
    return 1.1 * float(np.linalg.eigvalsh(T)[-1])


def cheb4(P, S, k, lmax, r):
    """k-th order Chebyshev polynomial of the fourth kind accelerating the smoother S (same recurrence as
    orc_cheb4_jacobi with dinv o . replaced by S .):  d_0 = (4/3)(1/lmax) S r;  z += d;  res -= A d;
    d_i = ((2i-1)/(2i+3)) d_(i-1) + ((8i+4)/(2i+3)) (1/lmax) S res_i"""
    res = O._f64(r).copy()
    d = (4.0 / (3.0 * lmax)) * S.apply(res)
    z = d.copy()
    for i in range(1, k + 1):
        res = res - P.apply_A(d)
        d = ((2.0 * i - 1.0) / (2.0 * i + 3.0)) * d + ((8.0 * i + 4.0) / ((2.0 * i + 3.0) * lmax)) * S.apply(res)
        z = z + d
    return z


class MultigridSchwarz:
    """The V-cycle of semoracle.Multigrid (same levels, transfers and cycle, reading R19) with the Chebyshev-JACOBI smoother of
    every level of order >= 2 replaced by the fourth-kind Chebyshev-SCHWARZ smoother; the last level (order 1) keeps the
    first-kind Chebyshev-Jacobi coarse smoother."""

    def __init__(self, mg, k_smooth=1, lmax=None):
        self.mg, self.k = mg, int(k_smooth)
        self.S, self.lmax = [], []
        for l, P in enumerate(mg.levels[:-1]):
            xl, yl, zl = mg.coords[l]
            S = Schwarz(P, xl, yl, zl)
            self.S.append(S)
            if lmax is not None:
                self.lmax.append(float(lmax[l]))
            else:
                v0 = P.mask * O.gs(P.gid, P.n_unique, O._splitmix_uniform(O.MG_LMAX_SEED + l, P.n))
                self.lmax.append(lanczos_lmax(P, S, v0, 10))

    def vcycle(self, r, l=0):
        mg = self.mg
        if l == len(mg.levels) - 1:
            return mg.vcycle(r, level=l)                                      # coarse level: as in Multigrid
        P = mg.levels[l]
        z = cheb4(P, self.S[l], self.k, self.lmax[l], r)
        res = r - P.apply_A(z)
        z = z + mg.prolong(l, self.vcycle(mg.restrict(l, res), l + 1))
        res = r - P.apply_A(z)
        return z + cheb4(P, self.S[l], self.k, self.lmax[l], res)

    def pcg(self, b, rtol=1e-10, maxit=1000):
        P = self.mg.levels[0]
        x = np.zeros(P.n); r = O._f64(b).copy()
        bn = np.sqrt(P.dot(r, r)); hist = [bn]
        z = self.vcycle(r); rho = P.dot(r, z); p = z.copy()
        it = 0
        while it < maxit and hist[-1] > rtol * bn:
            q = P.apply_A(p)
            a = rho / P.dot(p, q)
            x += a * p; r -= a * q
            hist.append(np.sqrt(P.dot(r, r))); it += 1
            z = self.vcycle(r); rn = P.dot(r, z)
            p = z + (rn / rho) * p; rho = rn
        return dict(x=x, iters=it, hist=np.array(hist))
