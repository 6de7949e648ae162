"""ctypes/numpy wrapper around oracle/semoracle.c.

TEST INFRASTRUCTURE ONLY (see the header of semoracle.c): imported by tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.  The product
package (paper_2501_13240_b200) never imports this module.

Every function takes and returns host numpy arrays (fp64 / int32), laid out as the C file
states: local node l = e*Np + k*n1^2 + j*n1 + i ("(ijk) ordering").
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "semoracle.c")
_SRCS = [_SRC, os.path.join(_HERE, "semimage.c"), os.path.join(_HERE, "semflow.c")]
_LIB = os.path.join(_HERE, "libsemoracle.so")
_lib = None


def build(force=False):
    """Compile semoracle.c -> libsemoracle.so (gcc -O2, OpenMP, no FP contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(f) for f in _SRCS):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
               "-o", _LIB] + _SRCS + ["-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Op(C.Structure):
    _fields_ = [("E", C.c_int64), ("N", C.c_int32), ("pad_", C.c_int32), ("n", C.c_int64),
                ("n_unique", C.c_int64), ("geo", C.c_void_p), ("D", C.c_void_p), ("gid", C.c_void_p),
                ("mask", C.c_void_p), ("invmult", C.c_void_p), ("lam", C.c_double)]


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.orc_min_spacing.restype = C.c_double
        _lib.orc_dot.restype = C.c_double
        _lib.orc_geo.restype = C.c_int64
        _lib.orc_numbering.restype = C.c_int64
        _lib.orc_metrics.restype = C.c_int64
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads():
    return int(lib().orc_num_threads())


def gll(N):
    """c-1: (xi, rho), each [N+1]."""
    xi = np.zeros(N + 1); rho = np.zeros(N + 1)
    assert lib().orc_gll(C.c_int(N), _p(xi), _p(rho)) == 0
    return xi, rho


def dhat(N, xi=None):
    """c-2: D[i, j] = l'_j(xi_i), [N+1, N+1]."""
    if xi is None:
        xi = gll(N)[0]
    D = np.zeros((N + 1, N + 1))
    assert lib().orc_dhat(C.c_int(N), _p(_f64(xi)), _p(D)) == 0
    return D


def geo_factors(E, N, x, y, z):
    """c-3: geo [E, 7, Np]; raises ValueError on a non-positive Jacobian."""
    xi, rho = gll(N); D = dhat(N, xi)
    Np = (N + 1) ** 3
    x, y, z = _f64(x), _f64(y), _f64(z)
    geo = np.zeros((E, 7, Np))
    bad = lib().orc_geo(C.c_int64(E), C.c_int(N), _p(x), _p(y), _p(z), _p(D), _p(rho), _p(geo))
    if bad >= 0:
        raise ValueError(f"non-positive Jacobian in element {bad}")
    return geo


def axhelm(E, N, geo, lam, u, lam0=None, lam1=None, D=None):
    """c-4: w = D^T G D u + lam B u on every element."""
    if D is None:
        D = dhat(N)
    u = _f64(u); w = np.zeros_like(u)
    l0 = _f64(lam0) if lam0 is not None else None
    l1 = _f64(lam1) if lam1 is not None else None
    lib().orc_axhelm(C.c_int64(E), C.c_int(N), _p(geo), _p(_f64(D)), C.c_double(lam), _p(l0), _p(l1), _p(u), _p(w))
    return w


def min_spacing(E, N, x, y, z):
    return float(lib().orc_min_spacing(C.c_int64(E), C.c_int(N), _p(_f64(x)), _p(_f64(y)), _p(_f64(z))))


def numbering(E, N, x, y, z, period, tol=None):
    """c-6: (gid int32 [n], n_unique).  tol defaults to 1e-8 * min node spacing."""
    x, y, z = _f64(x), _f64(y), _f64(z)
    if tol is None:
        tol = 1e-8 * min_spacing(E, N, x, y, z)
    per = _f64(period)
    gid = np.zeros(E * (N + 1) ** 3, dtype=np.int32)
    nu = lib().orc_numbering(C.c_int64(E), C.c_int(N), _p(x), _p(y), _p(z), _p(per), C.c_double(tol), _p(gid))
    if nu < 0:
        raise ValueError("coordinate matching is not an equivalence relation at this tolerance")
    return gid, int(nu)


def gs(gid, n_unique, w):
    """c-7: QQ^T w (returns a new array)."""
    out = _f64(w).copy()
    lib().orc_gs(C.c_int64(out.size), _p(gid), C.c_int64(n_unique), _p(out))
    return out


def dirichlet_mask(E, N, face_tag, tags, gid, n_unique):
    mask = np.zeros(E * (N + 1) ** 3)
    ft = np.ascontiguousarray(face_tag, dtype=np.int32)
    lib().orc_mask(C.c_int64(E), C.c_int(N), _p(ft), C.c_uint32(tags), _p(gid), C.c_int64(n_unique), _p(mask))
    return mask


def diag_local(E, N, geo, lam, D=None):
    if D is None:
        D = dhat(N)
    d = np.zeros(E * (N + 1) ** 3)
    lib().orc_diag_local(C.c_int64(E), C.c_int(N), _p(geo), _p(_f64(D)), C.c_double(lam), _p(d))
    return d


def minmax_hist(v, nbins, lo, hi):
    v = _f64(v); mm = np.zeros(2); h = np.zeros(nbins, dtype=np.uint64)
    lib().orc_minmax_hist(C.c_int64(v.size), _p(v), C.c_int(nbins), C.c_double(lo), C.c_double(hi), _p(mm), _p(h))
    return mm[0], mm[1], h


def vmag(vx, vy, vz):
    vx, vy, vz = _f64(vx), _f64(vy), _f64(vz); out = np.zeros_like(vx)
    lib().orc_vmag(C.c_int64(vx.size), _p(vx), _p(vy), _p(vz), _p(out))
    return out


class Problem:
    """Mesh + operator state of the oracle: geo, numbering, mask, invmult, dinv (c-3 .. c-8)."""

    def __init__(self, E, N, x, y, z, face_tag, period, lam=0.0, dirichlet_tags=0, gid=None):
        self.E, self.N, self.Np = E, N, (N + 1) ** 3
        self.n = E * self.Np
        self.xi, self.rho = gll(N)
        self.D = dhat(N, self.xi)
        self.geo = geo_factors(E, N, x, y, z)
        if gid is None:
            self.gid, self.n_unique = numbering(E, N, x, y, z, period)
        else:
            self.gid = np.ascontiguousarray(gid, dtype=np.int32); self.n_unique = int(self.gid.max()) + 1
        self.face_tag = np.ascontiguousarray(face_tag, dtype=np.int32)
        self.invmult = np.zeros(self.n)
        lib().orc_invmult(C.c_int64(self.n), _p(self.gid), C.c_int64(self.n_unique), _p(self.invmult))
        self.set_operator(lam, dirichlet_tags)

    def set_operator(self, lam, dirichlet_tags):
        self.lam, self.tags = float(lam), int(dirichlet_tags)
        self.mask = dirichlet_mask(self.E, self.N, self.face_tag, self.tags, self.gid, self.n_unique)
        self._op = _Op(self.E, self.N, 0, self.n, self.n_unique, _p(self.geo), _p(self.D), _p(self.gid),
                       _p(self.mask), _p(self.invmult), self.lam)
        self.dinv = np.zeros(self.n)
        lib().orc_dinv(C.byref(self._op), _p(self.dinv))

    def apply_A(self, v):
        v = _f64(v); out = np.zeros(self.n); tmp = np.zeros(self.n)
        lib().orc_apply_A(C.byref(self._op), _p(v), _p(out), _p(tmp))
        return out

    def dot(self, a, b):
        return float(lib().orc_dot(C.byref(self._op), _p(_f64(a)), _p(_f64(b))))

    def assemble_rhs(self, f):
        b = np.zeros(self.n)
        lib().orc_assemble_rhs(C.byref(self._op), _p(_f64(f)), _p(b))
        return b

    def cheb_jacobi(self, k, lmax, r):
        z = np.zeros(self.n); work = np.zeros(4 * self.n)
        lib().orc_cheb_jacobi(C.byref(self._op), C.c_int(k), C.c_double(lmax), _p(self.dinv), _p(_f64(r)), _p(z), _p(work))
        return z

    def cheb4_jacobi(self, k, lmax, r):
        """fourth-kind Chebyshev-Jacobi smoother (f-1)"""
        z = np.zeros(self.n); work = np.zeros(4 * self.n)
        lib().orc_cheb4_jacobi(C.byref(self._op), C.c_int(k), C.c_double(lmax), _p(self.dinv), _p(_f64(r)), _p(z), _p(work))
        return z

    def lanczos_lmax(self, v0, steps=10):
        """largest Ritz value of D^-1/2 A D^-1/2 after `steps` Lanczos steps, times 1.1 (c-10)."""
        a = np.zeros(steps); b = np.zeros(steps)
        m = lib().orc_lanczos(C.byref(self._op), _p(self.dinv), _p(_f64(v0)), C.c_int(steps), _p(a), _p(b))
        T = np.diag(a[:m]) + np.diag(b[:m - 1], 1) + np.diag(b[:m - 1], -1)
        return 1.1 * float(np.linalg.eigvalsh(T)[-1])

    def mean(self, v):
        """mean over the unique nodes, <v,1> / n_unique (reading R20)"""
        return float(np.sum(_f64(v) * self.invmult)) / self.n_unique

    def pcg(self, b, x0=None, precond=1, cheb_k=2, lmax=0.0, rtol=1e-10, atol=0.0, maxit=10000, hist_len=0, null_mean=False):
        """c-9.  Returns dict(x, iters, status, r0, rn, hist).  null_mean (R20, operators whose null space is the
        constants): solve A x = b - mean(b) and return the solution of zero mean."""
        if null_mean:
            assert self.lam == 0.0 and np.all(self.mask == 1.0)
            r = self.pcg(_f64(b) - self.mean(b), x0, precond, cheb_k, lmax, rtol, atol, maxit, hist_len)
            r["x"] = r["x"] - self.mean(r["x"])
            return r
        x = np.zeros(self.n) if x0 is None else _f64(x0).copy()
        hist = np.zeros(max(hist_len, 1)); out3 = np.zeros(3)
        st = lib().orc_pcg(C.byref(self._op), C.c_int(precond), C.c_int(cheb_k), C.c_double(lmax), _p(self.dinv),
                           _p(_f64(b)), _p(x), C.c_double(rtol), C.c_double(atol), C.c_int(maxit),
                           C.c_int(1 if x0 is None else 0), _p(hist), C.c_int(hist_len), _p(out3))
        it = int(out3[0])
        return dict(x=x, iters=it, status=int(st), r0=out3[1], rn=out3[2], hist=hist[:min(hist_len, it + 1)])


# ---------------------------------------------------------------------------------------------------------------
# f-1  p-multigrid V-cycle preconditioner (semoracle.c: orc_mg_*; reading R19)
class _MgLevel(C.Structure):
    _fields_ = [("op", _Op), ("dinv", C.c_void_p), ("lmax", C.c_double), ("J", C.c_void_p)]


class _Mg(C.Structure):
    _fields_ = [("nlevels", C.c_int32), ("k_smooth", C.c_int32), ("k_coarse", C.c_int32), ("kind", C.c_int32), ("coarse_frac", C.c_double),
                ("lev", _MgLevel * 8)]


def interp_matrix(Nfrom, Nto):
    """J[(Nto+1), (Nfrom+1)]: Lagrange basis of the order-Nfrom GLL nodes evaluated at the order-Nto GLL nodes."""
    J = np.zeros((Nto + 1, Nfrom + 1))
    if lib().orc_interp_matrix(C.c_int(Nfrom), C.c_int(Nto), _p(J)):
        raise ValueError("interp_matrix")
    return J


def interp3(E, J, v, transpose=False):
    """per element J x J x J (or its transpose) applied to v; J is [nf1, nc1]."""
    nf1, nc1 = J.shape
    out = np.zeros(E * (nc1 if transpose else nf1) ** 3)
    lib().orc_interp3(C.c_int64(E), C.c_int(nf1), C.c_int(nc1), _p(np.ascontiguousarray(J)), C.c_int(1 if transpose else 0),
                      _p(_f64(v)), _p(out))
    return out


MG_LMAX_SEED = 250113240 + 900      # + level: start vector of the per-level lambda_max estimate (R19)


def _splitmix_uniform(seed, n):
    """U[-1,1) per index from the counter-based splitmix64 of the input recipe, restated here."""
    with np.errstate(over="ignore"):
        z = np.uint64(seed) + (np.arange(n, dtype=np.uint64) + np.uint64(1)) * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (2.0 ** -53) * 2.0 - 1.0


class Multigrid:
    """Levels of the p-multigrid preconditioner for the operator (lam, tags) on a mesh: level 0 is order N, level l
    the same elements at order orders[l] with coordinates interpolated from level 0.  lmax[l] = 1.1 x the largest
    Ritz value of a 10-step Lanczos from the start vector M QQ^T u, u ~ U[-1,1) per local node from splitmix64 with
    seed MG_LMAX_SEED + l (a ROUGH vector: a smooth one, e.g. M QQ^T B 1, underestimates lambda_max by 20 % on
    meshes of some thousand elements and the V-cycle loses definiteness), or given."""

    def __init__(self, E, N, x, y, z, face_tag, period, lam, tags, orders, k_smooth=2, k_coarse=2, lmax=None, v0_of=None,
                 kind=1, coarse_frac=0.1, fp32=False):
        assert orders[0] == N and all(a > b for a, b in zip(orders, orders[1:])) and len(orders) <= 8
        self.orders = list(orders)
        self.k_smooth, self.k_coarse = int(k_smooth), int(k_coarse)
        self.levels, self.J, self.coords = [], [], []
        for l, Nl in enumerate(orders):
            if l == 0:
                xl, yl, zl = _f64(x), _f64(y), _f64(z)
            else:
                Jc = interp_matrix(N, Nl)                       # fine Lagrange basis at the coarse nodes
                xl, yl, zl = (interp3(E, Jc, a) for a in (x, y, z))
            self.coords.append((xl, yl, zl))
            self.levels.append(Problem(E, Nl, xl, yl, zl, face_tag, period, lam=lam, dirichlet_tags=tags))
        for l in range(len(orders) - 1):
            self.J.append(interp_matrix(orders[l + 1], orders[l]))      # [n1_l, n1_{l+1}]
        if lmax is None:
            lmax = []
            for l, P in enumerate(self.levels):
                v0 = v0_of(P) if v0_of is not None else P.mask * gs(P.gid, P.n_unique, _splitmix_uniform(MG_LMAX_SEED + l, P.n))
                lmax.append(P.lanczos_lmax(v0, 10))
        self.lmax = [float(v) for v in lmax]
        self._mg = _Mg()
        self._mg.nlevels, self._mg.k_smooth, self._mg.k_coarse = len(orders), self.k_smooth, self.k_coarse
        self.coarse_frac = self._mg.coarse_frac = float(coarse_frac)   # last level: first-kind interval [coarse_frac, 1] lmax
        self.kind = self._mg.kind = int(kind)          # 4 = fourth-kind Chebyshev smoother (orc_cheb4_jacobi), else first kind
        self.fp32 = bool(fp32)
        self._r32 = []          # float-rounded level data (R21), kept alive here
        for l, P in enumerate(self.levels):
            if self.fp32:       # FP32 storage: the level operators see the factors, diagonal and multiplicities as stored
                r32 = lambda a: np.ascontiguousarray(a, dtype=np.float32).astype(np.float64)
                geo32, dinv32, inv32 = r32(P.geo), r32(P.dinv), r32(P.invmult)
                self._r32.append((geo32, dinv32, inv32))
                self._mg.lev[l].op = _Op(P.E, P.N, 0, P.n, P.n_unique, _p(geo32), _p(P.D), _p(P.gid), _p(P.mask), _p(inv32), P.lam)
                self._mg.lev[l].dinv = dinv32.ctypes.data
            else:
                self._mg.lev[l].op = P._op
                self._mg.lev[l].dinv = P.dinv.ctypes.data
            self._mg.lev[l].lmax = self.lmax[l]
            self._mg.lev[l].J = self.J[l].ctypes.data if l < len(self.J) else None

    def prolong(self, l, vc):
        vf = np.zeros(self.levels[l].n)
        lib().orc_mg_prolong(C.byref(self._mg), C.c_int(l), _p(_f64(vc)), _p(vf))
        return vf

    def restrict(self, l, rf):
        rc = np.zeros(self.levels[l + 1].n); tmp = np.zeros(self.levels[l].n)
        lib().orc_mg_restrict(C.byref(self._mg), C.c_int(l), _p(_f64(rf)), _p(rc), _p(tmp))
        return rc

    def vcycle(self, r, level=0):
        z = np.zeros(self.levels[level].n)
        if self.fp32:
            assert level == 0
            lib().orc_mg_vcycle_fp32(C.byref(self._mg), _p(_f64(r)), _p(z))
        else:
            lib().orc_mg_vcycle(C.byref(self._mg), C.c_int(level), _p(_f64(r)), _p(z))
        return z

    def pcg(self, b, x0=None, rtol=1e-10, atol=0.0, maxit=10000, hist_len=0, null_mean=False):
        P = self.levels[0]
        if null_mean:
            assert P.lam == 0.0 and np.all(P.mask == 1.0)
            r = self.pcg(_f64(b) - P.mean(b), x0, rtol, atol, maxit, hist_len)
            r["x"] = r["x"] - P.mean(r["x"])
            return r
        x = np.zeros(P.n) if x0 is None else _f64(x0).copy()
        hist = np.zeros(max(hist_len, 1)); out3 = np.zeros(3)
        if self.fp32:
            st = lib().orc_pcg_mg_fp32(C.byref(P._op), C.byref(self._mg), _p(_f64(b)), _p(x), C.c_double(rtol), C.c_double(atol),
                                       C.c_int(maxit), C.c_int(1 if x0 is None else 0), _p(hist), C.c_int(hist_len), _p(out3))
        else:
            st = lib().orc_pcg_mg(C.byref(self._mg), _p(_f64(b)), _p(x), C.c_double(rtol), C.c_double(atol), C.c_int(maxit),
                                  C.c_int(1 if x0 is None else 0), _p(hist), C.c_int(hist_len), _p(out3))
        it = int(out3[0])
        return dict(x=x, iters=it, status=int(st), r0=out3[1], rn=out3[2], hist=hist[:min(hist_len, it + 1)])


# ---------------------------------------------------------------------------------------------------------------
# f-4  in-situ image consumer (semimage.c; reading R24)
class ImgView(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("origin", C.c_double * 3), ("u", C.c_double * 3),
                ("v", C.c_double * 3), ("du", C.c_double), ("dv", C.c_double)]


class ImgCmap(C.Structure):
    _fields_ = [("lo", C.c_double), ("hi", C.c_double), ("ncolors", C.c_int32), ("rgb", (C.c_uint8 * 3) * 16),
                ("background", C.c_uint32)]


def make_view(width, height, origin, u, v, du, dv):
    vw = ImgView(width, height)
    for c in range(3):
        vw.origin[c], vw.u[c], vw.v[c] = float(origin[c]), float(u[c]), float(v[c])
    vw.du, vw.dv = float(du), float(dv)
    return vw


def make_cmap(lo, hi, colors, background=0xff000000):
    cm = ImgCmap(float(lo), float(hi), len(colors))
    for m, col in enumerate(colors):
        for c in range(3):
            cm.rgb[m][c] = int(col[c])
    cm.background = int(background)
    return cm


def colormap(cm, val):
    val = _f64(val); out = np.zeros(val.size, dtype=np.uint32)
    lib().orc_colormap(C.byref(cm), C.c_int64(val.size), _p(val), _p(out))
    return out


def image_slice(E, N, x, y, z, field, vw, cm):
    """(rgba uint32 [H, W], cell_of int64 [H, W])"""
    rgba = np.zeros(vw.width * vw.height, dtype=np.uint32); cell = np.zeros(vw.width * vw.height, dtype=np.int64)
    lib().orc_image_slice(C.c_int64(E), C.c_int(N), _p(_f64(x)), _p(_f64(y)), _p(_f64(z)), _p(_f64(field)), C.byref(vw), C.byref(cm),
                          _p(rgba), _p(cell))
    return rgba.reshape(vw.height, vw.width), cell.reshape(vw.height, vw.width)


def image_isosurface(E, N, x, y, z, field, iso, cfield, vw, cm, light, dlo, dhi):
    """(rgba uint32 [H, W], key uint64 [H, W]); key >> 32 = depth quantised to 2^-32 of [dlo, dhi]"""
    rgba = np.zeros(vw.width * vw.height, dtype=np.uint32); key = np.zeros(vw.width * vw.height, dtype=np.uint64)
    lt = _f64(light)
    lib().orc_image_isosurface(C.c_int64(E), C.c_int(N), _p(_f64(x)), _p(_f64(y)), _p(_f64(z)), _p(_f64(field)), C.c_double(iso),
                               _p(_f64(cfield)) if cfield is not None else None, C.byref(vw), C.byref(cm), _p(lt),
                               C.c_double(dlo), C.c_double(dhi), _p(rgba), _p(key))
    return rgba.reshape(vw.height, vw.width), key.reshape(vw.height, vw.width)
