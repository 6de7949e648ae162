"""Thin ctypes binding over libsemb200.so (include/semb200.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; torch supplies device memory
(`tensor.data_ptr()`) and the stream (`torch.cuda.current_stream().cuda_stream`).  There is no
CPU fallback: loading fails loudly when the library is missing, and every compute call raises
SembError when the library reports an error (e.g. no CUDA device).
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("SEMB_LIB") or os.path.join(_HERE, "libsemb200.so")       # SEMB_LIB: an A/B build of the same sources

SEMB_OK, SEMB_MAXIT = 0, 1
ERRORS = {-1: "SEMB_EINVAL", -2: "SEMB_ENOMEM", -3: "SEMB_ECUDA", -4: "SEMB_EGEOM", -5: "SEMB_EBREAKDOWN",
          -6: "SEMB_EMATCH", -7: "SEMB_ENOTFOUND"}

# every symbol include/semb200.h declares (tests check that the library exports all of them)
SYMBOLS = ["semb_gll", "semb_setup", "semb_destroy", "semb_last_error", "semb_mesh_info", "semb_apply_axhelm",
           "semb_set_geometry_mode", "semb_gather_scatter", "semb_apply_mask", "semb_assemble_rhs", "semb_apply_operator", "semb_jacobi_diag",
           "semb_pcg_solve", "semb_step_solve", "semb_mg_vcycle", "semb_mg_transfer", "semb_mg_level_size", "semb_estimate_lmax", "semb_cheb_jacobi", "semb_schwarz_apply", "semb_publish_field", "semb_publish_state",
           "semb_export_field", "semb_field_minmax_hist", "semb_vector_magnitude_minmax_hist", "semb_gradient", "semb_weak_divergence", "semb_flow_explicit_terms", "semb_boussinesq_step", "semb_colormap_apply", "semb_image_slice", "semb_image_isosurface", "semb_apply_axhelm_host", "semb_pcg_solve_host", "semb_read_device", "semb_stream_probe", "semb_version",
           "semb_field_minmax_hist_noalloc", "semb_noalloc_last_error"]


class SembError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{ERRORS.get(code, code)}: {msg}")
        self.code = code


class Info(C.Structure):
    _fields_ = [("E", C.c_int64), ("N", C.c_int32), ("n1", C.c_int32), ("Np", C.c_int64), ("n", C.c_int64),
                ("n_unique", C.c_int64), ("n_shared", C.c_int64), ("n_gs", C.c_int64), ("tol", C.c_double),
                ("gid", C.c_void_p), ("geo", C.c_void_p), ("invmult", C.c_void_p), ("gs_offsets", C.c_void_p),
                ("gs_ids", C.c_void_p)]


class PcgOpts(C.Structure):
    _fields_ = [("lam", C.c_double), ("dirichlet_tags", C.c_uint32), ("precond", C.c_int32),
                ("cheb_degree", C.c_int32), ("cheb_lmax", C.c_double), ("rtol", C.c_double), ("atol", C.c_double),
                ("maxit", C.c_int32), ("x0_is_zero", C.c_int32), ("check_every", C.c_int32), ("profile", C.c_int32),
                ("mg_nlevels", C.c_int32), ("mg_orders", C.c_int32 * 8), ("mg_smooth_degree", C.c_int32),
                ("mg_coarse_degree", C.c_int32), ("mg_lmax", C.c_double * 8), ("mg_smoother_kind", C.c_int32), ("pad_", C.c_int32),
                ("mg_coarse_lmin_frac", C.c_double), ("null_mean", C.c_int32), ("mg_fp32", C.c_int32), ("mg_schwarz", C.c_int32), ("pad2_", C.c_int32)]


def _mg_fill(o, mg_orders=None, mg_smooth=0, mg_coarse=0, mg_lmax=None, mg_kind=1, mg_coarse_frac=0.0):
    """p-multigrid fields of a PcgOpts (precond == 3)."""
    orders = list(mg_orders) if mg_orders is not None else []
    o.mg_nlevels = len(orders)
    for i, v in enumerate(orders):
        o.mg_orders[i] = int(v)
    o.mg_smooth_degree, o.mg_coarse_degree = int(mg_smooth), int(mg_coarse)
    for i, v in enumerate(mg_lmax or []):
        o.mg_lmax[i] = float(v)
    o.mg_smoother_kind = int(mg_kind)
    o.mg_coarse_lmin_frac = float(mg_coarse_frac)
    return o


class PcgStats(C.Structure):
    _fields_ = [("iters", C.c_int32), ("status", C.c_int32), ("b_norm", C.c_double), ("r0_norm", C.c_double),
                ("r_norm", C.c_double), ("lmax_used", C.c_double), ("hist", C.c_void_p), ("hist_len", C.c_int32),
                ("profiled", C.c_int32), ("axhelm_ms", C.c_double), ("launches", C.c_int64)]


class SolveItem(C.Structure):
    _fields_ = [("opts", PcgOpts), ("b", C.c_void_p), ("x", C.c_void_p)]


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class Allocator(C.Structure):
    """semb_allocator: every device buffer the library owns comes from alloc(bytes, user) / goes to free(ptr, user)."""
    _fields_ = [("alloc", ALLOC_FN), ("free", FREE_FN), ("user", C.c_void_p)]


class TorchAllocator:
    """semb_allocator backed by torch's caching allocator: the library then owns no memory outside torch's pool."""

    def __init__(self):
        import torch
        self.live = {}
        self.peak_bytes = self.calls = 0

        def _alloc(nbytes, _user):
            try:
                t = torch.empty(int(nbytes), dtype=torch.uint8, device="cuda")
            except RuntimeError:
                return None
            self.live[t.data_ptr()] = t
            self.calls += 1
            self.peak_bytes = max(self.peak_bytes, sum(v.numel() for v in self.live.values()))
            return t.data_ptr()

        def _free(ptr, _user):
            self.live.pop(ptr, None)

        self._a, self._f = ALLOC_FN(_alloc), FREE_FN(_free)           # keep the thunks alive
        self.struct = Allocator(self._a, self._f, None)


class FieldDesc(C.Structure):
    _fields_ = [("name", C.c_char_p), ("ptr", C.c_void_p), ("dtype", C.c_int32), ("memspace", C.c_int32),
                ("count", C.c_int64), ("stride", C.c_int64), ("cycle", C.c_int64), ("time", C.c_double)]


class FlowOpts(C.Structure):
    _fields_ = [("Ra", C.c_double), ("Pr", C.c_double), ("dt", C.c_double), ("tags_u", C.c_uint32), ("tags_T", C.c_uint32),
                ("rtol", C.c_double), ("precond_p", C.c_int32), ("precond_u", C.c_int32), ("mg_fp32", C.c_int32), ("maxit", C.c_int32),
                ("mg_schwarz", C.c_int32), ("pad_", C.c_int32), ("forcing", C.c_void_p * 4)]


class FlowStateC(C.Structure):
    _fields_ = [("u", C.c_void_p * 3), ("theta", C.c_void_p), ("p", C.c_void_p), ("u1", C.c_void_p * 3), ("theta1", C.c_void_p),
                ("N1", C.c_void_p * 4), ("C1", C.c_void_p * 3), ("step_index", C.c_int64)]


class FlowStats(C.Structure):
    _fields_ = [("iters", C.c_int32 * 5), ("status", C.c_int32 * 5)]


class FlowState:
    """device arrays of a Boussinesq run (semb_flow_state): torch owns the memory, the library the arithmetic"""

    def __init__(self, n):
        import torch
        z = lambda: torch.zeros(n, dtype=torch.float64, device="cuda")
        self.u = [z() for _ in range(3)]; self.theta = z(); self.p = z()
        self.u1 = [z() for _ in range(3)]; self.theta1 = z()
        self.N1 = [z() for _ in range(4)]; self.C1 = [z() for _ in range(3)]
        self.c = FlowStateC()
        for i in range(3):
            self.c.u[i] = self.u[i].data_ptr(); self.c.u1[i] = self.u1[i].data_ptr(); self.c.C1[i] = self.C1[i].data_ptr()
        for i in range(4):
            self.c.N1[i] = self.N1[i].data_ptr()
        self.c.theta, self.c.p, self.c.theta1 = self.theta.data_ptr(), self.p.data_ptr(), self.theta1.data_ptr()
        self.c.step_index = 0


class ImageView(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("origin", C.c_double * 3), ("u", C.c_double * 3),
                ("v", C.c_double * 3), ("du", C.c_double), ("dv", C.c_double), ("depth_lo", C.c_double), ("depth_hi", C.c_double)]


class Colormap(C.Structure):
    _fields_ = [("lo", C.c_double), ("hi", C.c_double), ("ncolors", C.c_int32), ("rgb", (C.c_uint8 * 3) * 16),
                ("background", C.c_uint32)]


def image_view(width, height, origin, u, v, du, dv, depth_lo=0.0, depth_hi=1.0):
    vw = ImageView(width, height)
    for c in range(3):
        vw.origin[c], vw.u[c], vw.v[c] = float(origin[c]), float(u[c]), float(v[c])
    vw.du, vw.dv, vw.depth_lo, vw.depth_hi = float(du), float(dv), float(depth_lo), float(depth_hi)
    return vw


def colormap(lo, hi, colors, background=0xff000000):
    cm = Colormap(float(lo), float(hi), len(colors))
    for m, col in enumerate(colors):
        for c in range(3):
            cm.rgb[m][c] = int(col[c])
    cm.background = int(background)
    return cm


_lib = None


def lib():
    """Load libsemb200.so (build it with `python -m paper_2501_13240_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2501_13240_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.semb_last_error.restype = C.c_char_p
        L.semb_last_error.argtypes = [C.c_void_p]
        L.semb_version.restype = C.c_char_p
        _lib = L
    return _lib


def version():
    return lib().semb_version().decode()


def gll(N):
    """(xi, rho, D) of order N from the library (host)."""
    xi = np.zeros(N + 1); rho = np.zeros(N + 1); D = np.zeros((N + 1, N + 1))
    rc = lib().semb_gll(C.c_int(N), xi.ctypes.data_as(C.c_void_p), rho.ctypes.data_as(C.c_void_p),
                        D.ctypes.data_as(C.c_void_p))
    if rc:
        raise SembError(rc, f"semb_gll(N={N})")
    return xi, rho, D


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dp(t):
    """device pointer of a contiguous CUDA tensor (or None)."""
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "expected a contiguous CUDA tensor"
    return C.c_void_p(t.data_ptr())


class Mesh:
    """Handle of one mesh on the current CUDA device (semb_setup ... semb_destroy)."""

    def __init__(self, E, N, x, y, z, face_tag, period, gid=None, allocator=None):
        import torch
        self._allocator = allocator                                    # TorchAllocator (kept alive with the handle) or None
        assert x.dtype == torch.float64 and y.dtype == torch.float64 and z.dtype == torch.float64
        self._h = C.c_void_p()
        ft = np.ascontiguousarray(face_tag, dtype=np.int32)
        per = np.ascontiguousarray(period, dtype=np.float64)
        assert ft.size == 6 * E and x.numel() == E * (N + 1) ** 3
        rc = lib().semb_setup(C.c_int64(E), C.c_int(N), _dp(x), _dp(y), _dp(z), ft.ctypes.data_as(C.c_void_p),
                              per.ctypes.data_as(C.c_void_p), _dp(gid),
                              C.byref(allocator.struct) if allocator is not None else None, _stream(), C.byref(self._h))
        if rc:
            raise SembError(rc, lib().semb_last_error(None).decode())
        self.info = Info()
        self._check(lib().semb_mesh_info(self._h, C.byref(self.info)))
        self.E, self.N, self.n, self.Np = int(self.info.E), int(self.info.N), int(self.info.n), int(self.info.Np)
        self.n_unique, self.n_shared, self.n_gs = int(self.info.n_unique), int(self.info.n_shared), int(self.info.n_gs)
        self._keep = []

    def _check(self, rc):
        if rc < 0:
            raise SembError(rc, lib().semb_last_error(self._h).decode())
        return rc

    def close(self):
        if self._h:
            lib().semb_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- read-only views of handle-owned arrays (copied to host for tests) -------------------
    def _to_host(self, ptr, count, dtype):
        out = np.empty(count, dtype=dtype)
        if count:
            self._check(lib().semb_read_device(C.c_void_p(ptr), out.ctypes.data_as(C.c_void_p), C.c_size_t(out.nbytes)))
        return out

    def gid_host(self):
        return self._to_host(self.info.gid, self.n, np.int32)

    def geo_host(self):
        return self._to_host(self.info.geo, self.n * 7, np.float64).reshape(self.E, 7, self.Np)

    def invmult_host(self):
        return self._to_host(self.info.invmult, self.n, np.float64)

    def gs_lists_host(self):
        return (self._to_host(self.info.gs_offsets, self.n_gs + 1, np.int32),
                self._to_host(self.info.gs_ids, self.n_shared, np.int32))

    # ---- the hot path ------------------------------------------------------------------------
    def apply_axhelm(self, u, w, lam=0.0, lam0=None, lam1=None, nfields=1):
        self._check(lib().semb_apply_axhelm(self._h, C.c_double(lam), _dp(lam0), _dp(lam1), _dp(u), _dp(w),
                                            C.c_int(nfields), _stream()))
        return w

    def set_geometry_mode(self, mode, tol=0.0):
        """0 stored fp64 factors, 1 float-stored factors, 2 affine elements, 3 trilinear elements (semb_set_geometry_mode).
        Returns the measured (trilinear, affine) deviations, (-1, -1) if they were never measured."""
        dev = (C.c_double * 2)(-1.0, -1.0)
        self._check(lib().semb_set_geometry_mode(self._h, C.c_int(mode), C.c_double(tol), dev if mode >= 2 else None, _stream()))
        return dev[0], dev[1]

    def gather_scatter(self, w, nfields=1):
        self._check(lib().semb_gather_scatter(self._h, _dp(w), C.c_int(nfields), _stream()))
        return w

    def apply_mask(self, w, tags, nfields=1):
        self._check(lib().semb_apply_mask(self._h, C.c_uint32(tags), _dp(w), C.c_int(nfields), _stream()))
        return w

    def assemble_rhs(self, f, b, tags):
        self._check(lib().semb_assemble_rhs(self._h, C.c_uint32(tags), _dp(f), _dp(b), _stream()))
        return b

    def apply_operator(self, v, out, lam, tags):
        self._check(lib().semb_apply_operator(self._h, C.c_double(lam), C.c_uint32(tags), _dp(v), _dp(out), _stream()))
        return out

    def jacobi_diag(self, dinv_out, lam, tags):
        self._check(lib().semb_jacobi_diag(self._h, C.c_double(lam), C.c_uint32(tags), _dp(dinv_out), _stream()))
        return dinv_out

    def pcg_solve(self, b, x, lam=0.0, tags=0, precond=1, cheb_degree=2, cheb_lmax=0.0, rtol=1e-10, atol=0.0,
                  maxit=10000, x0_is_zero=True, check_every=0, hist_len=0, profile=False, mg_orders=None, mg_smooth=0,
                  mg_coarse=0, mg_lmax=None, mg_kind=1, mg_coarse_frac=0.0, null_mean=False, mg_fp32=False, mg_schwarz=False):
        """Returns dict(iters, status, b_norm, r0_norm, r_norm, lmax_used, hist).  precond: 0 none, 1 Jacobi,
        2 Chebyshev-Jacobi, 3 p-multigrid V-cycle (mg_orders e.g. [7, 3, 1]; None = default)."""
        o = PcgOpts(lam, tags, precond, cheb_degree, cheb_lmax, rtol, atol, maxit, 1 if x0_is_zero else 0, check_every, 1 if profile else 0)
        _mg_fill(o, mg_orders, mg_smooth, mg_coarse, mg_lmax, mg_kind, mg_coarse_frac)
        o.null_mean = 1 if null_mean else 0
        o.mg_fp32 = 1 if mg_fp32 else 0
        o.mg_schwarz = 1 if mg_schwarz else 0
        hist = np.zeros(max(hist_len, 1))
        st = PcgStats()
        st.hist = hist.ctypes.data_as(C.c_void_p).value if hist_len > 0 else None
        st.hist_len = hist_len
        rc = self._check(lib().semb_pcg_solve(self._h, C.byref(o), _dp(b), _dp(x), C.byref(st), _stream()))
        return dict(iters=int(st.iters), status=int(rc), b_norm=st.b_norm, r0_norm=st.r0_norm, r_norm=st.r_norm,
                    lmax_used=st.lmax_used, hist=hist[:min(hist_len, st.iters + 1)], axhelm_ms=st.axhelm_ms,
                    profiled=int(st.profiled), launches=int(st.launches))

    def step_solve(self, solves):
        """One time step's solves back to back (semb_step_solve).  solves: list of dicts with keys b, x (device
        tensors) and the pcg_solve keyword options.  Returns (status, [dict(iters, status, r_norm, b_norm)])."""
        k = len(solves)
        items = (SolveItem * max(k, 1))()
        stats = (PcgStats * max(k, 1))()
        for i, sv in enumerate(solves):
            o = PcgOpts(sv.get("lam", 0.0), sv.get("tags", 0), sv.get("precond", 1), sv.get("cheb_degree", 2),
                        sv.get("cheb_lmax", 0.0), sv.get("rtol", 1e-10), sv.get("atol", 0.0), sv.get("maxit", 10000),
                        1 if sv.get("x0_is_zero", True) else 0, sv.get("check_every", 0), 0)
            _mg_fill(o, sv.get("mg_orders"), sv.get("mg_smooth", 0), sv.get("mg_coarse", 0), sv.get("mg_lmax"), sv.get("mg_kind", 1),
                     sv.get("mg_coarse_frac", 0.0))
            o.null_mean = 1 if sv.get("null_mean", False) else 0
            o.mg_fp32 = 1 if sv.get("mg_fp32", False) else 0
            o.mg_schwarz = 1 if sv.get("mg_schwarz", False) else 0
            items[i].opts = o
            items[i].b = _dp(sv["b"]).value
            items[i].x = _dp(sv["x"]).value
            stats[i].hist = None
            stats[i].hist_len = 0
        rc = self._check(lib().semb_step_solve(self._h, C.c_int(k), items, stats, _stream()))
        return int(rc), [dict(iters=int(st.iters), status=int(st.status), r_norm=st.r_norm, b_norm=st.b_norm,
                              launches=int(st.launches)) for st in stats[:k]]

    def _mg_opts(self, lam, tags, mg_orders, mg_smooth, mg_coarse, mg_lmax, mg_kind=1, mg_coarse_frac=0.0):
        o = PcgOpts(lam, tags, 3, 0, 0.0, 0.0, 0.0, 0, 1, 0, 0)
        return _mg_fill(o, mg_orders, mg_smooth, mg_coarse, mg_lmax, mg_kind, mg_coarse_frac)

    def schwarz_apply(self, r, out, lam=0.0, tags=0):
        self._check(lib().semb_schwarz_apply(self._h, C.c_double(lam), C.c_uint32(tags), _dp(r), _dp(out), _stream()))
        return out

    def mg_vcycle(self, r, z, lam=0.0, tags=0, mg_orders=None, mg_smooth=0, mg_coarse=0, mg_lmax=None, mg_kind=1,
                  mg_coarse_frac=0.0, mg_fp32=False, mg_schwarz=False):
        """z = one p-multigrid V-cycle applied to r; returns the Chebyshev bounds used per level."""
        o = self._mg_opts(lam, tags, mg_orders, mg_smooth, mg_coarse, mg_lmax, mg_kind, mg_coarse_frac)
        o.mg_fp32 = 1 if mg_fp32 else 0
        o.mg_schwarz = 1 if mg_schwarz else 0
        used = (C.c_double * 8)()
        self._check(lib().semb_mg_vcycle(self._h, C.byref(o), _dp(r), _dp(z), used, _stream()))
        nl = len(mg_orders) if mg_orders is not None else 8
        return [used[i] for i in range(nl) if used[i] > 0.0]

    def mg_level_size(self, level, lam=0.0, tags=0, mg_orders=None):
        o = self._mg_opts(lam, tags, mg_orders, 0, 0, None)
        lib().semb_mg_level_size.restype = C.c_int64
        return int(self._check(lib().semb_mg_level_size(self._h, C.byref(o), C.c_int(level))))

    def mg_transfer(self, level, restrict, vin, vout, lam=0.0, tags=0, mg_orders=None):
        o = self._mg_opts(lam, tags, mg_orders, 0, 0, [1.0] * 8)
        self._check(lib().semb_mg_transfer(self._h, C.byref(o), C.c_int(level), C.c_int(1 if restrict else 0), _dp(vin),
                                           _dp(vout), _stream()))

    def pcg_solve_host(self, b_host, x_host, lam=0.0, tags=0, precond=1, cheb_degree=2, cheb_lmax=0.0, rtol=1e-10,
                       atol=0.0, maxit=10000, check_every=0):
        """pcg_solve with HOST buffers (torch CPU tensors, ideally pinned, or numpy arrays)."""
        def hp(a):
            return C.c_void_p(a.data_ptr()) if hasattr(a, "data_ptr") else a.ctypes.data_as(C.c_void_p)
        o = PcgOpts(lam, tags, precond, cheb_degree, cheb_lmax, rtol, atol, maxit, 1, check_every, 0)
        st = PcgStats()
        rc = self._check(lib().semb_pcg_solve_host(self._h, C.byref(o), hp(b_host), hp(x_host), C.byref(st), _stream()))
        return dict(iters=int(st.iters), status=int(rc), r_norm=st.r_norm, b_norm=st.b_norm, launches=int(st.launches))

    def estimate_lmax(self, v0, lam, tags, steps=10):
        out = C.c_double(0.0)
        self._check(lib().semb_estimate_lmax(self._h, C.c_double(lam), C.c_uint32(tags), _dp(v0), C.c_int(steps),
                                             C.byref(out), _stream()))
        return out.value

    def cheb_jacobi(self, r, z, lam, tags, k, lmax):
        self._check(lib().semb_cheb_jacobi(self._h, C.c_double(lam), C.c_uint32(tags), C.c_int(k), C.c_double(lmax),
                                           _dp(r), _dp(z), _stream()))
        return z

    # ---- in-situ hand-off --------------------------------------------------------------------
    def publish_field(self, name, t):
        self._keep.append(t)
        self._check(lib().semb_publish_field(self._h, name.encode(), _dp(t), C.c_int64(t.numel())))

    def publish_state(self, cycle, time):
        self._check(lib().semb_publish_state(self._h, C.c_int64(cycle), C.c_double(time), _stream()))

    def export_field(self, name):
        d = FieldDesc()
        self._check(lib().semb_export_field(self._h, name.encode(), C.byref(d)))
        return d

    def gradient(self, phi, gx, gy, gz):
        self._check(lib().semb_gradient(self._h, _dp(phi), _dp(gx), _dp(gy), _dp(gz), _stream()))

    def weak_divergence(self, gx, gy, gz, out):
        self._check(lib().semb_weak_divergence(self._h, _dp(gx), _dp(gy), _dp(gz), _dp(out), _stream()))

    def flow_explicit_terms(self, ux, uy, uz, theta, N4, omega3, forcing=None):
        f = (C.c_void_p * 4)(*[(t.data_ptr() if t is not None else None) for t in (forcing or [None] * 4)])
        self._check(lib().semb_flow_explicit_terms(self._h, _dp(ux), _dp(uy), _dp(uz), _dp(theta), f if forcing else None, _dp(N4), _dp(omega3), _stream()))

    def boussinesq_step(self, state, Ra, Pr, dt, tags_u, tags_T, rtol=1e-10, precond_p=3, precond_u=1, mg_fp32=False, maxit=0, forcing=None,
                        mg_schwarz=False):
        """one time step on `state` (FlowState); returns (status, iterations of the pressure, u_x, u_y, u_z, theta solves)"""
        o = FlowOpts(Ra, Pr, dt, tags_u, tags_T, rtol, precond_p, precond_u, 1 if mg_fp32 else 0, maxit, 1 if mg_schwarz else 0, 0)
        for i, t in enumerate(forcing or []):
            o.forcing[i] = t.data_ptr() if t is not None else None
        st = FlowStats()
        rc = self._check(lib().semb_boussinesq_step(self._h, C.byref(o), C.byref(state.c), C.byref(st), _stream()))
        return int(rc), [int(v) for v in st.iters]

    def image_slice(self, desc, view, cmap, key, rgba=None):
        """planar slice of an exported field into key (uint64/int64 [H*W]) and rgba (int32/uint32 [H*W] or None)"""
        self._check(lib().semb_image_slice(self._h, C.byref(desc), C.byref(view), C.byref(cmap), _dp(key), _dp(rgba), _stream()))

    def image_isosurface(self, desc, iso, color_desc, view, cmap, light, key, rgba=None):
        lt = (C.c_double * 3)(*[float(v) for v in light])
        self._check(lib().semb_image_isosurface(self._h, C.byref(desc), C.c_double(iso), C.byref(color_desc) if color_desc is not None else None,
                                                C.byref(view), C.byref(cmap), lt, _dp(key), _dp(rgba), _stream()))

    def apply_axhelm_host(self, u_host, w_host, lam=0.0):
        """End-to-end call with HOST numpy buffers (copies inside the library)."""
        self._check(lib().semb_apply_axhelm_host(self._h, C.c_double(lam), u_host.ctypes.data_as(C.c_void_p),
                                                 w_host.ctypes.data_as(C.c_void_p)))
        return w_host


def stream_probe(src, dst, nread):
    """measurement aid: dst[l] = sum_c src[c*n + l] (semb_stream_probe)"""
    rc = lib().semb_stream_probe(_dp(src), _dp(dst), C.c_int64(dst.numel()), C.c_int(nread), _stream())
    if rc:
        raise SembError(rc, "semb_stream_probe")


def vector_magnitude_minmax_hist(dx, dy, dz, nbins, lo, hi, minmax_dev, hist_dev):
    """min / max / histogram of |v| from the three component descriptors, computed on the fly (nothing written)"""
    rc = lib().semb_vector_magnitude_minmax_hist(C.byref(dx), C.byref(dy), C.byref(dz), C.c_int(nbins), C.c_double(lo), C.c_double(hi),
                                                 _dp(minmax_dev), _dp(hist_dev), _stream())
    if rc:
        raise SembError(rc, "semb_vector_magnitude_minmax_hist")


def colormap_apply(cmap, val, rgba):
    rc = lib().semb_colormap_apply(C.byref(cmap), _dp(val), C.c_int64(val.numel()), _dp(rgba), _stream())
    if rc:
        raise SembError(rc, "semb_colormap_apply")


def field_minmax_hist(desc, nbins, lo, hi, minmax_dev, hist_dev):
    """In-device consumer: minmax_dev (float64[2]) and hist_dev (int64/uint64[nbins]) CUDA tensors."""
    rc = lib().semb_field_minmax_hist(C.byref(desc), C.c_int(nbins), C.c_double(lo), C.c_double(hi), _dp(minmax_dev),
                                      _dp(hist_dev), _stream())
    if rc:
        raise SembError(rc, "semb_field_minmax_hist")


NOALLOC_MAX_BINS = 4096          # include/semb200.h: SEMB_NOALLOC_MAX_BINS


def field_minmax_hist_noalloc(desc, nbins, lo, hi, minmax_dev, hist_dev):
    """field_minmax_hist through the entry point that allocates nothing (static device scratch, nbins <= NOALLOC_MAX_BINS;
    calls that overlap on the GPU race on that scratch: include/semb200.h)."""
    L = lib()
    L.semb_noalloc_last_error.restype = C.c_char_p
    rc = L.semb_field_minmax_hist_noalloc(C.byref(desc), C.c_int(nbins), C.c_double(lo), C.c_double(hi), _dp(minmax_dev),
                                          _dp(hist_dev), _stream())
    if rc:
        raise SembError(rc, L.semb_noalloc_last_error().decode())
