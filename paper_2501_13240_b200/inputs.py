"""Seeded synthetic inputs shared by the CUDA path and the oracle (numpy only).

This module holds NONE of the method's arithmetic: it only produces input buffers (node
coordinates, face tags, random vectors, right-hand-side source fields).  The GLL parameters
`xi` at which nodes are placed are passed IN by the caller (tests pass the oracle's, the
product path passes the library's `semb_gll`), so nothing here restates the method.

The meshes stand in for the paper's RBC cells, none of which are available:
  * boxes with periodic x,y and walls at z = 0,1 (§4.1), optionally with the
    tanh vertical clustering of the element map (§4.1);
  * a cylindrical cell of aspect ratio 1 (BASELINE.json configs[2],[4]) as a 5-block
    "butterfly" O-grid (reading R5; a single-block square->disk map has J = 0 at
    four nodes).
Recipe and seeds: DESIGN.md "Input recipe".

Layout everywhere: local node l = e*Np + k*n1^2 + j*n1 + i, i fastest.
Face order per element: r-, r+, s-, s+, t-, t+ ; tag 0 = none, 1 = plates z=0/1, 2 = side wall.
"""
import numpy as np

BASE_SEED = 250113240
_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def splitmix64(seed, idx):
    """Counter-based splitmix64: idx (uint64 array) -> uint64 array."""
    with np.errstate(over="ignore"):
        z = np.uint64(seed) + (idx.astype(np.uint64) + np.uint64(1)) * np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def uniform(seed, n, lo=-1.0, hi=1.0, chunk=1 << 24):
    """n doubles uniform in [lo, hi): u01 = (z >> 11) * 2^-53 per index."""
    out = np.empty(n, dtype=np.float64)
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        z = splitmix64(seed, np.arange(s, e, dtype=np.uint64))
        out[s:e] = (z >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)
    if lo != 0.0 or hi != 1.0:
        out *= (hi - lo); out += lo
    return out


def tanh_layers(nz, s):
    """Element boundaries z_k = (1 + tanh(s (2k/nz - 1)) / tanh(s)) / 2 (reading R6)."""
    k = np.arange(nz + 1, dtype=np.float64)
    zb = 0.5 * (1.0 + np.tanh(s * (2.0 * k / nz - 1.0)) / np.tanh(s))
    zb[0] = 0.0; zb[-1] = 1.0
    return zb


class Mesh:
    def __init__(self, E, N, x, y, z, face_tag, period, name, meta=None):
        self.E, self.N = int(E), int(N)
        self.Np = (N + 1) ** 3
        self.n = self.E * self.Np
        self.x, self.y, self.z = x, y, z
        self.face_tag = face_tag
        self.period = np.asarray(period, dtype=np.float64)
        self.name = name
        self.meta = meta or {}


def box_mesh(nx, ny, nz, N, xi, periodic=(False, False, False), deform=0.0, zstretch=0.0, name="box"):
    """Unit cube of nx*ny*nz hexahedra, element e = (ez*ny + ey)*nx + ex.

    Nodes come from the integer lattice index ((ex + a_i) * hx with a = (xi+1)/2, a_0 = 0 and
    a_N = 1 exactly), so copies of a shared node are bitwise equal.  `deform` displaces every
    node in all three coordinates by deform*h*sin(2 pi x) sin(2 pi y) sin(2 pi z) evaluated at
    the undisplaced position (zero on the boundary).  `zstretch` > 0 clusters the element
    layers towards z = 0,1 with tanh_layers.
    """
    n1 = N + 1
    a = (np.asarray(xi, dtype=np.float64) + 1.0) * 0.5
    E = nx * ny * nz
    hx, hy = 1.0 / nx, 1.0 / ny
    X1 = (np.arange(nx, dtype=np.float64)[:, None] + a[None, :]) * hx          # [nx, n1]
    Y1 = (np.arange(ny, dtype=np.float64)[:, None] + a[None, :]) * hy
    if zstretch > 0.0:
        zb = tanh_layers(nz, zstretch)
        Z1 = zb[:-1, None] * (1.0 - a[None, :]) + zb[1:, None] * a[None, :]
    else:
        Z1 = (np.arange(nz, dtype=np.float64)[:, None] + a[None, :]) * (1.0 / nz)
    shape = (nz, ny, nx, n1, n1, n1)                                           # ez,ey,ex,k,j,i
    x = np.broadcast_to(X1[None, None, :, None, None, :], shape).reshape(-1).copy()
    y = np.broadcast_to(Y1[None, :, None, None, :, None], shape).reshape(-1).copy()
    z = np.broadcast_to(Z1[:, None, None, :, None, None], shape).reshape(-1).copy()
    if deform != 0.0:
        h = 1.0 / max(nx, ny, nz)
        d = np.sin(2 * np.pi * x); d *= np.sin(2 * np.pi * y); d *= np.sin(2 * np.pi * z); d *= deform * h
        x += d; y += d; z += d
    ft = np.zeros((nz, ny, nx, 6), dtype=np.int32)
    if not periodic[0]:
        ft[:, :, 0, 0] = 2; ft[:, :, nx - 1, 1] = 2
    if not periodic[1]:
        ft[:, 0, :, 2] = 2; ft[:, ny - 1, :, 3] = 2
    if not periodic[2]:
        ft[0, :, :, 4] = 1; ft[nz - 1, :, :, 5] = 1
    period = [1.0 if p else 0.0 for p in periodic]
    return Mesh(E, N, x, y, z, ft.reshape(-1), period, name,
                dict(nx=nx, ny=ny, nz=nz, periodic=tuple(periodic), deform=deform, zstretch=zstretch))


def trilinear_box_mesh(nx, ny, nz, N, xi, jitter=0.2, seed=BASE_SEED + 77, zstretch=0.0, name="box_trilinear"):
    """Unit cube of nx*ny*nz hexahedra with STRAIGHT edges that are not parallelepipeds: the interior lattice vertices are
    displaced by jitter * h * U[-1,1) per coordinate (seeded, counter RNG on the vertex index; boundary vertices stay), and
    every node is the trilinear interpolant of its element's 8 vertices at the GLL parameters -- the class of elements whose
    geometric factors can be rebuilt from 8 vertices.  jitter = 0 gives affine bricks."""
    n1 = N + 1
    a = (np.asarray(xi, dtype=np.float64) + 1.0) * 0.5
    zb = tanh_layers(nz, zstretch) if zstretch > 0.0 else np.arange(nz + 1, dtype=np.float64) / nz
    V = np.empty((nz + 1, ny + 1, nx + 1, 3))
    V[..., 0] = (np.arange(nx + 1, dtype=np.float64) / nx)[None, None, :]
    V[..., 1] = (np.arange(ny + 1, dtype=np.float64) / ny)[None, :, None]
    V[..., 2] = zb[:, None, None]
    if jitter != 0.0:
        hmin = np.array([1.0 / nx, 1.0 / ny, np.diff(zb).min()])
        d = uniform(seed, V.size).reshape(V.shape) * (jitter * hmin)[None, None, None, :]
        d[0] = 0; d[-1] = 0; d[:, 0] = 0; d[:, -1] = 0; d[:, :, 0] = 0; d[:, :, -1] = 0
        V = V + d
    w = np.stack([1.0 - a, a])                                                   # [2, n1]
    out = []
    for c in range(3):
        acc = np.zeros((nz, ny, nx, n1, n1, n1))
        for vk in range(2):
            for vj in range(2):
                for vi in range(2):
                    corner = V[vk:vk + nz, vj:vj + ny, vi:vi + nx, c]
                    acc += corner[..., None, None, None] * (w[vk][:, None, None] * w[vj][None, :, None] * w[vi][None, None, :])
        out.append(acc.reshape(-1))
    ft = np.zeros((nz, ny, nx, 6), dtype=np.int32)
    ft[:, :, 0, 0] = 2; ft[:, :, nx - 1, 1] = 2; ft[:, 0, :, 2] = 2; ft[:, ny - 1, :, 3] = 2
    ft[0, :, :, 4] = 1; ft[nz - 1, :, :, 5] = 1
    return Mesh(nx * ny * nz, N, out[0], out[1], out[2], ft.reshape(-1), [0.0, 0.0, 0.0], name,
                dict(nx=nx, ny=ny, nz=nz, jitter=jitter, zstretch=zstretch))


def _east_block(zeta, eta, c, R):
    """point(zeta, eta) = (1-zeta) (c, c eta) + zeta R (cos(pi eta/4), sin(pi eta/4))."""
    px = (1.0 - zeta) * c + zeta * R * np.cos(np.pi * eta / 4.0)
    py = (1.0 - zeta) * c * eta + zeta * R * np.sin(np.pi * eta / 4.0)
    return px, py


def ogrid_mesh(n_c, n_r, n_z, N, xi, R=0.5, c=0.2, zstretch=2.5, name="ogrid"):
    """Cylinder of radius R, height 1: central square [-c,c]^2 of n_c x n_c elements plus four
    outer blocks of n_r (radial) x n_c (tangential) elements, n_z tanh-clustered layers.
    Per layer the element order is: centre (ey*n_c + ex), then east, north, west, south blocks
    (each es*n_r + er).  Outer blocks: local r = radial, s = tangential (counter-clockwise),
    t = z.  Seam nodes of neighbouring blocks come from different formulas and agree only to
    rounding -- this exercises the coordinate-matching tolerance of the numbering."""
    n1 = N + 1
    a = (np.asarray(xi, dtype=np.float64) + 1.0) * 0.5
    per_layer = n_c * n_c + 4 * n_r * n_c
    E = per_layer * n_z
    # --- one layer, 2-D (x, y) per element [per_layer, n1(j), n1(i)]
    X2 = np.empty((per_layer, n1, n1)); Y2 = np.empty((per_layer, n1, n1))
    g = -c + 2.0 * c * (np.arange(n_c, dtype=np.float64)[:, None] + a[None, :]) / n_c       # [n_c, n1]
    cx = np.broadcast_to(g[None, :, None, :], (n_c, n_c, n1, n1))                            # ey,ex,j,i -> x(ex,i)
    cy = np.broadcast_to(g[:, None, :, None], (n_c, n_c, n1, n1))
    X2[:n_c * n_c] = cx.reshape(-1, n1, n1); Y2[:n_c * n_c] = cy.reshape(-1, n1, n1)
    zeta = (np.arange(n_r, dtype=np.float64)[:, None] + a[None, :]) / n_r                    # [n_r, n1]
    eta = -1.0 + 2.0 * (np.arange(n_c, dtype=np.float64)[:, None] + a[None, :]) / n_c        # [n_c, n1]
    Zt = np.broadcast_to(zeta[None, :, None, :], (n_c, n_r, n1, n1))                         # es,er,j,i
    Et = np.broadcast_to(eta[:, None, :, None], (n_c, n_r, n1, n1))
    ex_, ey_ = _east_block(Zt, Et, c, R)
    ex_ = ex_.reshape(-1, n1, n1); ey_ = ey_.reshape(-1, n1, n1)
    nb = n_r * n_c
    o = n_c * n_c
    for q, (bx, by) in enumerate([(ex_, ey_), (-ey_, ex_), (-ex_, -ey_), (ey_, -ex_)]):      # rotations by 90 deg
        X2[o + q * nb:o + (q + 1) * nb] = bx; Y2[o + q * nb:o + (q + 1) * nb] = by
    zb = tanh_layers(n_z, zstretch) if zstretch > 0 else np.linspace(0.0, 1.0, n_z + 1)
    Z1 = zb[:-1, None] * (1.0 - a[None, :]) + zb[1:, None] * a[None, :]                      # [n_z, n1]
    shape = (n_z, per_layer, n1, n1, n1)                                                      # ez, e2, k, j, i
    x = np.broadcast_to(X2[None, :, None, :, :], shape).reshape(-1).copy()
    y = np.broadcast_to(Y2[None, :, None, :, :], shape).reshape(-1).copy()
    z = np.broadcast_to(Z1[:, None, :, None, None], shape).reshape(-1).copy()
    ft = np.zeros((n_z, per_layer, 6), dtype=np.int32)
    ft[0, :, 4] = 1; ft[n_z - 1, :, 5] = 1
    outer = np.zeros(per_layer, dtype=bool)
    for q in range(4):
        idx = o + q * nb + np.arange(n_c) * n_r + (n_r - 1)
        outer[idx] = True
    ft[:, outer, 1] = 2
    return Mesh(E, N, x, y, z, ft.reshape(-1), [0.0, 0.0, 0.0], name,
                dict(n_c=n_c, n_r=n_r, n_z=n_z, R=R, c=c, zstretch=zstretch))


def ogrid_unique_nodes(n_c, n_r, n_z, N):
    """closed form: [(n_c N + 1)^2 + 4 n_r n_c N^2] (n_z N + 1)  (dagger)."""
    return ((n_c * N + 1) ** 2 + 4 * n_r * n_c * N * N) * (n_z * N + 1)


# ---------------------------------------------------------------------------------------
# source fields

def manufactured_sin(mesh, kx=1.0, ky=1.0, kz=1.0):
    """u* = sin(kx pi x) sin(ky pi y) sin(kz pi z) and f = -laplace(u*) at the nodes."""
    u = np.sin(kx * np.pi * mesh.x) * np.sin(ky * np.pi * mesh.y) * np.sin(kz * np.pi * mesh.z)
    f = (kx * kx + ky * ky + kz * kz) * np.pi ** 2 * u
    return u, f


def divergence_source(mesh, seed, modes=8):
    """f = div v for a seeded random (NOT divergence-free, reading R8) velocity field of unit rms:
    v_c = sum_m a_cm sin(2 pi kappa_cm . x + phi_cm), a ~ N(0,1) (Box-Muller from the counter RNG),
    integer kappa in [1,4]^3, phi ~ U[0, 2 pi).  Returns f at the nodes."""
    u1 = uniform(seed, 3 * modes, 0.0, 1.0); u2 = uniform(seed + 1, 3 * modes, 0.0, 1.0)
    amp = np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2 * np.pi * u2)
    kap = 1 + np.floor(uniform(seed + 2, 9 * modes, 0.0, 4.0)).astype(np.int64).reshape(3, modes, 3)
    phi = uniform(seed + 3, 3 * modes, 0.0, 2 * np.pi).reshape(3, modes)
    amp = amp.reshape(3, modes)
    scale = 1.0 / np.sqrt(0.5 * np.sum(amp ** 2))          # rms of a sum of independent sines
    f = np.zeros(mesh.n)
    ph = np.empty(mesh.n)
    for cdir in range(3):
        for m in range(modes):
            k = kap[cdir, m]
            np.multiply(mesh.x, 2 * np.pi * k[0], out=ph)
            ph += (2 * np.pi * k[1]) * mesh.y
            ph += (2 * np.pi * k[2]) * mesh.z
            ph += phi[cdir, m]
            np.cos(ph, out=ph)
            f += (scale * amp[cdir, m] * 2 * np.pi * k[cdir]) * ph
    return f


# ---------------------------------------------------------------------------------------
# BASELINE.json configs (index -> mesh + parameters); `scale` < 1 gives the reduced members of
# the same mesh family used where the oracle must finish in seconds.

def config_mesh(cfg, xi_of_N, small=False):
    """xi_of_N: callable N -> GLL nodes.  Returns (Mesh, params dict)."""
    if cfg == 0:
        N = 7
        m = box_mesh(4, 4, 4, N, xi_of_N(N), periodic=(True, True, False), name="cfg0_cube4_affine")
        return m, dict(lam=0.0, tags=0b10, precond=1)
    if cfg in (1, 3):
        N = 7
        ne = {1: 16, 3: 64}[cfg]
        if small:
            ne = {1: 6, 3: 8}[cfg]
        m = box_mesh(ne, ne, ne, N, xi_of_N(N), deform=0.05, name=f"cfg{cfg}_box{ne}_deformed")
        return m, dict(lam=1e4, tags=0b10, precond=1)
    if cfg == 2:
        N = 7
        nc, nr, nz = (24, 18, 32) if not small else (4, 3, 4)
        m = ogrid_mesh(nc, nr, nz, N, xi_of_N(N), name=f"cfg2_ogrid_{nc}_{nr}_{nz}")
        return m, dict(lam=0.0, tags=0b10, precond=2, cheb_k=2)
    if cfg == 4:
        N = 9
        nc, nr, nz = (20, 15, 40) if not small else (4, 3, 4)
        m = ogrid_mesh(nc, nr, nz, N, xi_of_N(N), name=f"cfg4_ogrid_{nc}_{nr}_{nz}_N9")
        return m, dict(lam=1.5 / 5e-4, tags=0b10, precond=1, dt=5e-4, steps=10)
    raise ValueError(cfg)


def seed_for(cfg, array_id):
    return BASE_SEED + 1000 * cfg + array_id
