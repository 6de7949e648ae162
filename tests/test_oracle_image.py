"""Pins of the image-consumer oracle (oracle/semimage.c; reading R24): closed forms and
geometry that numpy can state without the oracle -- colour ramps, which sub-cell of a box contains a pixel, the value of
a linear field at the pixel, the disc footprint of the cylinder, an iso-PLANE (exact) and an iso-SPHERE (second-order
accurate) under an orthographic view."""
import numpy as np
import pytest

from paper_2501_13240_b200 import inputs as I

GRAY = [(0, 0, 0), (255, 255, 255)]
COOLWARM = [(59, 76, 192), (141, 176, 254), (221, 221, 221), (244, 154, 123), (180, 4, 38)]


def unpack(rgba):
    return np.stack([(rgba >> s) & 0xff for s in (0, 8, 16, 24)], axis=-1).astype(np.int64)


def test_colormap_closed_forms(orc):
    cm = orc.make_cmap(0.0, 1.0, GRAY)
    v = np.linspace(-0.25, 1.25, 1001)
    ch = unpack(orc.colormap(cm, v))
    expect = np.floor(np.clip(v, 0, 1) * 255.0 + 0.5).astype(np.int64)
    assert np.array_equal(ch[:, 0], expect) and np.array_equal(ch[:, 1], expect) and np.array_equal(ch[:, 2], expect)
    assert np.all(ch[:, 3] == 255)
    # the control points are hit exactly and the segments are linear in between
    cm = orc.make_cmap(2.0, 6.0, COOLWARM)
    ch = unpack(orc.colormap(cm, np.array([2.0, 3.0, 4.0, 5.0, 6.0, 3.5, 1.0, 9.0])))
    assert np.array_equal(ch[:5, :3], np.array(COOLWARM))
    mid = np.floor(0.5 * (np.array(COOLWARM[1]) + np.array(COOLWARM[2])) + 0.5)
    assert np.array_equal(ch[5, :3], mid.astype(np.int64))
    assert np.array_equal(ch[6, :3], COOLWARM[0]) and np.array_equal(ch[7, :3], COOLWARM[-1])      # clamped


def test_slice_of_a_box_finds_the_right_subcell_and_value(orc, xi_of):
    """Horizontal and vertical slices of a stretched box: the sub-cell that claims a pixel is the one numpy finds by
    searching the node planes, and the colour is the map of the LINEAR field's exact value at the pixel centre."""
    N, (nx, ny, nz) = 4, (3, 2, 4)
    m = I.box_mesh(nx, ny, nz, N, xi_of(N), zstretch=2.0)
    f = 0.3 * m.x - 0.2 * m.y + 0.9 * m.z + 0.1
    cm = orc.make_cmap(0.0, 1.2, COOLWARM, background=0xff102030)
    xs, ys, zs = np.unique(m.x), np.unique(m.y), np.unique(m.z)
    Wd, Ht = 96, 64
    for plane in ("z", "y"):
        if plane == "z":
            z0 = 0.0371
            vw = orc.make_view(Wd, Ht, (0.0, 0.0, z0), (1, 0, 0), (0, 1, 0), 1.0 / Wd, 1.0 / Ht)
            PX, PY = np.meshgrid((np.arange(Wd) + 0.5) / Wd, (np.arange(Ht) + 0.5) / Ht)
            P = np.stack([PX, PY, np.full_like(PX, z0)], -1)
        else:
            y0 = 0.61
            vw = orc.make_view(Wd, Ht, (0.0, y0, 0.0), (1, 0, 0), (0, 0, 1), 1.0 / Wd, 1.0 / Ht)
            PX, PZ = np.meshgrid((np.arange(Wd) + 0.5) / Wd, (np.arange(Ht) + 0.5) / Ht)
            P = np.stack([PX, np.full_like(PX, y0), PZ], -1)
        rgba, cell = orc.image_slice(m.E, N, m.x, m.y, m.z, f, vw, cm)
        assert np.all(cell >= 0)                                                  # the plane lies inside the box everywhere
        # sub-cell by search: global lattice interval -> (element, local interval); pixels on a node plane are skipped
        gi = [np.searchsorted(a, P[..., c], side="right") - 1 for c, a in enumerate((xs, ys, zs))]
        onplane = np.zeros(PX.shape, dtype=bool)
        for c, a in enumerate((xs, ys, zs)):
            onplane |= np.min(np.abs(P[..., c][..., None] - a[None, None, :]), axis=-1) < 1e-12
        ex, ey, ez = gi[0] // N, gi[1] // N, gi[2] // N
        expect = ((ez * ny + ey) * nx + ex) * N ** 3 + ((gi[2] % N) * N + gi[1] % N) * N + gi[0] % N
        assert np.array_equal(cell[~onplane], expect[~onplane])
        val = 0.3 * P[..., 0] - 0.2 * P[..., 1] + 0.9 * P[..., 2] + 0.1
        ref = unpack(orc.colormap(cm, val.ravel())).reshape(Ht, Wd, 4)
        diff = np.abs(unpack(rgba) - ref)
        assert diff.max() <= 1 and (diff > 0).mean() < 0.01                       # interpolation error 1e-16: only at rounding ties


def test_slice_of_the_cylinder_has_a_disc_footprint(orc, xi_of):
    m, _ = I.config_mesh(2, xi_of, small=True)
    f = m.x * m.x + m.y * m.y
    cm = orc.make_cmap(0.0, 0.25, GRAY, background=0xffff00ff)
    Wd = 80
    vw = orc.make_view(Wd, Wd, (-0.55, -0.55, 0.3), (1, 0, 0), (0, 1, 0), 1.1 / Wd, 1.1 / Wd)
    rgba, cell = orc.image_slice(m.E, m.N, m.x, m.y, m.z, f, vw, cm)
    c = -0.55 + (np.arange(Wd) + 0.5) * 1.1 / Wd
    X, Y = np.meshgrid(c, c)
    rad = np.sqrt(X * X + Y * Y)
    assert np.all(cell[rad < 0.5 - 0.004] >= 0) and np.all(cell[rad > 0.5 + 1e-9] < 0)      # isoparametric N = 7 boundary: 1e-9 of the circle
    assert np.all(rgba[cell < 0] == 0xffff00ff)
    inside = rad < 0.49
    gray = unpack(rgba)[..., 0]
    assert np.abs(gray[inside] - np.floor(np.clip(rad[inside] ** 2 / 0.25, 0, 1) * 255 + 0.5)).max() <= 3   # trilinear sub-cell error of x^2 + y^2


def test_isosurface_of_a_linear_field_is_the_exact_plane(orc, xi_of):
    """f = z: the level set is the plane z = z0 in every tetrahedron exactly, so depth, coverage and the shaded colour are
    closed forms: shade = 0.25 + 0.75 |n . l| with n = e_z."""
    N = 3
    m = I.box_mesh(2, 3, 2, N, xi_of(N), deform=0.0)
    z0 = 0.4321
    Wd, Ht = 50, 40
    light = np.array([0.0, 0.6, 0.8])
    cm = orc.make_cmap(0.0, 1.0, [(200, 100, 40), (200, 100, 40)], background=0xff000000)
    # looking down -z: u = x, v = -y ... keep it right-handed: u = y, v = x => w = u x v = -z; origin above the box
    vw = orc.make_view(Wd, Ht, (0.0, 0.0, 2.0), (0, 1, 0), (1, 0, 0), 1.0 / Wd, 1.0 / Ht)
    rgba, key = orc.image_isosurface(m.E, N, m.x, m.y, m.z, m.z, z0, None, vw, cm, light, 0.0, 4.0)
    depth = (key >> np.uint64(32)).astype(np.float64) / 4294967295.0 * 4.0
    assert np.abs(depth - (2.0 - z0)).max() <= 4.0 / 2 ** 32 + 1e-12             # every pixel sees the plane at distance 2 - z0
    shade = 0.25 + 0.75 * 0.8
    expect = np.floor(np.array([200, 100, 40]) * shade + 0.5).astype(np.int64)
    ch = unpack(rgba)
    assert np.array_equal(np.unique(ch[..., :3].reshape(-1, 3), axis=0), expect[None, :])


def test_isosurface_of_a_sphere(orc, xi_of):
    """f = |X - c|^2, iso = R^2, seen along -z: silhouette = disc of radius R, depth = zc-distance minus sqrt(R^2 - rho^2);
    the linear tetrahedra are second-order accurate in the sub-cell size."""
    N = 6
    m = I.box_mesh(3, 3, 3, N, xi_of(N))
    c, R = np.array([0.5, 0.5, 0.5]), 0.3
    f = (m.x - c[0]) ** 2 + (m.y - c[1]) ** 2 + (m.z - c[2]) ** 2
    Wd = 120
    cm = orc.make_cmap(0.0, 1.0, GRAY, background=0xff0000ff)
    vw = orc.make_view(Wd, Wd, (0.0, 0.0, 2.0), (0, 1, 0), (1, 0, 0), 1.0 / Wd, 1.0 / Wd)
    rgba, key = orc.image_isosurface(m.E, N, m.x, m.y, m.z, f, R * R, m.z, vw, cm, [0, 0, 1], 0.0, 4.0)
    pc = (np.arange(Wd) + 0.5) / Wd
    A, B = np.meshgrid(pc, pc)                      # image a = y, b = x
    rho = np.sqrt((A - 0.5) ** 2 + (B - 0.5) ** 2)
    hit = (key >> np.uint64(32)) != np.uint64(0xffffffff)
    hsub = 1.0 / 3 / N
    assert np.all(hit[rho < R - hsub]) and not np.any(hit[rho > R + 1e-9])
    area = hit.sum() / Wd ** 2                                                     # chords lie inside the sphere: slightly smaller disc
    assert 0.97 * np.pi * R * R < area <= np.pi * R * R * 1.001
    depth = (key >> np.uint64(32)).astype(np.float64) / 4294967295.0 * 4.0
    sel = rho < 0.8 * R
    expect = 2.0 - (0.5 + np.sqrt(R * R - rho[sel] ** 2))                         # the NEAR side of the sphere (z = 0.5 + ..)
    assert np.abs(depth[sel] - expect).max() < 1.5 * hsub ** 2 / R
    # colour = z of the surface point through the gray ramp, shaded by |n_z|: brightest at the pole
    g = unpack(rgba)[..., 0]
    pole = g[Wd // 2, Wd // 2]
    assert 0 <= np.floor(255 * 0.8 * 1.0 + 0.5) - pole <= 6 and np.all(g[sel] <= pole + 2)      # flat facets: |n_z| >= 0.97 next to the pole
