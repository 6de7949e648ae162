"""GPU parity of the in-situ image consumer (csrc/image.cu) against oracle/semimage.c: RGBA bytes, claiming sub-cell ids
and depth keys are compared EXACTLY (integer / byte work: bit-exact bar), on boxes, stretched boxes, deformed boxes and the
cylinder O-grid, for horizontal, vertical and oblique planes and an iso-surface coloured by a second field."""
import numpy as np
import pytest

from paper_2501_13240_b200 import inputs as I

pytestmark = pytest.mark.gpu
COOLWARM = [(59, 76, 192), (141, 176, 254), (221, 221, 221), (244, 154, 123), (180, 4, 38)]


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


MESHES = {
    "box_stretched_N4": lambda xi: I.box_mesh(3, 2, 4, 4, xi(4), zstretch=2.0),
    "box_deformed_N7":  lambda xi: I.box_mesh(3, 3, 2, 7, xi(7), deform=0.05),
    "ogrid_N7":         lambda xi: I.config_mesh(2, xi, small=True)[0],
    "jitter_N5":        lambda xi: I.trilinear_box_mesh(3, 3, 3, 5, xi(5), jitter=0.2),
    "N1":               lambda xi: I.box_mesh(5, 4, 3, 1, xi(1), deform=0.05),
}


def unit(v):
    v = np.asarray(v, dtype=np.float64)
    return v / np.linalg.norm(v)


def views(name, W, H):
    """(label, origin, u, v, du, dv) per mesh: horizontal, vertical and oblique planes through the domain"""
    if name.startswith("ogrid"):
        return [("z", (-0.55, -0.55, 0.3), (1, 0, 0), (0, 1, 0), 1.1 / W, 1.1 / H),
                ("y", (-0.55, 0.013, 0.0), (1, 0, 0), (0, 0, 1), 1.1 / W, 1.0 / H),
                ("oblique", (-0.6, -0.2, 0.1), unit((1, 0.3, 0.1)), unit(np.cross(np.cross((1, 0.3, 0.1), (0, 0.2, 1)), (1, 0.3, 0.1))), 1.3 / W, 1.0 / H)]
    return [("z", (0.0, 0.0, 0.0371), (1, 0, 0), (0, 1, 0), 1.0 / W, 1.0 / H),
            ("x", (0.43, 0.0, 0.0), (0, 1, 0), (0, 0, 1), 1.0 / W, 1.0 / H),
            ("wall", (0.0, 0.0, 0.0), (1, 0, 0), (0, 1, 0), 1.0 / W, 1.0 / H),          # the plate itself: d = 0 on a whole face
            ("oblique", (-0.1, 0.1, 0.2), unit((1, 0.2, 0.3)), unit(np.cross(np.cross((1, 0.2, 0.3), (0, 1, 0.1)), (1, 0.2, 0.3))), 1.4 / W, 1.1 / H)]


@pytest.mark.parametrize("name", list(MESHES))
def test_slices_are_bit_exact(torch_cuda, semb, orc, xi_of, name):
    torch = torch_cuda
    m = MESHES[name](xi_of)
    T = (1.0 - m.z) + 0.05 * I.uniform(31, m.n) + 0.2 * np.sin(3 * m.x) * np.cos(2 * m.y)
    G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    try:
        Td = dev(torch, T)
        G.publish_field("temperature", Td)
        G.publish_state(1, 0.0)
        d = G.export_field("temperature")
        W, H = 97, 61
        key = torch.zeros(W * H, dtype=torch.int64, device="cuda"); rgba = torch.zeros(W * H, dtype=torch.int32, device="cuda")
        hits = 0
        for label, o, u, v, du, dv in views(name, W, H):
            cm_o = orc.make_cmap(0.0, 1.0, COOLWARM, background=0xff102030)
            cm_g = semb.colormap(0.0, 1.0, COOLWARM, background=0xff102030)
            ref_rgba, ref_cell = orc.image_slice(m.E, m.N, m.x, m.y, m.z, T, orc.make_view(W, H, o, u, v, du, dv), cm_o)
            G.image_slice(d, semb.image_view(W, H, o, u, v, du, dv), cm_g, key, rgba)
            k = key.cpu().numpy().view(np.uint64).reshape(H, W)
            cell = (k >> np.uint64(32)).astype(np.int64)
            cell[cell == 0xffffffff] = -1
            assert np.array_equal(cell, ref_cell), (name, label, int((cell != ref_cell).sum()))
            assert np.array_equal(rgba.cpu().numpy().view(np.uint32).reshape(H, W), ref_rgba), (name, label)
            assert np.array_equal((k & np.uint64(0xffffffff)).astype(np.uint32), ref_rgba)
            hits += int((ref_cell >= 0).sum())
        assert hits > W * H                                          # the views really cut the mesh
    finally:
        G.close()


@pytest.mark.parametrize("name", ["box_stretched_N4", "box_deformed_N7", "ogrid_N7", "N1"])
def test_isosurface_is_bit_exact(torch_cuda, semb, orc, xi_of, name):
    torch = torch_cuda
    m = MESHES[name](xi_of)
    c0 = (0.0, 0.0, 0.5) if name.startswith("ogrid") else (0.5, 0.5, 0.5)
    f = (m.x - c0[0]) ** 2 + 1.3 * (m.y - c0[1]) ** 2 + 0.8 * (m.z - c0[2]) ** 2 + 0.02 * np.sin(9 * m.x + 5 * m.z)
    T = 1.0 - m.z
    G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    try:
        G.publish_field("f", dev(torch, f)); G.publish_field("temperature", dev(torch, T))
        df, dT = G.export_field("f"), G.export_field("temperature")
        W, H = 83, 59
        key = torch.zeros(W * H, dtype=torch.int64, device="cuda"); rgba = torch.zeros(W * H, dtype=torch.int32, device="cuda")
        light = unit((0.3, -0.5, 0.8))
        for (o, u, v, du, dv, dlo, dhi), colour in [(((-0.2 + c0[0] - 0.5, -0.2 + c0[1] - 0.5, 2.0), (0, 1, 0), (1, 0, 0), 1.4 / W, 1.4 / H, 0.0, 4.0), True),
                                                    (((c0[0] - 0.9, c0[1] - 0.6, -0.5), unit((1, 0.2, 0.1)), unit(np.cross(np.cross((1, 0.2, 0.1), (0.1, 1, 0.3)), (1, 0.2, 0.1))), 1.8 / W, 1.6 / H, -2.0, 3.0), False)]:
            for iso in (0.06, 0.11):
                ref_rgba, ref_key = orc.image_isosurface(m.E, m.N, m.x, m.y, m.z, f, iso, T if colour else None, orc.make_view(W, H, o, u, v, du, dv),
                                                         orc.make_cmap(0.0, 1.0, COOLWARM, background=0xff000000), light, dlo, dhi)
                G.image_isosurface(df, iso, dT if colour else None, semb.image_view(W, H, o, u, v, du, dv, dlo, dhi),
                                   semb.colormap(0.0, 1.0, COOLWARM, background=0xff000000), light, key, rgba)
                k = key.cpu().numpy().view(np.uint64).reshape(H, W)
                assert np.array_equal(k, ref_key), (name, iso, int((k != ref_key).sum()))
                assert np.array_equal(rgba.cpu().numpy().view(np.uint32).reshape(H, W), ref_rgba)
                assert ((ref_key >> np.uint64(32)) != np.uint64(0xffffffff)).sum() > 50       # the surface is in view
    finally:
        G.close()


def test_colormap_and_argument_checks(torch_cuda, semb, orc, xi_of):
    torch = torch_cuda
    v = I.uniform(3, 100001) * 1.5
    out = torch.zeros(v.size, dtype=torch.int32, device="cuda")
    semb.colormap_apply(semb.colormap(-1.0, 1.2, COOLWARM), dev(torch, v), out)
    assert np.array_equal(out.cpu().numpy().view(np.uint32), orc.colormap(orc.make_cmap(-1.0, 1.2, COOLWARM), v))
    m = I.box_mesh(2, 2, 2, 3, xi_of(3))
    G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
    try:
        t = dev(torch, m.z.copy())
        G.publish_field("t", t)
        d = G.export_field("t")
        key = torch.zeros(64, dtype=torch.int64, device="cuda")
        free0 = torch.cuda.mem_get_info()[0]
        G.image_slice(d, semb.image_view(8, 8, (0, 0, 0.5), (1, 0, 0), (0, 1, 0), 0.125, 0.125), semb.colormap(0, 1, COOLWARM), key)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0                 # the consumer allocates nothing
        with pytest.raises(semb.SembError):                          # a field that is not over the mesh's nodes
            bad = semb.FieldDesc(b"x", t.data_ptr(), 1, 1, m.n - 1, 1, 0, 0.0)
            G.image_slice(bad, semb.image_view(8, 8, (0, 0, 0.5), (1, 0, 0), (0, 1, 0), 0.125, 0.125), semb.colormap(0, 1, COOLWARM), key)
        with pytest.raises(semb.SembError):                          # host memory is refused
            bad = semb.FieldDesc(b"x", t.data_ptr(), 1, 0, m.n, 1, 0, 0.0)
            G.image_slice(bad, semb.image_view(8, 8, (0, 0, 0.5), (1, 0, 0), (0, 1, 0), 0.125, 0.125), semb.colormap(0, 1, COOLWARM), key)
    finally:
        G.close()


def test_degenerate_views(torch_cuda, semb, orc, xi_of):
    """Edge cases: a plane that misses the mesh (all background), a 1 x 1 image, an iso value outside the field's range, and a
    one-element mesh of order 1 (a single sub-cell)."""
    torch = torch_cuda
    for m in (I.box_mesh(2, 2, 2, 3, xi_of(3), deform=0.03), I.box_mesh(1, 1, 1, 1, xi_of(1))):
        T = 1.0 - m.z + 0.1 * m.x
        G = semb.Mesh(m.E, m.N, dev(torch, m.x), dev(torch, m.y), dev(torch, m.z), m.face_tag, m.period)
        try:
            Td = dev(torch, T)
            G.publish_field("t", Td)
            d = G.export_field("t")
            cm_o, cm_g = orc.make_cmap(0.0, 1.0, COOLWARM, background=0xff112233), semb.colormap(0.0, 1.0, COOLWARM, background=0xff112233)
            for W, H, o in ((16, 9, (0.0, 0.0, 1.5)), (1, 1, (0.2, 0.3, 0.5)), (7, 5, (0.0, 0.0, 1.0))):
                key = torch.zeros(W * H, dtype=torch.int64, device="cuda"); rgba = torch.zeros(W * H, dtype=torch.int32, device="cuda")
                G.image_slice(d, semb.image_view(W, H, o, (1, 0, 0), (0, 1, 0), 1.0 / W, 1.0 / H), cm_g, key, rgba)
                ref_rgba, ref_cell = orc.image_slice(m.E, m.N, m.x, m.y, m.z, T, orc.make_view(W, H, o, (1, 0, 0), (0, 1, 0), 1.0 / W, 1.0 / H), cm_o)
                assert np.array_equal(rgba.cpu().numpy().view(np.uint32).reshape(H, W), ref_rgba)
                if o[2] > 1.0:
                    assert np.all(ref_cell < 0) and np.all(ref_rgba == 0xff112233)
                for iso in (5.0, 0.55):
                    G.image_isosurface(d, iso, None, semb.image_view(W, H, (0.0, 0.0, 2.0), (0, 1, 0), (1, 0, 0), 1.0 / W, 1.0 / H, 0.0, 4.0), cm_g,
                                       (0, 0, 1), key, rgba)
                    rr, rk = orc.image_isosurface(m.E, m.N, m.x, m.y, m.z, T, iso, None, orc.make_view(W, H, (0.0, 0.0, 2.0), (0, 1, 0), (1, 0, 0), 1.0 / W, 1.0 / H),
                                                  cm_o, (0, 0, 1), 0.0, 4.0)
                    assert np.array_equal(key.cpu().numpy().view(np.uint64).reshape(H, W), rk)
                    if iso > 2.0:
                        assert np.all(rr == 0xff112233)
        finally:
            G.close()
