"""GPU parity of the ray-marching renderer (the paper's own GPU
kernel) against oracle/render_oracle.cpp. Both sides evaluate the same
binary32 operations in the same order with explicit fused multiply-adds only, so the images
are compared bit for bit where the input volume is shared."""
import math

import numpy as np
import pytest

import oracle
import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hlb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1906_11925_b200 as m
    return m


def rotation(axis, deg):
    a = np.asarray(axis, dtype=np.float64)
    a /= np.linalg.norm(a)
    t = math.radians(deg)
    K = np.array([[0, -a[2], a[1]], [a[2], 0, -a[0]], [-a[1], a[0], 0]])
    return (np.eye(3) + math.sin(t) * K + (1 - math.cos(t)) * K @ K).astype(np.float32)


def rainbow_lut(alpha=0.04):
    t = np.linspace(0, 1, 256)
    lut = np.stack([t, np.sin(math.pi * t), 1 - t, alpha * (0.2 + t)], axis=1)
    return lut.astype(np.float32)


VIEWS = [
    dict(rot=np.eye(3), zoom=1.0, step=1.0, tf_scale=1.0, tf_offset=0.0, opacity=1.0),
    dict(rot=rotation((0, 0, 1), 30), zoom=1.7, step=0.5, tf_scale=2.0, tf_offset=-0.3, opacity=0.7),
    dict(rot=rotation((1, 2, 3), 77), zoom=0.8, step=0.37, tf_scale=0.9, tf_offset=0.05, opacity=3.0),
    dict(rot=rotation((1, -1, 0.2), 200), zoom=3.1, step=0.8, tf_scale=1.0, tf_offset=0.0, opacity=25.0),
]


@pytest.mark.parametrize("shape", [(17, 23, 31), (1, 9, 14), (40, 40, 40), (5, 1, 1)])
@pytest.mark.parametrize("view", range(len(VIEWS)))
def test_render_volume_equals_oracle_bitwise(hlb, shape, view):
    rng = np.random.default_rng(10 * view + shape[0])
    vol = rng.random(shape).astype(np.float32) ** 3
    kw = VIEWS[view]
    lut = rainbow_lut()
    for width, height in ((33, 21), (64, 64)):
        ref, inside = oracle.render(vol, width, height, lut=lut, **kw)
        v = hlb.make_view(width, height, **kw)
        img = hlb.hlb_render_volume(vol, v, lut)
        assert img.shape == ref.shape == (height, width, 4)
        assert np.array_equal(img, ref), float(np.max(np.abs(img - ref)))
    if min(shape) > 4 and view < 3:
        assert inside > 0 and np.max(ref[..., 3]) > 0.05           # the comparison is not of black images


def clear_lut(first_opaque=1, alpha=0.06):
    """A look-up table whose entries below `first_opaque` are fully transparent: value 0 then
    contributes nothing and the renderer may skip empty macro-cells."""
    lut = rainbow_lut(alpha)
    lut[:first_opaque, 3] = 0.0
    return lut


SKIP_VIEWS = VIEWS + [
    dict(rot=rotation((1, 0, 0), 90), zoom=1.3, step=0.25, tf_scale=1.0, tf_offset=0.0, opacity=2.0),
    dict(rot=rotation((0, 1, 0), 90.0001), zoom=2.0, step=0.11, tf_scale=1.5, tf_offset=0.0, opacity=1.0),
    dict(rot=rotation((3, 1, -2), 131), zoom=0.9, step=1.9, tf_scale=1.0, tf_offset=0.001, opacity=1.0),
]


def sparse_volume(shape, seed):
    """Mostly exact zeros with a few blobs, a thin diagonal tube and isolated voxels on cell faces."""
    rng = np.random.default_rng(seed)
    vol = np.zeros(shape, dtype=np.float32)
    nz, ny, nx = shape
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    for _ in range(3):
        c = rng.random(3) * np.array(shape)
        r = 2.0 + 5.0 * rng.random()
        m = (z - c[0]) ** 2 + (y - c[1]) ** 2 + (x - c[2]) ** 2 < r * r
        vol[m] = rng.random(int(m.sum())).astype(np.float32)
    t = np.linspace(0, 1, 4 * max(shape))
    vol[(t * (nz - 1)).astype(int), (t * (ny - 1)).astype(int), (t * (nx - 1)).astype(int)] = 0.8
    for k in range(0, min(shape), 8):                # single voxels exactly on macro-cell corners
        vol[k, k, k] = 1.0
        if k + 7 < min(shape):
            vol[k + 7, k, k + 7] = 0.6
    return vol


@pytest.mark.parametrize("shape", [(41, 57, 70), (64, 64, 64), (9, 130, 17), (3, 8, 100), (70, 140, 200)])
@pytest.mark.parametrize("view", range(len(SKIP_VIEWS)))
def test_empty_space_skipping_keeps_the_image_bitwise(hlb, shape, view):
    """With a transfer function that is transparent at value 0 the kernel jumps over empty 8^3
    macro-cells; the image must not change by a single bit (oracle: no skipping at all)."""
    vol = sparse_volume(shape, 7 * view + shape[2])
    kw = SKIP_VIEWS[view]
    for lut in (clear_lut(1), clear_lut(40)):
        ref, inside = oracle.render(vol, 80, 56, lut=lut, **kw)
        img = hlb.hlb_render_volume(vol, hlb.make_view(80, 56, **kw), lut)
        assert np.array_equal(img, ref), float(np.max(np.abs(img - ref)))
    assert inside > 0
    if view in (0, 1, 4):
        assert np.max(ref[..., 3]) > 0.01


def test_empty_volume_renders_black(hlb):
    vol = np.zeros((33, 20, 47), dtype=np.float32)
    img = hlb.hlb_render_volume(vol, hlb.make_view(40, 40, rot=rotation((1, 1, 0), 50)), clear_lut())
    assert not img.any()
    vol[:] = -0.0                                    # not +0: cells are not "empty", result the same
    img = hlb.hlb_render_volume(vol, hlb.make_view(40, 40, rot=rotation((1, 1, 0), 50)), clear_lut())
    assert not img.any()


@pytest.mark.parametrize("scheme", ["two_lattice", "aa"])
def test_render_of_a_running_simulation(hlb, scheme):
    """hlb_render: the speed field of the current state scattered into the voxel box and
    ray-marched; compared (a) bit for bit with the oracle renderer fed the GPU's own field,
    (b) with the whole chain oracle LB -> oracle renderer."""
    wl = W.with_velocity_inlet(W.by_name("aneurysm", small=True), u_in=0.02)
    flags = hlb.HLB_AA if scheme == "aa" else hlb.HLB_TWO_LATTICE
    g = hlb.hlb_geometry_create(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, flags)
    g.hlb_set_iolet_velocity(wl.iolet_kind, wl.iolet_u)
    o = oracle.Oracle(wl.site_type, wl.periodic, wl.tau, wl.iolet_rho, threads=0)
    o.set_iolet_velocity(wl.iolet_kind, wl.iolet_u)
    lut = clear_lut(1, 0.08) if scheme == "aa" else rainbow_lut(0.08)   # with / without skipping
    vox = wl.fluid_voxels()
    for n, field in ((80, 0), (35, 1)):
        g.hlb_step(n)
        o.step(n)
        rho, u = g.hlb_get_macroscopic()
        rho_o, u_o = o.get_macroscopic()
        scale = 1.0 / (np.max(np.linalg.norm(u_o, axis=1)) if field == 0 else np.max(np.abs(rho_o - 1.0)))
        kw = dict(rot=rotation((0.3, 1, 0.2), 40), zoom=1.5, step=0.5, tf_scale=float(scale),
                  tf_offset=0.0 if field == 0 else 0.5, opacity=1.0)
        view = hlb.make_view(96, 64, field=field, **kw)
        img = g.hlb_render(view, lut)
        for (r_, u_), tol in (((rho, u), 0.0), ((rho_o, u_o), 2e-5)):
            s = np.sqrt(u_[:, 0] ** 2 + u_[:, 1] ** 2 + u_[:, 2] ** 2) if field == 0 else r_ - 1.0
            vol = np.zeros(wl.site_type.size, dtype=np.float32)
            vol[vox] = s.astype(np.float32)
            ref, _ = oracle.render(vol.reshape(wl.site_type.shape), 96, 64, lut=lut, **kw)
            assert np.max(np.abs(img - ref)) <= max(tol, 1e-6), (n, field, tol)
        assert np.max(img[..., 3]) > 0.2
        dev = g.hlb_render_device(view, lut)
        assert np.array_equal(dev.cpu().numpy(), img)
    g.close()


def test_render_argument_errors(hlb):
    vol = np.ones((4, 4, 4), dtype=np.float32)
    lut = rainbow_lut()
    for bad in (dict(zoom=0.0), dict(step=-1.0)):
        with pytest.raises(hlb.HlbError) as e:
            hlb.hlb_render_volume(vol, hlb.make_view(8, 8, **bad), lut)
        assert e.value.code == hlb.HLB_EINVAL
    with pytest.raises(hlb.HlbError):
        hlb.hlb_render_volume(vol, hlb.make_view(0, 8), lut)
    st = np.ones((3, 3, 3), dtype=np.uint8)
    g = hlb.hlb_geometry_create(st, 7, 0.8, [])
    with pytest.raises(hlb.HlbError):
        g.hlb_render(hlb.make_view(8, 8, field=5), lut)
    assert np.all(g.hlb_render(hlb.make_view(8, 8), lut)[..., :3] >= 0.0)
    g.close()
