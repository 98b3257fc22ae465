"""Pins for the renderer oracle (oracle/render_oracle.cpp). The paper
prints no image or pixel value (its figures are absent), so these are closed forms and
invariants of direct volume rendering by front-to-back compositing."""
import math

import numpy as np
import pytest

import oracle

IDENT = np.eye(3, dtype=np.float32)


def flat_lut(rgb=(0.2, 0.5, 0.9), alpha=0.01):
    lut = np.zeros((256, 4), dtype=np.float32)
    lut[:, :3] = rgb
    lut[:, 3] = alpha
    return lut


def test_trilinear_sampling_reproduces_a_linear_field_and_the_voxel_values():
    nz, ny, nx = 5, 6, 7
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    vol = (0.25 * x - 0.5 * y + 2.0 * z + 1.0).astype(np.float32)
    rng = np.random.default_rng(0)
    for _ in range(50):
        p = rng.uniform(0, 1, 3) * np.array([nx - 1, ny - 1, nz - 1])
        assert oracle.render_sample(vol, p) == pytest.approx(0.25 * p[0] - 0.5 * p[1] + 2.0 * p[2] + 1.0, abs=2e-6)
    assert oracle.render_sample(vol, (3, 2, 4)) == vol[4, 2, 3]
    assert oracle.render_sample(vol, (6, 5, 4)) == vol[4, 5, 6]          # the upper corner
    rnd = rng.random((nz, ny, nx)).astype(np.float32)                      # x is the fastest axis
    assert oracle.render_sample(rnd, (2.5, 1, 3)) == pytest.approx(0.5 * (rnd[3, 1, 2] + rnd[3, 1, 3]), abs=1e-7)
    assert oracle.render_sample(rnd, (2, 1.5, 3)) == pytest.approx(0.5 * (rnd[3, 1, 2] + rnd[3, 2, 2]), abs=1e-7)
    assert oracle.render_sample(rnd, (2, 1, 3.5)) == pytest.approx(0.5 * (rnd[3, 1, 2] + rnd[4, 1, 2]), abs=1e-7)


def test_uniform_volume_composites_to_the_closed_form():
    """Constant colour c and sample opacity a along n samples: A = 1 - (1-a)^n, C = c A."""
    n = 16
    vol = np.ones((n, n, n), dtype=np.float32)
    alpha, rgb = 0.01, (0.2, 0.5, 0.9)
    img, inside = oracle.render(vol, 8, 8, IDENT, 1.0, 1.0, 1.0, 0.0, 1.0, flat_lut(rgb, alpha))
    # axis-aligned view, step 1: the samples at view z = -T + k fall inside [0, n-1] for exactly
    # n of the k (T = n sqrt(3)/2 is irrational, so none sits on the faces)... or n - 1: count them
    T = np.float32(0.5) * np.sqrt(np.float32(3 * n * n))
    zs = np.float32(0.5 * (n - 1)) + (-T + np.arange(int(math.floor(2 * T)) + 1, dtype=np.float32))
    per_ray = int(np.count_nonzero((zs >= 0) & (zs <= n - 1)))
    assert per_ray in (n - 1, n)
    assert inside == per_ray * 64
    A = 1.0 - (1.0 - alpha) ** per_ray
    assert np.allclose(img[..., 3], A, atol=2e-6)
    for c in range(3):
        assert np.allclose(img[..., c], rgb[c] * A, atol=2e-6)


def test_zero_opacity_and_rays_that_miss_give_black():
    vol = np.ones((8, 8, 8), dtype=np.float32)
    img, _ = oracle.render(vol, 6, 6, IDENT, 1.0, 0.5, 1.0, 0.0, 1.0, flat_lut(alpha=0.0))
    assert np.all(img == 0.0)
    img, inside = oracle.render(vol, 32, 32, IDENT, 1.0, 0.5, 1.0, 0.0, 1.0, flat_lut(alpha=0.05))
    assert np.all(img[0, 0] == 0.0) and np.all(img[31, 31] == 0.0)       # 16 voxels off the centre
    assert img[16, 16, 3] > 0.3 and inside > 0


def test_early_termination_saturates_at_the_threshold():
    vol = np.ones((32, 4, 4), dtype=np.float32)
    img, _ = oracle.render(vol, 2, 2, IDENT, 1.0, 0.25, 1.0, 0.0, 1.0, flat_lut(alpha=0.5))
    assert np.all(img[..., 3] >= 0.995) and np.all(img[..., 3] <= 1.0)


def test_transfer_function_scale_and_offset_select_the_lut_entry():
    vol = np.full((6, 6, 6), 0.5, dtype=np.float32)
    lut = np.zeros((256, 4), dtype=np.float32)
    lut[:, 3] = 0.02
    lut[:, 0] = np.arange(256) / 255.0                                     # red ramp
    for scale, offset in ((1.0, 0.0), (2.0, -0.5), (0.0, 0.25), (4.0, 0.0), (1.0, -1.0)):
        img, _ = oracle.render(vol, 2, 2, IDENT, 1.0, 1.0, scale, offset, 1.0, lut)
        t = min(1.0, max(0.0, 0.5 * scale + offset))
        red = int(t * 255 + 0.5) / 255.0
        assert np.allclose(img[..., 0], red * img[..., 3], atol=1e-6)
        assert np.all(img[..., 1:3] == 0.0)


def test_rotating_volume_and_camera_together_changes_nothing():
    """A quarter turn about z applied to the data and, through `rot`, to the camera."""
    rng = np.random.default_rng(3)
    vol = rng.random((9, 9, 9)).astype(np.float32)
    lut = flat_lut(alpha=0.03)
    lut[:, 0] = np.linspace(0, 1, 256)
    a, _ = oracle.render(vol, 12, 12, IDENT, 1.0, 0.5, 1.0, 0.0, 1.0, lut)
    vol_r = np.ascontiguousarray(np.rot90(vol, k=1, axes=(1, 2)))         # rotate in the x-y plane
    # np.rot90 on axes (y, x): new[y', x'] = old[x', n-1-y']  <=>  x = y', y = n-1-x' ... view map:
    rot = np.array([[0, 1, 0], [-1, 0, 0], [0, 0, 1]], dtype=np.float32)
    b, _ = oracle.render(vol_r, 12, 12, rot, 1.0, 0.5, 1.0, 0.0, 1.0, lut)
    rot2 = np.array([[0, -1, 0], [1, 0, 0], [0, 0, 1]], dtype=np.float32)
    c, _ = oracle.render(vol_r, 12, 12, rot2, 1.0, 0.5, 1.0, 0.0, 1.0, lut)
    assert min(np.max(np.abs(a - b)), np.max(np.abs(a - c))) < 1e-6
    assert np.max(np.abs(a - np.transpose(a, (1, 0, 2)))) > 1e-3           # the test can tell views apart


def test_zoom_scales_the_footprint():
    vol = np.ones((8, 8, 8), dtype=np.float32)
    lut = flat_lut(alpha=0.05)
    a, _ = oracle.render(vol, 32, 32, IDENT, 1.0, 0.5, 1.0, 0.0, 1.0, lut)
    b, _ = oracle.render(vol, 32, 32, IDENT, 2.0, 0.5, 1.0, 0.0, 1.0, lut)
    na, nb = np.count_nonzero(a[..., 3] > 0), np.count_nonzero(b[..., 3] > 0)
    assert nb == pytest.approx(4 * na, rel=0.35) and nb > na


def test_argument_errors():
    vol = np.ones((2, 2, 2), dtype=np.float32)
    with pytest.raises(ValueError):
        oracle.render(vol, 4, 4, IDENT, 0.0, 1.0, 1.0, 0.0, 1.0, flat_lut())
    with pytest.raises(ValueError):
        oracle.render(vol, 4, 4, IDENT, 1.0, 0.0, 1.0, 0.0, 1.0, flat_lut())
