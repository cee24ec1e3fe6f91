"""Pins of the oracle's ray-marcher (NEXT-2; section 4; readings R1-R6).

Nothing here calls the CUDA path.  Each reading is tied to a closed form, a hand-worked case or a
library routine (scipy.ndimage.map_coordinates for the trilinear fetch).
"""
import numpy as np
import pytest

import oracle
from paper_2009_02702_b200 import synth


def _view(**kw):
    v = dict(width=1, height=1, eye=np.zeros(3), right=np.array([0.0, 1.0, 0.0]), up=np.array([0.0, 0.0, 1.0]),
             forward=np.array([1.0, 0.0, 0.0]), tan_half_fov=0.5, spacing=np.ones(3), step_voxels=0.5,
             ref_step_voxels=1.0, lod_bias=0.0, ess_threshold=-1.0, alpha_cutoff=1.0)
    v.update(kw)
    return v


def _constant_pyramid(dims_xyz, node_of_level=lambda l: 0):
    return [np.full((z, y, x), node_of_level(l), dtype=np.uint32) for l, (x, y, z) in enumerate(oracle.mip_dims(dims_xyz))]


# ------------------------------------------------------------------------------------------ R1
def test_pixel_ray_hand_worked_and_symmetric():
    """W=4, H=2, tan_half_fov=0.5: pixel (0,0) has u = (2*0.5/4 - 1)*0.5*2 = -0.75, v = (1 - 0.5)*0.5 = 0.25."""
    v = _view(width=4, height=2)
    d = oracle.pixel_ray(v, 0, 0)
    np.testing.assert_allclose(np.linalg.norm(d), 1.0, atol=1e-15)
    f, r, u = d @ v["forward"], d @ v["right"], d @ v["up"]
    np.testing.assert_allclose([r / f, u / f], [-0.75, 0.25], atol=1e-15)
    d2 = oracle.pixel_ray(v, 3, 1)                      # the opposite pixel mirrors about the view axis
    np.testing.assert_allclose([d2 @ v["right"], d2 @ v["up"], d2 @ v["forward"]], [-r, -u, f], atol=1e-15)
    np.testing.assert_allclose(oracle.pixel_ray(_view(), 0, 0), [1, 0, 0], atol=1e-15)   # 1x1 image looks along forward


# ------------------------------------------------------------------------------------------ R3
def _identity_palette(n):
    i = np.arange(n, dtype=np.float64)
    return np.stack([i, 10 * i + 1, np.cos(i), (i + 1) / (n + 1)], axis=1)


def test_sample_lod_hand_worked_2x2x2():
    l0 = np.arange(8, dtype=np.uint32).reshape(2, 2, 2)           # [z][y][x]: node = 4z + 2y + x
    l1 = np.full((1, 1, 1), 8, dtype=np.uint32)
    pal = _identity_palette(9)
    s = lambda p, lam: oracle.sample_lod([l0, l1], pal, p, lam)
    np.testing.assert_allclose(s((0.5, 0.5, 0.5), 0), pal[0], atol=1e-15)            # a voxel centre
    np.testing.assert_allclose(s((1.5, 0.5, 0.5), 0), pal[1], atol=1e-15)            # x is the fastest axis
    np.testing.assert_allclose(s((0.5, 1.5, 0.5), 0), pal[2], atol=1e-15)
    np.testing.assert_allclose(s((0.5, 0.5, 1.5), 0), pal[4], atol=1e-15)
    np.testing.assert_allclose(s((1.0, 1.0, 1.0), 0), pal[:8].mean(axis=0), atol=1e-14)   # the cell centre
    np.testing.assert_allclose(s((0.75, 0.5, 0.5), 0), 0.75 * pal[0] + 0.25 * pal[1], atol=1e-15)
    np.testing.assert_allclose(s((0.1, 0.2, 0.0), 0), pal[0], atol=1e-15)            # clamp to edge
    np.testing.assert_allclose(s((1.9, 2.0, 1.6), 0), pal[7], atol=1e-15)
    np.testing.assert_allclose(s((0.3, 1.2, 0.9), 1), pal[8], atol=1e-15)            # coarsest level: one voxel
    np.testing.assert_allclose(s((0.5, 0.5, 0.5), 0.25), 0.75 * pal[0] + 0.25 * pal[8], atol=1e-15)
    np.testing.assert_allclose(s((0.5, 0.5, 0.5), 7.0), pal[8], atol=1e-15)          # lambda clamps to l_max


def test_trilinear_is_scipy_map_coordinates_on_every_level():
    """Voxel i of level l is centred at (i + 1/2) 2^l; clamp-to-edge == mode='nearest'."""
    ndi = pytest.importorskip("scipy.ndimage")
    dims = (13, 7, 5)
    levels, n = [], 0
    for (x, y, z) in oracle.mip_dims(dims):
        levels.append((np.arange(x * y * z, dtype=np.uint32) + n).reshape(z, y, x))
        n += x * y * z
    pal = synth.random_attr(n, 4, seed=5).astype(np.float64)
    pts = synth.random_attr(40, 3, seed=6).astype(np.float64) * np.array(dims)
    for l in range(len(levels)):
        vol = pal[levels[l]]                                       # [z, y, x, 4]
        for p in pts:
            u = p / 2.0 ** l - 0.5
            ref = [ndi.map_coordinates(vol[..., ch], [[u[2]], [u[1]], [u[0]]], order=1, mode="nearest")[0] for ch in range(4)]
            np.testing.assert_allclose(oracle.sample_lod(levels, pal, p, float(l)), ref, atol=1e-13)


# ------------------------------------------------------------------------------------------ R4/R5
@pytest.mark.parametrize("spacing,axis,length", [((1, 1, 1), 0, 8.0), ((1, 1, 7), 2, 56.0), ((2, 3, 4), 1, 24.0)])
@pytest.mark.parametrize("bias", [0.0, 3.0])
def test_homogeneous_volume_closed_form(spacing, axis, length, bias):
    """One segment, colour c, opacity a: the clipped intervals telescope, so whatever the steps are
    A = 1 - (1 - a)^(path / (ref s_ref)) and C = c A (Beer-Lambert)."""
    levels = _constant_pyramid((8, 8, 8))
    pal = np.array([[0.2, 0.5, 0.9, 0.3]])
    e = np.eye(3)
    fwd = e[axis]
    ext = 8.0 * np.array(spacing, dtype=np.float64)
    eye = 0.5 * ext - fwd * (0.5 * ext[axis] + 11.0)
    v = _view(eye=eye, forward=fwd, right=e[(axis + 1) % 3], up=e[(axis + 2) % 3], spacing=np.array(spacing, float),
              lod_bias=bias, ref_step_voxels=2.0, step_voxels=0.37)
    img, (n_eval, n_skip) = oracle.render(levels, pal, v)
    A = 1.0 - (1.0 - 0.3) ** (length / (2.0 * min(spacing)))
    np.testing.assert_allclose(img[0, 0], [0.2 * A, 0.5 * A, 0.9 * A, A], rtol=0, atol=1e-12)
    assert n_eval > 0 and n_skip == 0


def test_cube_diagonal_path_length_and_miss():
    levels = _constant_pyramid((8, 8, 8))
    pal = np.array([[1.0, 1.0, 1.0, 0.05]])
    fwd = np.ones(3) / np.sqrt(3.0)
    right = np.array([1.0, -1.0, 0.0]) / np.sqrt(2.0)
    up = np.cross(right, fwd)
    v = _view(eye=-5.0 * fwd, forward=fwd, right=right, up=up)
    img, _ = oracle.render(levels, pal, v)
    A = 1.0 - 0.95 ** (8.0 * np.sqrt(3.0))
    np.testing.assert_allclose(img[0, 0, 3], A, atol=1e-9)         # corner to corner (rounding may clip ~1e-15 of it)
    v_miss = _view(eye=-5.0 * fwd, forward=-fwd, right=right, up=up)
    assert (oracle.render(levels, pal, v_miss)[0] == 0).all()
    v_in = _view(eye=np.array([4.0, 4.0, 4.0]), forward=np.array([1.0, 0, 0]))       # eye inside: path = 4
    np.testing.assert_allclose(oracle.render(levels, pal, v_in)[0][0, 0, 3], 1.0 - 0.95 ** 4.0, atol=1e-12)


def test_front_to_back_compositing_hand_worked():
    """4x1x1 volume seen along +x from just outside, lambda = 0, steps of 0.5 voxel: eight samples at
    x = 0.25, 0.75, ...; colour along x is the piecewise-linear interpolant of the voxel colours."""
    l0 = np.array([0, 1, 2, 3], dtype=np.uint32).reshape(1, 1, 4)
    levels = [l0, np.array([4, 5], dtype=np.uint32).reshape(1, 1, 2), np.array([[[6]]], dtype=np.uint32)]
    pal = np.array([[1, 0, 0, 0.8], [0, 1, 0, 0.1], [0, 0, 1, 0.6], [1, 1, 0, 0.0], [9, 9, 9, 1], [9, 9, 9, 1], [9, 9, 9, 1]], float)
    v = _view(eye=np.array([-0.25, 0.5, 0.5]), tan_half_fov=0.01)          # rho < 1 everywhere: lambda = 0
    img, (n_eval, _) = oracle.render(levels, pal, v)
    assert n_eval == 8
    xs = 0.25 + 0.5 * np.arange(8)
    C, A = np.zeros(3), 0.0
    for x in xs:
        c = np.array([np.interp(x, [0.5, 1.5, 2.5, 3.5], pal[:4, ch]) for ch in range(4)])
        a = 1.0 - (1.0 - c[3]) ** 0.5
        C += (1 - A) * a * c[:3]
        A += (1 - A) * a
    np.testing.assert_allclose(img[0, 0], [*C, A], atol=1e-12)
    # reversing the view changes the colour (order matters), not the opacity
    v2 = _view(eye=np.array([4.25, 0.5, 0.5]), forward=np.array([-1.0, 0, 0]), right=np.array([0, -1.0, 0]),
               tan_half_fov=0.01)
    img2, _ = oracle.render(levels, pal, v2)
    np.testing.assert_allclose(img2[0, 0, 3], A, atol=1e-12)
    assert np.abs(img2[0, 0, :3] - C).max() > 0.05


# ------------------------------------------------------------------------------------------ R2
@pytest.mark.parametrize("bias,spacing,expect", [
    (0.0, 1.0, (0.0, 0.5, 0.5)),        # rho = 2^1.5 -> lambda = 1.5: half level 1 (green), half level 2 (blue)
    (-0.5, 1.0, (0.0, 1.0, 0.0)),       # bias is additive
    (-1.5, 1.0, (1.0, 0.0, 0.0)),       # lambda = 0: level 0 (red)
    (-9.0, 1.0, (1.0, 0.0, 0.0)),       # clamped below
    (0.0, 2.0, (0.5, 0.5, 0.0)),        # voxels twice as large -> rho halves -> lambda = 0.5
])
def test_lod_is_log2_of_voxels_per_pixel_linear_in_depth(bias, spacing, expect):
    """A slab one voxel thick whose mip levels have different colours, seen head-on through ONE sample:
    rho = z (2 tan / H) / s_ref with z = 64 sqrt(2), tan = 0.25, H = 16  ->  2^1.5 voxels per pixel."""
    dims = (1, 64, 64)
    levels = _constant_pyramid(dims, node_of_level=lambda l: min(l, 3))
    pal = np.array([[1, 0, 0, 0.5], [0, 1, 0, 0.5], [0, 0, 1, 0.5], [1, 1, 1, 0.5]], float)
    z = 64.0 * np.sqrt(2.0)                                   # world units, whatever the voxel size
    v = _view(eye=np.array([-z, 32.0 * spacing, 32.0 * spacing]), tan_half_fov=0.25, lod_bias=bias, step_voxels=1.0,
              spacing=np.full(3, spacing))
    v["height"], v["width"] = 16, 16
    img, (n_eval, _) = oracle.render(levels, pal, v)
    d = oracle.pixel_ray(v, 8, 8)
    px = img[8, 8]
    assert n_eval >= 16 * 16
    # a pixel next to the axis: its path is 1 / cos > 1 voxel, so a second, ~1e-3 voxel long interval a
    # hair deeper follows the first -- hence the tolerance; a wrong factor in rho moves the mix by > 0.1
    np.testing.assert_allclose(px[:3] / px[3], expect, atol=2e-4)
    assert abs(d @ v["forward"]) > 0.999


def test_lod_clamps_to_coarsest_level():
    levels = _constant_pyramid((1, 64, 64), node_of_level=lambda l: l)
    pal = _identity_palette(7)
    pal[:, 3] = 0.5
    v = _view(eye=np.array([-100.0, 32.0, 32.0]), lod_bias=20.0, step_voxels=1.0)
    img, _ = oracle.render(levels, pal, v)
    np.testing.assert_allclose(img[0, 0, :3] / img[0, 0, 3], pal[6, :3], atol=1e-12)


# ------------------------------------------------------------------------------------------ R6
def _direct_pyramid(S, tf):
    """One palette entry per mip voxel holding the direct histogram colour (pinned O-2): a pyramid that
    is consistent with the definition, built without any graph."""
    ids, seg = oracle.leaf_index(S)
    H = oracle.histogram_mipmap(seg, ids.size)
    levels, pal, n = [], [], 0
    for l, h in enumerate(H):
        c = oracle.direct_colour(h, l, tf).reshape(-1, 4)
        levels.append((np.arange(c.shape[0], dtype=np.uint32) + n).reshape(h.shape[:3]))
        pal.append(c)
        n += c.shape[0]
    return levels, np.concatenate(pal)


def test_empty_space_skipping_never_changes_the_image():
    """A ball of coloured segments in an exactly transparent background: skipped samples have their whole
    footprint inside a block of opacity 0, so the image is identical with and without ESS (L271)."""
    n = 32
    z, y, x = np.mgrid[:n, :n, :n]
    r2 = (x - 15.5) ** 2 + (y - 13.5) ** 2 + (z - 17.5) ** 2
    S = np.where(r2 < 7.5 ** 2, 1 + ((x // 3 + y // 5 + z // 4) % 5), 0).astype(np.uint32)
    tf = synth.random_tf(6, 9).astype(np.float64)
    tf[0, 3] = 0.0
    levels, pal = _direct_pyramid(S, tf)
    base = synth.orbit_view((n, n, n), width=40, height=30, distance=0.9, ess_threshold=-1.0)
    img0, (e0, s0) = oracle.render(levels, pal, base)
    img1, (e1, s1) = oracle.render(levels, pal, dict(base, ess_threshold=1e-8))
    assert s0 == 0 and s1 > 0 and e1 + s1 == e0 and s1 > 0.2 * e0, (e0, e1, s1)
    np.testing.assert_allclose(img1, img0, rtol=0, atol=1e-13)
    assert img0[..., 3].max() > 0.5 and (img0[..., 3] == 0).any()


def test_render_pixels_is_render_restricted_to_those_pixels():
    dims = (13, 7, 5)
    levels, n = [], 0
    for (x, y, z) in oracle.mip_dims(dims):
        levels.append((np.arange(x * y * z, dtype=np.uint32) + n).reshape(z, y, x))
        n += x * y * z
    pal = synth.random_attr(n, 4, seed=5).astype(np.float64)
    view = synth.orbit_view(dims, width=9, height=7, distance=0.8)
    img, st = oracle.render(levels, pal, view)
    ij = [(0, 0), (8, 6), (4, 3), (2, 5)]
    px, _ = oracle.render_pixels(levels, pal, view, ij)
    np.testing.assert_array_equal(px, np.stack([img[j, i] for i, j in ij]))
    every = [(i, j) for j in range(7) for i in range(9)]
    px_all, st_all = oracle.render_pixels(levels, pal, view, every)
    np.testing.assert_array_equal(px_all.reshape(7, 9, 4), img)
    assert st_all == st


def test_empty_mode_state_machine_hand_worked():
    """R6: the hierarchy is consulted only in empty mode (on entry, and after a skipped or transparent sample).
    32 x 1 x 1 voxels, opaque for x < 8 and x >= 24, exactly transparent in between; ray along +x, lambda = 0,
    2-voxel steps: samples at x = 1, 3, ..., 31 (footprint = voxels floor(x - 1/2), +1; block margin 2^l1 / 2 = 1).
      x = 1 .. 7   evaluated (x = 1 climbs first -- the ray enters in empty mode -- and finds [0, 4) occupied)
      x = 9        evaluated although it lies in the empty block [8, 16): the sample before it was opaque;
                   its opacity is 0, so the ray is in empty mode from here
      x = 11, 13   skipped (9 <= x < 15);  x = 15 evaluated (outside the margin), transparent
      x = 17       skipped at once: still in empty mode, new block [16, 24), 17 <= x < 23;  x = 19, 21 skipped
      x = 23       evaluated (voxels 22, 23 are empty -> transparent), x = 25 .. 31 evaluated (opaque)
    => 11 samples evaluated, 5 skipped; an eager climb before every sample would have skipped x = 9 too."""
    x = np.arange(32)
    S = np.where((x < 8) | (x >= 24), 1, 0).astype(np.uint32).reshape(1, 1, 32)
    tf = np.array([[0.3, 0.3, 0.3, 0.0], [0.9, 0.2, 0.1, 0.5]])
    levels, pal = _direct_pyramid(S, tf)
    v = _view(eye=np.array([-1.0, 0.5, 0.5]), tan_half_fov=1e-4, step_voxels=2.0, ess_threshold=1e-8)
    img, (n_eval, n_skip) = oracle.render(levels, pal, v)
    assert (n_eval, n_skip) == (11, 5)
    img0, (e0, s0) = oracle.render(levels, pal, dict(v, ess_threshold=-1.0))
    assert (e0, s0) == (16, 0)
    np.testing.assert_allclose(img, img0, atol=1e-15)
