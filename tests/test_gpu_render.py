"""NEXT-2: mg_render (CUDA ray-marcher over the paletted mipmap) against the CPU fp64 oracle.

The oracle's inputs never come from the CUDA path: its palette is oracle.graph_eval (fp64) on the
same graph, the GPU's is what mg_propagate wrote (fp32).

Tolerance: the kernel computes the ray parameter, the step and the sample
positions in fp64 with the oracle's formulas, so the samples coincide to ~1e-12 voxels; what
differs is fp32 colour arithmetic: the palette (<= 2e-7), the fractional LOD (log2f: <= 2e-6 on
the blend factor), trilinear weights and the opacity correction -- a relative error of a few 1e-7
on each sample's contribution; the contributions are summed in fp64 and their weights sum to <= 1.
Bound used: 5e-6 max-abs on every channel of every pixel (measured: <= 2e-7).  The sample counters
are diagnostics decided by fp comparisons on both sides (fp32 palette vs fp64 palette on `alpha < threshold`): the totals must be equal, the split is compared
to 0.1 %.
"""
import numpy as np
import pytest

import oracle
from paper_2009_02702_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 5e-6


@pytest.fixture(scope="module")
def mg():
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2009_02702_b200 import mg as _mg
    torch.cuda.set_device(0)
    return _mg


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _trivial_graph(mg, n_nodes):
    """n_nodes leaves, no internal node: the palette IS the transfer function."""
    z = np.zeros(n_nodes, np.uint32)
    return mg.Graph(z, z, np.zeros(n_nodes, np.float32), n_nodes,
                    level_offsets=np.array([0, n_nodes], dtype=np.uint64))


def _gpu_render(mg, g, levels, pal32_dev, view, align=1):
    """levels: list of uint32 [Z,Y,X]; concatenated with each level padded to `align` voxels."""
    offs, dims, flat, pos = [], [], [], 0
    for lv in levels:
        offs.append(pos)
        dims.append((lv.shape[2], lv.shape[1], lv.shape[0]))
        pad = (-lv.size) % align
        flat.append(np.concatenate([lv.reshape(-1), np.zeros(pad, np.uint32)]))
        pos += lv.size + pad
    d_idx = _dev(np.concatenate(flat).view(np.int32))
    H, W = int(view["height"]), int(view["width"])
    out = torch.full((H, W, 4), float("nan"), dtype=torch.float32, device="cuda")
    stats = torch.zeros(4, dtype=torch.int64, device="cuda")
    g.render(d_idx, (offs, dims), pal32_dev, view, out, stats)
    torch.cuda.synchronize()
    if view["ess_threshold"] >= 0 and 3 <= len(levels) <= 18:
        # the same image through mg_render_ex with the empty-space mask of mg_ess_mask_build: the mask holds exactly the
        # comparisons of R6's climb, so image AND counters must be bit-identical
        mask = torch.full((levels[2].size,), -1, dtype=torch.int16, device="cuda")
        g.ess_mask_build(d_idx, (offs, dims), pal32_dev, view["ess_threshold"], mask)
        out_m = torch.full((H, W, 4), float("nan"), dtype=torch.float32, device="cuda")
        stats_m = torch.zeros(4, dtype=torch.int64, device="cuda")
        g.render(d_idx, (offs, dims), pal32_dev, view, out_m, stats_m, ess_mask_device=mask)
        torch.cuda.synchronize()
        assert torch.equal(out, out_m) and torch.equal(stats, stats_m), (stats.tolist(), stats_m.tolist())
    s = stats.cpu().numpy()
    assert s[2] <= s[0] and s[3] == 0 and (s[2] == 0 or view.get("flags", 0))
    return out.cpu().numpy().astype(np.float64), (int(s[0]), int(s[1]), int(s[2]))


def _volume_case(mg, seg, tf, view, **builder_params):
    """Builder graph of `seg` -> (GPU image via mg_propagate + mg_render, oracle image)."""
    from paper_2009_02702_b200 import builder
    r = builder.build(seg, **builder_params)
    gr = r.graph()
    levels = [r.node_idx(l) for l in range(r.info.n_mip_levels)]
    g = mg.Graph(gr["child_a"], gr["child_b"], gr["weight"], gr["n_leaves"], level_offsets=gr["level_offsets"],
                 leaf_segment_id=gr["leaf_segment_id"])
    nodes = torch.empty((gr["child_a"].size, 4), dtype=torch.float32, device="cuda")
    g.propagate(_dev(tf), nodes)
    got, gstats = _gpu_render(mg, g, levels, nodes, view, align=64)
    pal = oracle.graph_eval(gr["child_a"], gr["child_b"], gr["weight"], gr["n_leaves"], tf.astype(np.float64))
    ref, rstats = oracle.render(levels, pal, view)
    g.close()
    r.close()
    return got, gstats, ref, rstats


def _assert_image(got, gstats, ref, rstats, tol=TOL):
    n_uniform, gstats = gstats[2], gstats[:2]
    err = np.abs(got - ref).max()
    print(f"render max|err| = {err:.3e}, samples (evaluated, skipped): gpu {gstats} oracle {rstats}")
    assert err <= tol, err
    # t, the step and the accumulated opacity are fp64 on both sides, so the marches stop at the same sample
    tot_g, tot_r = sum(gstats), sum(rstats)
    assert tot_g == tot_r, (gstats, rstats)
    assert abs(gstats[0] - rstats[0]) <= max(2, 1e-3 * tot_r), (gstats, rstats)
    return n_uniform


VIEWS = {
    "default": dict(),
    "close_up": dict(distance=0.45, fov_deg=60.0, azimuth_deg=-70.0, elevation_deg=35.0),
    "far_coarse": dict(distance=3.0, lod_bias=1.5, azimuth_deg=200.0, elevation_deg=-15.0),
    "top_down": dict(elevation_deg=89.9, distance=1.2),
    "no_ess_cutoff": dict(ess_threshold=-1.0, alpha_cutoff=0.95, azimuth_deg=110.0),
    "big_steps": dict(step_voxels=1.7, ref_step_voxels=0.5, lod_bias=-0.7),
}


@pytest.mark.parametrize("flags", [0, 1])
@pytest.mark.parametrize("name", list(VIEWS))
def test_render_voronoi_ragged_matches_oracle(mg, name, flags):
    """37 x 29 x 23 (ragged ceil-halving chain), 12 segments, a third of them exactly transparent, b = 9."""
    dims = (37, 29, 23)
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, 12, 21))
    tf = synth.random_tf(int(np.unique(seg).size), 21, alpha_zero_frac=0.35)
    view = synth.orbit_view(dims, width=67, height=45, **VIEWS[name])      # 67 x 45: ragged tiles
    view["flags"] = flags                                                   # 1 = MG_VIEW_HISTOGRAM_MIPMAP
    got, gs, ref, rs = _volume_case(mg, seg, tf, view)
    n_uniform = _assert_image(got, gs, ref, rs)
    assert ref[..., 3].max() > 0.3
    if name in ("default", "close_up", "top_down"):
        assert gs[1] > 0, "empty-space skipping never triggered"
        assert (n_uniform > 0) == bool(flags), "the one-leaf shortcut never fired"


def test_render_anisotropic_spacing_matches_oracle(mg):
    """1 : 1 : 7 voxels (L277) and a z-stretched Voronoi metric, like config 3."""
    dims = (48, 40, 9)
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, 20, 22), zscale=7)
    tf = synth.random_tf(int(np.unique(seg).size), 22, alpha_zero_frac=0.3)
    view = synth.orbit_view(dims, spacing=(1.0, 1.0, 7.0), width=64, height=64, distance=0.8, elevation_deg=40.0)
    got, gs, ref, rs = _volume_case(mg, seg, tf, view)
    _assert_image(got, gs, ref, rs)
    got, gs, ref, rs = _volume_case(mg, seg, tf, dict(view, flags=1))
    assert _assert_image(got, gs, ref, rs) > 0


def _unit_view(**kw):
    v = dict(width=1, height=1, eye=np.zeros(3), right=np.array([0.0, 1.0, 0.0]), up=np.array([0.0, 0.0, 1.0]),
             forward=np.array([1.0, 0.0, 0.0]), tan_half_fov=0.5, spacing=np.ones(3), step_voxels=0.5,
             ref_step_voxels=1.0, lod_bias=0.0, ess_threshold=-1.0, alpha_cutoff=1.0)
    v.update(kw)
    return v


@pytest.mark.parametrize("spacing,axis,length", [((1, 1, 1), 0, 8.0), ((1, 1, 7), 2, 56.0), ((2, 3, 4), 1, 24.0)])
@pytest.mark.parametrize("bias", [0.0, 3.0])
def test_render_homogeneous_volume_closed_form(mg, spacing, axis, length, bias):
    """Beer-Lambert, straight from the mathematics (no oracle call): A = 1 - (1 - a)^(path / (ref s_ref))."""
    levels = [np.zeros((z, y, x), np.uint32) for (x, y, z) in oracle.mip_dims((8, 8, 8))]
    pal = np.array([[0.2, 0.5, 0.9, 0.3]], dtype=np.float32)
    e = np.eye(3)
    fwd = e[axis]
    ext = 8.0 * np.array(spacing, dtype=np.float64)
    eye = 0.5 * ext - fwd * (0.5 * ext[axis] + 11.0)
    v = _unit_view(eye=eye, forward=fwd, right=e[(axis + 1) % 3], up=e[(axis + 2) % 3],
                   spacing=np.array(spacing, float), lod_bias=bias, ref_step_voxels=2.0, step_voxels=0.37)
    g = _trivial_graph(mg, 1)
    img, (n_eval, n_skip, _) = _gpu_render(mg, g, levels, _dev(pal), v)
    A = 1.0 - (1.0 - 0.3) ** (length / (2.0 * min(spacing)))
    np.testing.assert_allclose(img[0, 0], [0.2 * A, 0.5 * A, 0.9 * A, A], rtol=0, atol=TOL)
    assert n_eval > 0 and n_skip == 0
    g.close()


def test_render_identity_pyramid_all_footprints_distinct(mg):
    """Every mip voxel has its own palette entry (no 'same node' shortcut, both levels fetched)."""
    dims = (13, 7, 5)
    levels, n = [], 0
    for (x, y, z) in oracle.mip_dims(dims):
        levels.append((np.arange(x * y * z, dtype=np.uint32) + n).reshape(z, y, x))
        n += x * y * z
    pal = synth.random_attr(n, 4, seed=5)
    pal[:, 3] *= 0.2
    g = _trivial_graph(mg, n)
    for kw in (dict(distance=0.7), dict(distance=2.5, lod_bias=2.2), dict(distance=1.0, ess_threshold=0.05)):
        view = synth.orbit_view(dims, width=33, height=31, **kw)
        got, gs = _gpu_render(mg, g, levels, _dev(pal), view)
        ref, rs = oracle.render(levels, pal.astype(np.float64), view)
        _assert_image(got, gs, ref, rs)
    g.close()


def test_render_ess_on_off_same_image_and_misses_are_zero(mg):
    """A ball in an exactly transparent background: ESS skips samples but cannot change the image (L271);
    rays that miss the box write zeros."""
    n = 32
    z, y, x = np.mgrid[:n, :n, :n]
    r2 = (x - 15.5) ** 2 + (y - 13.5) ** 2 + (z - 17.5) ** 2
    seg = np.where(r2 < 7.5 ** 2, 1 + ((x // 3 + y // 5 + z // 4) % 5), 0).astype(np.uint32)
    tf = synth.random_tf(6, 9)
    tf[0, 3] = 0.0
    base = synth.orbit_view((n, n, n), width=80, height=60, distance=1.4, fov_deg=70.0, ess_threshold=-1.0)
    got0, gs0, ref0, rs0 = _volume_case(mg, seg, tf, base)
    got1, gs1, ref1, rs1 = _volume_case(mg, seg, tf, dict(base, ess_threshold=1e-8))
    _assert_image(got0, gs0, ref0, rs0)
    _assert_image(got1, gs1, ref1, rs1)
    assert gs0[1] == 0 and gs1[1] > 0.2 * gs0[0]
    assert np.abs(got1 - got0).max() <= 1e-6
    miss = ref0[..., 3] == 0
    assert miss.any() and (got0[miss] == 0).all()


def test_render_eye_inside_volume(mg):
    dims = (24, 24, 24)
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, 9, 23))
    tf = synth.random_tf(int(np.unique(seg).size), 23)
    tf[:, 3] *= 0.1
    view = synth.orbit_view(dims, width=32, height=32, distance=0.1, fov_deg=90.0)
    got, gs, ref, rs = _volume_case(mg, seg, tf, view)
    _assert_image(got, gs, ref, rs)


def test_render_error_paths(mg):
    g = _trivial_graph(mg, 1)
    pal = _dev(np.array([[0.1, 0.2, 0.3, 0.4]], np.float32))
    idx = torch.zeros(16, dtype=torch.int32, device="cuda")
    out = torch.zeros((4, 4, 4), dtype=torch.float32, device="cuda")
    good_mip = ([0, 8], [(2, 2, 2), (1, 1, 1)])
    view = synth.orbit_view((2, 2, 2), width=4, height=4)
    g.render(idx, good_mip, pal, view, out)                                    # the good call works
    torch.cuda.synchronize()
    cases = [
        (good_mip, dict(view, width=0)),
        (good_mip, dict(view, step_voxels=0.0)),
        (good_mip, dict(view, step_voxels=1e-8)),                              # would march 3e8 steps per ray
        (good_mip, dict(view, spacing=np.array([1.0, -1.0, 1.0]))),
        (([0, 8], [(2, 2, 2), (2, 1, 1)]), view),                              # not ceil-halving
        (([0, 4], [(2, 2, 2), (1, 1, 1)]), view),                              # level 1 inside level 0
        (([], []), view),
    ]
    for mip, v in cases:
        with pytest.raises(mg.MgError) as ei:
            g.render(idx, mip, pal, v, out)
        assert ei.value.code == mg.MG_ERR_INVALID_ARG
    with pytest.raises(mg.MgError):
        g.render(idx, good_mip, pal.data_ptr() + 4, view, out)                 # misaligned palette
    with pytest.raises(mg.MgError):
        g.render(None, good_mip, pal, view, out)
    g.close()


def test_ess_mask_error_paths(mg):
    """mg_ess_mask_build needs a level 2 (3 .. 18 mip levels); mg_render_ex refuses a mask on a mipmap without one;
    with empty-space skipping off the mask is ignored."""
    g = _trivial_graph(mg, 4)
    pal = _dev(synth.random_tf(4, 90))
    two = [np.zeros((2, 2, 2), np.uint32), np.zeros((1, 1, 1), np.uint32)]
    d_idx = _dev(np.zeros(9, np.int32))
    mask = torch.zeros(8, dtype=torch.int16, device="cuda")
    desc = ([0, 8], [(2, 2, 2), (1, 1, 1)])
    with pytest.raises(mg.MgError):
        g.ess_mask_build(d_idx, desc, pal, 1e-8, mask)
    view = synth.orbit_view((2, 2, 2), width=8, height=8)
    img = torch.zeros((8, 8, 4), dtype=torch.float32, device="cuda")
    with pytest.raises(mg.MgError):
        g.render(d_idx, desc, pal, view, img, ess_mask_device=mask)
    g.render(d_idx, desc, pal, dict(view, ess_threshold=-1.0), img, ess_mask_device=mask)      # ESS off: not consulted
    torch.cuda.synchronize()
    with pytest.raises(mg.MgError):                                                            # NaN threshold
        g.ess_mask_build(d_idx, ([0, 64, 72, 73], [(4, 4, 4), (2, 2, 2), (1, 1, 1)]), pal, float("nan"), mask)
    g.close()
