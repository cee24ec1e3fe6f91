"""Seeded random cases for the NEXT rows against the oracle: the ray-marcher on random volumes (down to 1 x k x m),
images, views, spacings, thresholds and both mipmap modes; range queries (both work distributions and the naive scan)
and the device mipmap front end on random volumes and quantiser bitrates.  Helpers and tolerances are those of
test_gpu_render.py / test_gpu_query.py / test_gpu_mipmap.py."""
import os
import sys

import numpy as np
import pytest

import oracle
from paper_2009_02702_b200 import builder, synth

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import test_gpu_mipmap as M  # noqa: E402
import test_gpu_query as Q  # noqa: E402
import test_gpu_render as R  # noqa: E402

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

@pytest.fixture(scope="module")
def mg():
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2009_02702_b200 import mg as _mg
    torch.cuda.set_device(0)
    return _mg

def rnd(seed, stream, lo, hi):
    """A seeded integer in [lo, hi]."""
    return lo + int(int(synth.u64(seed, stream, np.arange(1, dtype=np.uint64))[0]) % (hi - lo + 1))

@pytest.mark.parametrize("seed", range(40))
def test_render_random(mg, seed):
    dims = (rnd(seed, 1, 1, 40), rnd(seed, 2, 1, 40), rnd(seed, 3, 1, 40))
    nseg = rnd(seed, 4, 1, 12)
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, min(nseg, dims[0]*dims[1]*dims[2]), 100 + seed))
    nl = int(np.unique(seg).size)
    tf = synth.random_tf(nl, 200 + seed, alpha_zero_frac=[0.0, 0.3, 0.7][seed % 3])
    tf[:, 3] *= [1.0, 0.2, 0.05][(seed // 3) % 3]
    view = synth.orbit_view(dims, spacing=(1.0, [1.0, 2.5][seed % 2], [1.0, 7.0, 0.5][seed % 3]), width=rnd(seed, 5, 1, 50), height=rnd(seed, 6, 1, 40),
                            azimuth_deg=rnd(seed, 7, 0, 359), elevation_deg=rnd(seed, 8, -89, 89), distance=[0.05, 0.6, 1.5, 4.0][seed % 4],
                            fov_deg=rnd(seed, 9, 10, 100), step_voxels=[0.5, 0.25, 1.3][seed % 3], lod_bias=[0.0, 1.0, -1.0, 2.5][(seed // 2) % 4],
                            ess_threshold=[1e-8, -1.0, 0.01][seed % 3], alpha_cutoff=[1.0, 0.9][seed % 2])
    view["flags"] = seed % 2
    got, gs, ref, rs = R._volume_case(mg, seg, tf, view)
    R._assert_image(got, gs, ref, rs)

@pytest.mark.parametrize("seed", range(25))
def test_query_and_front_random(mg, seed):
    dims = (rnd(seed, 11, 1, 50), rnd(seed, 12, 1, 50), rnd(seed, 13, 1, 50))
    nseg = min(rnd(seed, 14, 1, 15), dims[0]*dims[1]*dims[2])
    bits = [9, 0, 4, 12][seed % 4]
    seg_index, gr, levels, g, d_idx, mip = Q._volume(mg, dims, nseg, 300 + seed, quant_bits=bits)
    nl = gr["n_leaves"]
    lut = g.mixture_lut(gr["weight_sigma"])
    mu, dmu = oracle.mixture_lut(gr["child_a"], gr["child_b"], gr["weight"].astype(np.float64), gr["weight_sigma"], nl)
    boxes = Q._boxes(dims, 12, 400 + seed)
    boxes = [b for b in boxes if all(b[a] < b[3+a] for a in range(3))]
    for mode in (mg.MG_QUERY_FA, mg.MG_QUERY_FA_WALK):
        e, d, f = Q._query(lut, d_idx, mip, boxes, nl, mode)
        for q, box in enumerate(boxes):
            vol = np.prod([box[3+a]-box[a] for a in range(3)])
            re_, rd, rf = oracle.range_query_fa(levels, mu, dmu, box)
            np.testing.assert_allclose(e[q], re_, rtol=0, atol=1e-9*vol); np.testing.assert_allclose(d[q], rd, rtol=1e-9, atol=1e-12*vol); assert f[q] == rf
    e, d, f = Q._query(lut, d_idx, mip, boxes, nl, mg.MG_QUERY_NAIVE)
    for q, (x0,y0,z0,x1,y1,z1) in enumerate(boxes):
        assert np.array_equal(e[q], np.bincount(seg_index[z0:z1,y0:y1,x0:x1].reshape(-1), minlength=nl))
    lut.close(); g.close()
    # device front end + build_from_level1 == build
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, nseg, 300 + seed))
    ids, l0, l1, mv, mc, nm = M._front(mg, seg)
    a = builder.build(seg, quant_bits=bits); b = builder.build_from_level1(dims, ids, l1, mv[:nm], mc[:nm], quant_bits=bits)
    for k in ("child_a", "child_b", "weight", "level_offsets"): assert np.array_equal(a.graph()[k], b.graph()[k])
    for l in range(1, a.info.n_mip_levels): assert np.array_equal(a.node_idx(l), b.node_idx(l))
