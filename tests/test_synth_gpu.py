"""The GPU volume generators (libmg_synth.so) are bit-identical to the numpy recipes of synth.py."""
import numpy as np
import pytest

from paper_2009_02702_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sg():
    import torch
    assert torch.cuda.is_available()
    from paper_2009_02702_b200 import synth_gpu
    return synth_gpu


def test_config1_full_volume(sg):
    c = synth.CONFIGS[1]
    ref = synth.make_volume(c)
    got = sg.make_volume(c).cpu().numpy().view(np.uint32)
    assert np.array_equal(ref, got)


@pytest.mark.parametrize("cfg", [2, 3])
def test_voronoi_crops_of_full_size_configs(sg, cfg):
    """Crops (global coordinates, touching the far borders where the jitter clamp acts)."""
    c = synth.CONFIGS[cfg]
    X, Y, Z = c["dims"]
    for region in [(0, 3, 0, 5, 0, 40), (Z - 2, Z, Y - 4, Y, X - 33, X), (Z // 2, Z // 2 + 2, 100, 104, 500, 531)]:
        ref = synth.make_volume(c, region)
        got = sg.make_volume(c, region).cpu().numpy().view(np.uint32)
        assert np.array_equal(ref, got), (cfg, region)


def test_voronoi_more_seeds_than_one_smem_chunk(sg):
    dims = (40, 30, 20)
    seeds = synth.voronoi_seeds(dims, 3000, 9)
    ref = synth.voronoi_volume(dims, seeds, zscale=3, jitter=2, seed=9)
    got = sg.voronoi_volume(dims, seeds, zscale=3, jitter=2, seed=9).cpu().numpy().view(np.uint32)
    assert np.array_equal(ref, got)


def test_cylinders_scaled_and_crop(sg):
    c = synth.scaled_config(4, 0.12)
    ref = synth.make_volume(c)
    got = sg.make_volume(c).cpu().numpy().view(np.uint32)
    assert np.array_equal(ref, got)
    assert (ref == 0).mean() > 0.5
    c4 = dict(synth.CONFIGS[4], n_segments=400)          # full box, first 400 cylinders, a crop
    region = (290, 310, 470, 500, 280, 345)
    ref = synth.make_volume(c4, region)
    got = sg.make_volume(c4, region).cpu().numpy().view(np.uint32)
    assert np.array_equal(ref, got)
