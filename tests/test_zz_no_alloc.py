"""mg_index_ranges_static: the entry point for callers that cannot allocate device memory.

Some users of the library run inside a process whose own arena holds all of the GPU's memory (a renderer's resource
pool, a framework's caching allocator), or inside a frame loop where the device-wide wait of a cudaFree is not
affordable; mg_index_range's cudaMalloc / cudaFree per call is closed to them.  mg_index_ranges_static keeps its scratch
(one (min, max) pair per level, at most MG_INDEX_RANGES_STATIC_MAX_LEVELS levels) in a fixed array inside libmg.so,
which every call shares and which still holds the previous call's values when the next one starts.

The checks: the ranges equal mg_index_range's level by level (integers: exactly) on two calls in a row, the second on
data whose ranges lie strictly inside the first's (so pairs left over from the first call would show), and a request
beyond the array's size is refused.  This file sorts after every other test file on purpose: under `pytest -x` a
failure here hides nothing.  It builds all it needs itself, so it passes alone in a fresh process as well.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _levels(rng, sizes, lo, hi):
    return [rng.integers(lo, hi, size=n, dtype=np.uint32) for n in sizes]


def _both_paths(mg, torch, levels, lead=0):
    """Ranges of `levels` (concatenated behind `lead` unused elements, so that levels start at any 4-byte alignment)
    through mg_index_range level by level and through mg_index_ranges_static in one call."""
    flat = np.concatenate([np.zeros(lead, np.uint32)] + levels)
    off = lead + np.concatenate([[0], np.cumsum([lv.size for lv in levels])]).astype(np.uint64)
    d = torch.from_numpy(flat.view(np.int32)).cuda()
    want = [mg.index_range(d[int(off[l]):], int(off[l + 1] - off[l])) for l in range(len(levels))]
    lo, hi = mg.index_ranges_static(d, off)
    return want, list(zip(lo.tolist(), hi.tolist()))


def test_static_ranges_equal_the_allocating_path_on_two_calls_in_a_row():
    import torch
    from paper_2009_02702_b200 import mg
    rng = np.random.default_rng(20260)
    sizes = [300_001, 37_512, 4_689, 587, 74, 10, 2, 1]               # a mip chain: several CTAs down to one voxel
    first = _levels(rng, sizes, 0, 2_000_000)                            # wide ranges ...
    want1, got1 = _both_paths(mg, torch, first, lead=1)
    assert got1 == want1
    assert got1 == [(int(lv.min()), int(lv.max())) for lv in first]
    second = _levels(rng, sizes[:5], 700_000, 700_900)                   # ... then narrow ones inside them, fewer levels
    want2, got2 = _both_paths(mg, torch, second, lead=3)
    assert got2 == want2
    assert got2 == [(int(lv.min()), int(lv.max())) for lv in second]


def test_static_ranges_limit_and_empty_levels():
    import torch
    from paper_2009_02702_b200 import mg
    n_max = mg.MG_INDEX_RANGES_STATIC_MAX_LEVELS
    d = torch.arange(5, 5 + 4 * (n_max + 1), dtype=torch.int32, device="cuda")
    off = np.arange(0, 4 * (n_max + 1) + 1, 4, dtype=np.uint64)          # n_max + 1 levels of 4 voxels
    with pytest.raises(mg.MgError) as ei:
        mg.index_ranges_static(d, off)
    assert ei.value.code == mg.MG_ERR_INVALID_ARG and "MG_INDEX_RANGES_STATIC_MAX_LEVELS" in str(ei.value)
    lo, hi = mg.index_ranges_static(d, off[:n_max + 1])                  # exactly the maximum is served
    assert lo.tolist() == [5 + 4 * l for l in range(n_max)] and hi.tolist() == [8 + 4 * l for l in range(n_max)]
    lo, hi = mg.index_ranges_static(d, np.array([0, 3, 3, 7], np.uint64))   # an empty level reports (UINT32_MAX, 0)
    assert list(zip(lo.tolist(), hi.tolist())) == [(5, 7), (0xFFFFFFFF, 0), (8, 11)]
    with pytest.raises(mg.MgError):
        mg.index_ranges_static(d, np.array([0, 4, 2], np.uint64))        # decreasing offsets
