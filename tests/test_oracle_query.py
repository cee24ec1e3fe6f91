"""Pins of the oracle's mixture lookup table (Eq. 17-18) and footprint-assembly range queries (NEXT-4;
PAPER.md sections 3.5-3.6, L375-L377, Table 4).  Nothing here calls the CUDA path."""
import os

import numpy as np
import pytest

import oracle
from paper_2009_02702_b200 import synth


# ------------------------------------------------------------------------------ 1D decomposition
def test_fa_axis_tiles_every_range_with_maximal_aligned_pieces():
    for lo in range(0, 41):
        for hi in range(lo + 1, 42):
            segs = oracle.fa_axis(lo, hi, 10)
            x = lo
            for s, l in segs:
                assert s == x and s % (1 << l) == 0                     # contiguous, aligned to its own size
                big = 1 << (l + 1)
                assert s % big != 0 or s + big > hi                      # ... and not extendable (maximal)
                x += 1 << l
            assert x == hi
    assert oracle.fa_axis(0, 64, 10) == [(0, 6)]
    assert oracle.fa_axis(0, 64, 3) == [(8 * k, 3) for k in range(8)]     # capped at the coarsest level
    assert oracle.fa_axis(3, 20, 10) == [(3, 0), (4, 2), (8, 3), (16, 2)]  # hand-worked: 1 + 4 + 8 + 4


def _fetch_count(box_lo, side, max_level=30):
    segs = [oracle.fa_axis(box_lo[a], box_lo[a] + side, max_level) for a in range(3)]
    n = 0
    for _, lx in segs[0]:
        for _, ly in segs[1]:
            for _, lz in segs[2]:
                l = min(lx, ly, lz)
                n += 1 << (lx + ly + lz - 3 * l)
    return n


def test_fa_fetch_counts_reproduce_table_4(golden_dir):
    """Mean fetches over random alignments: inside the spread of the paper's three data sets (+- 12 %)."""
    rows = [l.split() for l in open(os.path.join(golden_dir, "table4_fetches.txt")) if l.strip() and l[0] != "#"]
    for r in rows:
        side, paper = int(r[0]), [float(v) for v in r[1:]]
        lo = (synth.u64(7, side, np.arange(1500, dtype=np.uint64)) % np.uint64(1024)).astype(np.int64).reshape(-1, 3)
        mean = np.mean([_fetch_count(b, side) for b in lo])
        assert 0.88 * min(paper) <= mean <= 1.12 * max(paper), (side, mean, paper)
        assert abs((1 - mean / side ** 3) - (1 - np.mean(paper) / side ** 3)) < 0.035    # the "saved" column


# ------------------------------------------------------------------------------ Eq. 17-18
def test_mixture_lut_hand_worked_eq18():
    """3 leaves; n3 = lerp(0, 1; w = 1/4, dw = 0.01); n4 = lerp(n3, 2; w = 1/2, dw = 0.02).
    n3: mu = (3/4, 1/4, 0); both children exact, so dmu_i = mu_i sqrt(2) (0.01 / 0.25) = mu_i 0.0565685...
    n4: mu = (3/8, 1/8, 1/2); component 0: rel^2 = (dmu3_0 / mu3_0)^2 + 2 (0.02 / 0.5)^2 = 0.0032 + 0.0032,
        component 2 comes from the exact leaf only: rel^2 = 2 (0.04)^2 = 0.0032."""
    a = np.array([0, 0, 0, 0, 3], np.uint32)
    b = np.array([0, 0, 0, 1, 2], np.uint32)
    w = np.array([0, 0, 0, 0.25, 0.5])
    sg = np.array([0, 0, 0, 0.01, 0.02])
    mu, dmu = oracle.mixture_lut(a, b, w, sg, 3)
    np.testing.assert_allclose(mu[3], [0.75, 0.25, 0.0], atol=1e-15)
    np.testing.assert_allclose(mu[4], [0.375, 0.125, 0.5], atol=1e-15)
    np.testing.assert_allclose(dmu[:3], 0.0)
    np.testing.assert_allclose(dmu[3], [0.75 * 0.05656854249, 0.25 * 0.05656854249, 0.0], atol=1e-10)
    np.testing.assert_allclose(dmu[4], [0.375 * 0.08, 0.125 * 0.08, 0.5 * 0.05656854249], atol=1e-10)


def test_mixture_lut_mu_is_symbolic_eval_and_zero_sigma_gives_zero_error():
    sizes = [7, 30, 20, 9, 3, 1]
    a, b, w, off = synth.random_dag_levels(sizes, seed=70)
    mu, dmu = oracle.mixture_lut(a, b, w, np.zeros(a.size), sizes[0])
    np.testing.assert_array_equal(mu, oracle.symbolic_eval(a, b, w, sizes[0]))       # O-5, pinned elsewhere
    assert (dmu == 0).all()
    sg = 0.003 * np.ones(a.size)
    mu2, dmu2 = oracle.mixture_lut(a, b, w, sg, sizes[0])
    assert ((dmu2 > 0) == (mu2 > 0))[sizes[0]:].all()                                 # an error wherever a component is
    _, dmu3 = oracle.mixture_lut(a, b, w, 2 * sg, sizes[0])
    np.testing.assert_allclose(dmu3, 2 * dmu2, rtol=1e-12)                            # Eq. 18 is homogeneous in dw


# ------------------------------------------------------------------------------ range queries
def _case(dims, n_seg, seed, quant_bits=9):
    """A volume, a Mixture Graph of its histogram mipmap and the per-level node indices, made HERE from the oracle's
    exact integer histograms (no product code): every distinct mixture (m_1 .. m_k on leaves i_1 < .. < i_k) becomes the
    chain n_1 = leaf i_1, n_j = (1 - w_j) n_{j-1} + w_j leaf i_j with w_j = m_j / (m_1 + .. + m_j) (Eq. 5-7 applied
    k - 1 times), nodes shared through a dictionary (L144).  quant_bits > 0: w is replaced by the mid-point of its
    2^b-bin and every node carries that bin's sigma = 2^-b / sqrt(12) (L176)."""
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, n_seg, seed))
    ids, seg_index = oracle.leaf_index(seg)
    nl = ids.size
    a, b, w, wq = [0] * nl, [0] * nl, [0.0] * nl, [0.0] * nl
    node_of, levels = {}, []
    for H in oracle.histogram_mipmap(seg_index, nl):
        flat = H.reshape(-1, nl)
        idx = np.zeros(flat.shape[0], dtype=np.uint32)
        for v, row in enumerate(flat):
            leaves = np.flatnonzero(row)
            node, mass = int(leaves[0]), int(row[leaves[0]])
            for j in leaves[1:]:
                mass += int(row[j])
                ratio = int(row[j]) / mass
                q = (min((1 << quant_bits) - 1, int(ratio * (1 << quant_bits))) + 0.5) / (1 << quant_bits) if quant_bits else ratio
                key = (node, int(j), q)
                if key not in node_of:
                    node_of[key] = len(a)
                    a.append(node); b.append(int(j)); w.append(ratio); wq.append(q)
                node = node_of[key]
            idx[v] = node
        levels.append(idx.reshape(H.shape[:3]))
    n = len(a)
    sigma = np.zeros(n)
    if quant_bits:
        sigma[nl:] = 2.0 ** -quant_bits / np.sqrt(12.0)
    g = dict(child_a=np.array(a, np.uint32), child_b=np.array(b, np.uint32), weight_exact=np.array(w), n_leaves=nl,
             weight=np.array(wq, np.float32), weight_sigma=sigma)
    return seg_index, g, levels


def _boxes(dims, n, seed):
    out = []
    for q in range(n):
        r = synth.u64(seed, q, np.arange(6, dtype=np.uint64))
        lo = [int(r[a] % np.uint64(dims[a])) for a in range(3)]
        hi = [lo[a] + 1 + int(r[3 + a] % np.uint64(dims[a] - lo[a])) for a in range(3)]
        out.append(lo + hi)
    out.append([0, 0, 0, *dims])                                            # the whole volume
    out.append([dims[0] - 1, dims[1] - 1, dims[2] - 1, *dims])             # one voxel in the far corner
    return out


@pytest.mark.parametrize("dims", [(32, 32, 32), (37, 29, 23)])
def test_fa_equals_brute_force_count_on_the_unquantised_graph(dims):
    """Exact weights: FA == naive == the plain count of voxels per segment in the box (np.bincount)."""
    seg_index, g, levels = _case(dims, 9, 31, quant_bits=0)
    nl = g["n_leaves"]
    mu, dmu = oracle.mixture_lut(g["child_a"], g["child_b"], g["weight_exact"], g["weight_sigma"], nl)
    assert (dmu == 0).all()
    for box in _boxes(dims, 25, 32):
        x0, y0, z0, x1, y1, z1 = box
        truth = np.bincount(seg_index[z0:z1, y0:y1, x0:x1].reshape(-1), minlength=nl).astype(np.float64)
        e, d, nf = oracle.range_query_fa(levels, mu, dmu, box)
        en, nn = oracle.range_query_naive(levels[0], mu, box)
        vol = (x1 - x0) * (y1 - y0) * (z1 - z0)
        np.testing.assert_allclose(e, truth, rtol=0, atol=1e-9 * vol)
        np.testing.assert_array_equal(en, truth)
        assert nn == vol and nf <= vol and (d == 0).all()
    e, d, nf = oracle.range_query_fa(levels, mu, dmu, [0, 0, 0, 32, 32, 32]) if dims == (32, 32, 32) else (None, None, 1)
    assert nf == 1                                                          # a whole power-of-two volume is ONE fetch


def test_quantised_query_sums_to_the_volume_and_error_bars_cover():
    """b = 9: 'the sum of the expectations always sum up exactly to the volume of the query region' (L251);
    the deviation from the true count stays within a few predicted error bars + is small (L251: ~0.3 %)."""
    dims = (37, 29, 23)
    seg_index, g, levels = _case(dims, 9, 33)
    nl = g["n_leaves"]
    mu, dmu = oracle.mixture_lut(g["child_a"], g["child_b"], g["weight"].astype(np.float64), g["weight_sigma"], nl)
    worst = 0.0
    for box in _boxes(dims, 25, 34):
        x0, y0, z0, x1, y1, z1 = box
        vol = (x1 - x0) * (y1 - y0) * (z1 - z0)
        truth = np.bincount(seg_index[z0:z1, y0:y1, x0:x1].reshape(-1), minlength=nl)
        e, d, nf = oracle.range_query_fa(levels, mu, dmu, box)
        assert abs(e.sum() - vol) <= 1e-9 * vol
        assert (e >= 0).all() and (d >= 0).all() and ((d > 0) <= (e > 0)).all()
        worst = max(worst, np.abs(e - truth).max() / vol)
    assert worst < 0.01, worst
