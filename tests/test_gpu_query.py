"""NEXT-4 on the GPU: mg_mixture_lut_build and mg_range_query against the CPU fp64 oracle.

Tolerances: the table is fp64 with the oracle's formulas (mu, dmu: relative 1e-12, the only
difference is fma contraction); leaf indices and row structure bit-exact.  Query results are sums of
the same terms in another order (fp64 atomics): |expect - oracle| <= 1e-9 x box volume, errors
relative 1e-9, fetch counts bit-exact.
"""
import numpy as np
import pytest

import oracle
from paper_2009_02702_b200 import builder, synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mg():
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2009_02702_b200 import mg as _mg
    torch.cuda.set_device(0)
    return _mg


def _dense(lut, n_leaves):
    rp, leaf, mu, dmu = lut.export()
    n = rp.size - 1
    M, D = np.zeros((n, n_leaves)), np.zeros((n, n_leaves))
    rows = np.repeat(np.arange(n), np.diff(rp).astype(np.int64))
    M[rows, leaf] = mu
    D[rows, leaf] = dmu
    for i in range(n):                                                    # rows sorted by leaf, no duplicates
        c = leaf[int(rp[i]):int(rp[i + 1])]
        assert (np.diff(c.astype(np.int64)) > 0).all()
    return M, D, rp


@pytest.mark.parametrize("sizes", [[7, 30, 20, 9, 3, 1], [16, 5000, 3000, 900, 200, 40, 8, 1], [3, 2]])
@pytest.mark.parametrize("with_sigma", [False, True])
def test_mixture_lut_matches_oracle_on_random_dags(mg, sizes, with_sigma):
    """Random DAGs: the children's supports overlap, so rows are shorter than their capacity."""
    a, b, w, off = synth.random_dag_levels(sizes, seed=80 + len(sizes))
    n = a.size
    sg = (0.01 * synth.random_attr(n, 1, seed=81).reshape(-1)).astype(np.float32) if with_sigma else None
    g = mg.Graph(a, b, w, sizes[0], level_offsets=off)
    lut = g.mixture_lut(sg)
    M, D, rp = _dense(lut, sizes[0])
    mu, dmu = oracle.mixture_lut(a, b, w.astype(np.float64), np.zeros(n) if sg is None else sg.astype(np.float64), sizes[0])
    assert ((M != 0) == (mu != 0)).all()
    np.testing.assert_allclose(M, mu, rtol=1e-12, atol=0)
    np.testing.assert_allclose(D, dmu, rtol=1e-12, atol=1e-300)
    np.testing.assert_allclose(M.sum(axis=1), 1.0, atol=1e-12)
    i = lut.info
    assert i.n_nodes == n and i.n_leaves == sizes[0] and i.nnz == int((mu != 0).sum()) and i.nnz <= i.capacity
    assert i.max_row_nnz == int((mu != 0).sum(axis=1).max())
    lut.close()
    g.close()


def _volume(mg, dims, n_seg, seed, **bp):
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, n_seg, seed))
    r = builder.build(seg, **bp)
    gr = r.graph()
    levels = [r.node_idx(l) for l in range(r.info.n_mip_levels)]
    g = mg.Graph(gr["child_a"], gr["child_b"], gr["weight"], gr["n_leaves"], level_offsets=gr["level_offsets"])
    offs, flat, pos = [], [], 0
    for lv in levels:
        offs.append(pos)
        pad = (-lv.size) % 64
        flat.append(np.concatenate([lv.reshape(-1), np.zeros(pad, np.uint32)]))
        pos += lv.size + pad
    d_idx = torch.from_numpy(np.concatenate(flat).view(np.int32)).cuda()
    mip = (offs, r.mip_dims)
    _, seg_index = oracle.leaf_index(seg)
    return seg_index, gr, levels, g, d_idx, mip


def _boxes(dims, n, seed):
    out = []
    for q in range(n):
        r = synth.u64(seed, q, np.arange(6, dtype=np.uint64))
        lo = [int(r[a] % np.uint64(dims[a])) for a in range(3)]
        hi = [lo[a] + 1 + int(r[3 + a] % np.uint64(dims[a] - lo[a])) for a in range(3)]
        out.append(lo + hi)
    out.append([0, 0, 0, *dims])
    out.append([dims[0] - 1, dims[1] - 1, dims[2] - 1, *dims])
    out.append([1, 1, 1, dims[0] - 1, dims[1] - 1, dims[2] - 1])
    return out


def _query(lut, d_idx, mip, boxes, n_leaves, mode, want_err=True):
    nq = len(boxes)
    e = torch.full((nq, n_leaves), float("nan"), dtype=torch.float64, device="cuda")
    d = torch.full((nq, n_leaves), float("nan"), dtype=torch.float64, device="cuda") if want_err else None
    f = torch.full((nq,), -1, dtype=torch.int64, device="cuda")
    lut.range_query(d_idx, mip, boxes, e, d, f, mode=mode)
    torch.cuda.synchronize()
    return e.cpu().numpy(), (d.cpu().numpy() if want_err else None), f.cpu().numpy()


@pytest.mark.parametrize("dims,quant_bits", [((37, 29, 23), 9), ((32, 32, 32), 9), ((37, 29, 23), 0), ((70, 9, 130), 6)])
def test_range_queries_match_oracle(mg, dims, quant_bits):
    seg_index, gr, levels, g, d_idx, mip = _volume(mg, dims, 11, 41, quant_bits=quant_bits)
    nl = gr["n_leaves"]
    lut = g.mixture_lut(gr["weight_sigma"])
    mu, dmu = oracle.mixture_lut(gr["child_a"], gr["child_b"], gr["weight"].astype(np.float64), gr["weight_sigma"], nl)
    boxes = _boxes(dims, 40, 42)
    e_fa, d_fa, f_fa = _query(lut, d_idx, mip, boxes, nl, mg.MG_QUERY_FA)
    e_nv, d_nv, f_nv = _query(lut, d_idx, mip, boxes, nl, mg.MG_QUERY_NAIVE)
    e_only, _, _ = _query(lut, d_idx, mip, boxes, nl, mg.MG_QUERY_FA, want_err=False)
    e_walk, d_walk, f_walk = _query(lut, d_idx, mip, boxes, nl, mg.MG_QUERY_FA_WALK)
    for q, box in enumerate(boxes):
        x0, y0, z0, x1, y1, z1 = box
        vol = (x1 - x0) * (y1 - y0) * (z1 - z0)
        re, rd, rf = oracle.range_query_fa(levels, mu, dmu, box)
        np.testing.assert_allclose(e_fa[q], re, rtol=0, atol=1e-9 * vol)
        np.testing.assert_allclose(e_only[q], re, rtol=0, atol=1e-9 * vol)
        np.testing.assert_allclose(e_walk[q], re, rtol=0, atol=1e-9 * vol)
        np.testing.assert_allclose(d_walk[q], rd, rtol=1e-9, atol=1e-12 * vol)
        assert f_walk[q] == rf
        np.testing.assert_allclose(d_fa[q], rd, rtol=1e-9, atol=1e-12 * vol)
        assert f_fa[q] == rf and f_nv[q] == vol
        truth = np.bincount(seg_index[z0:z1, y0:y1, x0:x1].reshape(-1), minlength=nl)
        np.testing.assert_array_equal(e_nv[q], truth)                      # level 0 is lossless (L223): integer sums, exact
        assert (d_nv[q] == 0).all()
        assert abs(e_fa[q].sum() - vol) <= 1e-9 * vol                      # L251
        if quant_bits == 0:                                                # exact ratios, but stored as fp32 weights
            np.testing.assert_allclose(e_fa[q], truth, rtol=0, atol=1e-6 * vol)
    lut.close()
    g.close()


def test_many_queries_and_buffer_regrowth(mg):
    """300 queries in one call after a 3-query call (the staging buffer grows), then a single big one
    (splits spread it over many CTAs)."""
    dims = (48, 40, 33)
    seg_index, gr, levels, g, d_idx, mip = _volume(mg, dims, 20, 43)
    nl = gr["n_leaves"]
    lut = g.mixture_lut(gr["weight_sigma"])
    for n in (3, 300, 1):
        boxes = _boxes(dims, n, 44 + n)[:n] if n > 1 else [[0, 0, 0, *dims]]
        e, d, f = _query(lut, d_idx, mip, boxes, nl, mg.MG_QUERY_NAIVE)
        for q, (x0, y0, z0, x1, y1, z1) in enumerate(boxes):
            truth = np.bincount(seg_index[z0:z1, y0:y1, x0:x1].reshape(-1), minlength=nl)
            np.testing.assert_array_equal(e[q], truth)
        e2, _, f2 = _query(lut, d_idx, mip, boxes, nl, mg.MG_QUERY_FA)
        np.testing.assert_allclose(e2.sum(axis=1), e.sum(axis=1), rtol=1e-12)
        assert (f2 <= f).all()
    lut.close()
    g.close()


def test_query_error_paths(mg):
    dims = (16, 16, 16)
    seg_index, gr, levels, g, d_idx, mip = _volume(mg, dims, 4, 45)
    nl = gr["n_leaves"]
    lut = g.mixture_lut(None)
    e = torch.zeros((1, nl), dtype=torch.float64, device="cuda")
    bad = [[0, 0, 0, 17, 16, 16], [4, 4, 4, 4, 8, 8], [5, 0, 0, 3, 1, 1]]
    for b in bad:
        with pytest.raises(mg.MgError) as ei:
            lut.range_query(d_idx, mip, [b], e)
        assert ei.value.code == mg.MG_ERR_INVALID_ARG
    with pytest.raises(mg.MgError):
        lut.range_query(d_idx, mip, [[0, 0, 0, 1, 1, 1]], e, mode=7)
    with pytest.raises(mg.MgError):
        lut.range_query(d_idx, (mip[0][:-1], mip[1][:-1]), [[0, 0, 0, 1, 1, 1]], e)      # pyramid cut below 1^3
    with pytest.raises(mg.MgError):
        lut.range_query(None, mip, [[0, 0, 0, 1, 1, 1]], e)
    with pytest.raises(ValueError):
        g.mixture_lut(np.zeros(3, np.float32))
    lut.range_query(d_idx, mip, [[0, 0, 0, 16, 16, 16]], e)                                # and the good call works
    torch.cuda.synchronize()
    assert abs(float(e.sum()) - 4096.0) < 1e-6
    lut.close()
    g.close()
