"""Host builder (a0-a2) checked against the oracle's DIRECT definitions (CPU only).

The builder's graph is not unique, so nothing here compares node lists with a stored
graph; the tests check what is unique: the mixtures it represents (I3, I4, I5), the validity of every
node (I2), the level structure (I9), the quantised error bound (I11, I12) and the paper's worked example.
"""
import numpy as np
import pytest

import oracle
from paper_2009_02702_b200 import builder, synth


def _voronoi(dims, n_seg, seed, zscale=1, jitter=0):
    seeds = synth.voronoi_seeds(dims, n_seg, seed)
    return synth.voronoi_volume(dims, seeds, zscale, jitter, seed)


def _check_structure(g, relabelled=True):
    a, b, w, off, nl = g["child_a"], g["child_b"], g["weight"], g["level_offsets"], g["n_leaves"]
    n = a.size
    idx = np.arange(n)
    internal = idx >= nl
    assert (a[internal] != b[internal]).all()                                  # I2
    assert (a[internal] < idx[internal]).all() and (b[internal] < idx[internal]).all()   # Eq. 8
    assert ((w[internal] > 0) & (w[internal] < 1)).all()                       # L176
    lev, depth = oracle.topo_levels(a, b, nl)                                  # I9
    assert off[0] == 0 and off[1] == nl and off[-1] == n and off.size == depth + 2
    if relabelled:
        for L in range(depth + 1):
            assert (lev[int(off[L]):int(off[L + 1])] == L).all()
    return depth


def test_fig2_worked_example_smallest_mass(golden_dir):
    """Fig. 2 (L103-L118): m = (0.1,0.2,0.3,0.4) -> (1,2,w=2/3), (3,5,w=1/2), (4,6,w=3/5) (1-based)."""
    r = builder.build_from_mixtures(4, [[(0, 1), (1, 2), (2, 3), (3, 4)]], quant_bits=0,
                                    pick_order=builder.PICK_SMALLEST_MASS, relabel=0)
    g = r.graph()
    assert r.info.n_nodes == 7
    assert list(zip(g["child_a"][4:], g["child_b"][4:])) == [(0, 1), (2, 4), (3, 5)]
    assert np.allclose(g["weight_exact"][4:], [2 / 3, 1 / 2, 3 / 5], rtol=0, atol=1e-15)
    assert r.node_idx(0).reshape(-1)[0] == 6
    mu = oracle.symbolic_eval(g["child_a"], g["child_b"], g["weight_exact"], 4)
    assert np.allclose(mu[6], [0.1, 0.2, 0.3, 0.4], rtol=0, atol=1e-15)


def test_fig4_node_reuse():
    """Fig. 4 (L172): m' = (0.2,0.4,0.1,0.3) re-uses lambda_5 (ratio 1:2) of m = (0.1,0.2,0.3,0.4)."""
    r = builder.build_from_mixtures(4, [[(0, 1), (1, 2), (2, 3), (3, 4)], [(0, 2), (1, 4), (2, 1), (3, 3)]],
                                    quant_bits=0, pick_order=builder.PICK_SMALLEST_MASS, relabel=0)
    g = r.graph()
    pairs = list(zip(g["child_a"][4:].tolist(), g["child_b"][4:].tolist()))
    assert pairs.count((0, 1)) == 1                      # ONE node mixes e1:e2 = 1:2, shared by both
    assert r.info.n_nodes < 4 + 6                        # fewer than two independent trees
    mu = oracle.symbolic_eval(g["child_a"], g["child_b"], g["weight_exact"], 4)
    idx = r.node_idx(0).reshape(-1)
    assert np.allclose(mu[idx[0]], [0.1, 0.2, 0.3, 0.4], atol=1e-15)
    assert np.allclose(mu[idx[1]], [0.2, 0.4, 0.1, 0.3], atol=1e-15)


def test_duplicate_and_pure_mixtures():
    r = builder.build_from_mixtures(3, [[(1, 5)], [(0, 2), (2, 2)], [(0, 7), (2, 7)], [(2, 1)]], quant_bits=0)
    idx = r.node_idx(0).reshape(-1)
    assert idx[0] == 1 and idx[3] == 2 and idx[1] == idx[2] == 3 and r.info.n_nodes == 4
    assert r.info.n_distinct_mixtures == 1


@pytest.mark.parametrize("dims,n_seg,pick", [((32, 32, 32), 16, 0), ((37, 29, 23), 12, 0), ((37, 29, 23), 12, 1),
                                             ((40, 24, 9), 40, 0)])
def test_unquantised_graph_reproduces_direct_histogram(dims, n_seg, pick):
    """I4: with exact ratios, mu[node_idx(v)] == H(v) and C_graph == C_dir for EVERY voxel of every
    level, power-of-two and ragged dims (L88 "always possible"); I5 level 0 is the leaf of S(v)."""
    S = _voronoi(dims, n_seg, seed=7)
    ids, seg_index = oracle.leaf_index(S)
    r = builder.build(S, quant_bits=0, pick_order=pick)
    g = r.graph()
    assert np.array_equal(g["leaf_segment_id"], ids)
    _check_structure(g)
    assert r.mip_dims == oracle.mip_dims(dims)
    H = oracle.histogram_mipmap(seg_index, ids.size)
    mu = oracle.symbolic_eval(g["child_a"], g["child_b"], g["weight_exact"], ids.size)
    assert np.abs(mu.sum(axis=1) - 1).max() < 1e-12 and mu.min() >= 0          # I3
    tf = synth.random_tf(ids.size, 3).astype(np.float64)
    c = oracle.graph_eval(g["child_a"], g["child_b"], g["weight_exact"], ids.size, tf)
    nnz = 0
    for l, counts in enumerate(H):
        idx = r.node_idx(l)
        h = counts.astype(np.float64) / 8.0 ** l
        assert np.abs(mu[idx] - h).max() < 1e-12
        assert np.abs(c[idx] - oracle.direct_colour(counts, l, tf)).max() < 1e-12
        nnz += int((counts != 0).sum())
    assert np.array_equal(r.node_idx(0), seg_index)                              # I5
    assert r.info.nnz_total == nnz
    assert r.info.n_voxels_total == sum(x * y * z for x, y, z in r.mip_dims)


@pytest.mark.parametrize("bits", [6, 9, 12])
def test_quantised_graph_error_bound_and_codebook(bits):
    """I11/I12: |C_graph - C_dir| <= 1/2 ||mu - H||_1 (max TF - min TF); the error shrinks with b
    (Table 3 trend, L361); level 0 stays lossless (L223); codewords lie inside their bins."""
    dims, n_seg = (48, 40, 33), 30
    S = _voronoi(dims, n_seg, seed=11)
    ids, seg_index = oracle.leaf_index(S)
    r = builder.build(S, quant_bits=bits)
    g = r.graph()
    _check_structure(g)
    H = oracle.histogram_mipmap(seg_index, ids.size)
    mu = oracle.symbolic_eval(g["child_a"], g["child_b"], g["weight"].astype(np.float64), ids.size)
    assert np.abs(mu.sum(axis=1) - 1).max() < 1e-12 and mu.min() >= 0
    tf = synth.random_tf(ids.size, 5).astype(np.float64)
    c = oracle.graph_eval(g["child_a"], g["child_b"], g["weight"], ids.size, tf)
    worst_l1, worst_c = 0.0, 0.0
    for l, counts in enumerate(H):
        idx = r.node_idx(l)
        l1 = np.abs(mu[idx] - counts.astype(np.float64) / 8.0 ** l).sum(axis=-1)
        dc = np.abs(c[idx] - oracle.direct_colour(counts, l, tf)).max(axis=-1)
        assert (dc <= 0.5 * l1 * (tf.max() - tf.min()) + 1e-12).all()
        worst_l1, worst_c = max(worst_l1, l1.max()), max(worst_c, dc.max())
    assert np.array_equal(r.node_idx(0), seg_index)
    # every lerp is off by < one bin width 2^-b; a path has at most `depth` of them
    assert worst_l1 <= 2.0 * r.info.depth * 2.0 ** -bits
    assert worst_c <= {6: 2e-2, 9: 2e-3, 12: 3e-4}[bits]
    cw, sg, cnt = r.codebook()
    nb = 1 << bits
    k = np.arange(nb)
    assert ((cw >= k / nb) & (cw <= (k + 1) / nb)).all() and (cw > 0).all() and (cw < 1).all()
    assert cnt.sum() > 0 and (sg <= 1.0 / nb).all()
    assert r.info.max_bin_sigma == pytest.approx(float(sg.max()))


def test_quantisation_merges_nodes_and_is_monotone():
    S = _voronoi((40, 40, 40), 60, seed=13)
    n = [builder.build(S, quant_bits=b).info.n_nodes for b in (0, 12, 6, 2)]
    assert n[0] >= n[1] >= n[2] >= n[3] and n[3] < n[0]


def test_relabel_off_gives_creation_order_and_same_values():
    S = _voronoi((24, 20, 17), 9, seed=5)
    r0, r1 = builder.build(S, quant_bits=9, relabel=0), builder.build(S, quant_bits=9, relabel=1)
    g0, g1 = r0.graph(), r1.graph()
    _check_structure(g0, relabelled=False)
    _check_structure(g1)
    tf = synth.random_tf(g0["n_leaves"], 1).astype(np.float64)
    c0 = oracle.graph_eval(g0["child_a"], g0["child_b"], g0["weight"], g0["n_leaves"], tf)
    c1 = oracle.graph_eval(g1["child_a"], g1["child_b"], g1["weight"], g1["n_leaves"], tf)
    for l in range(r0.info.n_mip_levels):
        assert np.array_equal(c0[r0.node_idx(l)], c1[r1.node_idx(l)])


def test_depth_is_logarithmic_and_levels_shrink():
    """Table 2 (L307): depth ~ log2(#segments), not chain-like; L213: many more nodes at small levels."""
    S = _voronoi((48, 48, 48), 150, seed=17)
    r = builder.build(S, quant_bits=9)
    off = r.graph()["level_offsets"].astype(np.int64)
    sizes = np.diff(off)
    assert r.info.depth <= 2 * int(np.ceil(np.log2(150))) + 2
    assert sizes[1] > sizes[-1] * 10 and sizes[1:4].sum() > 0.8 * sizes[1:].sum()


def test_sparse_ids_background_and_single_segment():
    S = np.zeros((5, 6, 7), dtype=np.uint32)
    r = builder.build(S)
    assert r.info.n_nodes == 1 and r.info.n_leaves == 1 and r.info.depth == 0
    assert all((r.node_idx(l) == 0).all() for l in range(r.info.n_mip_levels))
    S[2:, :, :] = 4000000000
    S[0, 0, 0] = 17
    r = builder.build(S, quant_bits=0)
    g = r.graph()
    assert g["leaf_segment_id"].tolist() == [0, 17, 4000000000]
    mu = oracle.symbolic_eval(g["child_a"], g["child_b"], g["weight_exact"], 3)
    ids, seg_index = oracle.leaf_index(S)
    H = oracle.histogram_mipmap(seg_index, 3)
    for l, counts in enumerate(H):
        assert np.abs(mu[r.node_idx(l)] - counts / 8.0 ** l).max() < 1e-12


def test_deterministic_across_thread_counts():
    S = _voronoi((40, 36, 30), 25, seed=19)
    r1, r8 = builder.build(S, quant_bits=9, n_threads=1), builder.build(S, quant_bits=9, n_threads=8)
    g1, g8 = r1.graph(), r8.graph()
    for k in ("child_a", "child_b", "weight", "level_offsets"):
        assert np.array_equal(g1[k], g8[k])
    for l in range(r1.info.n_mip_levels):
        assert np.array_equal(r1.node_idx(l), r8.node_idx(l))


def test_error_paths():
    with pytest.raises(builder.BuilderError):
        builder.build(np.zeros((2, 2, 2), np.uint32), quant_bits=17)
    with pytest.raises(builder.BuilderError):
        builder.build_from_mixtures(2, [[(1, 1), (0, 1)]])          # leaves not increasing
    with pytest.raises(builder.BuilderError):
        builder.build_from_mixtures(2, [[(0, 1), (5, 1)]])          # leaf out of range
    for name in builder.SYMBOLS:
        getattr(builder.lib, name)


def _front_end_numpy(seg):
    """Plain numpy statement of what the device front end computes (levels 0 and 1 of Eq. 4, pure / not pure):
    leaf numbers of level 0; per level-1 parent the leaf of its existing children if they agree, else 0xFFFFFFFF
    plus the list (voxel, 8 children with 0xFFFFFFFF for children outside the volume)."""
    ids, l0 = oracle.leaf_index(seg)
    Z, Y, X = l0.shape
    pz, py, px = -(-Z // 2), -(-Y // 2), -(-X // 2)
    pad = np.full((2 * pz, 2 * py, 2 * px), 0xFFFFFFFF, dtype=np.uint32)
    pad[:Z, :Y, :X] = l0
    ch = pad.reshape(pz, 2, py, 2, px, 2).transpose(0, 2, 4, 1, 3, 5).reshape(pz, py, px, 8)
    exists = ch != 0xFFFFFFFF
    first = ch[..., 0]                                              # child (0,0,0) always exists
    pure = ((ch == first[..., None]) | ~exists).all(axis=-1)
    level1 = np.where(pure, first, 0xFFFFFFFF).astype(np.uint32)
    mixed = np.flatnonzero(~pure.reshape(-1)).astype(np.uint32)
    return ids, l0, level1, mixed, ch.reshape(-1, 8)[mixed]


@pytest.mark.parametrize("dims,n_seg,bits", [((32, 32, 32), 9, 9), ((37, 29, 23), 12, 9), ((5, 1, 9), 4, 0), ((2, 2, 2), 3, 9)])
def test_build_from_level1_is_identical_to_build(dims, n_seg, bits):
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, n_seg, 61))
    ids, l0, level1, mixed, children = _front_end_numpy(seg)
    rng_order = np.argsort(synth.u64(61, 1, np.arange(mixed.size, dtype=np.uint64)))          # any order is allowed
    a = builder.build(seg, quant_bits=bits)
    b = builder.build_from_level1(dims, ids, level1, mixed[rng_order], children[rng_order], quant_bits=bits)
    ga, gb = a.graph(), b.graph()
    for k in ("child_a", "child_b", "weight", "weight_exact", "weight_sigma", "level_offsets", "leaf_segment_id"):
        assert np.array_equal(ga[k], gb[k]), k
    assert a.mip_dims == b.mip_dims
    for f in ("n_nodes", "n_leaves", "depth", "n_mip_levels", "n_voxels_total", "n_distinct_mixtures", "nnz_total"):
        assert getattr(a.info, f) == getattr(b.info, f), f
    assert np.array_equal(a.node_idx(0), l0)                      # level 0 IS the leaf number (what the caller keeps)
    with pytest.raises(builder.BuilderError):
        b.node_idx(0)
    for l in range(1, a.info.n_mip_levels):
        assert np.array_equal(a.node_idx(l), b.node_idx(l)), l


def test_build_from_level1_rejects_inconsistent_input():
    dims = (8, 8, 8)
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, 5, 62))
    ids, l0, level1, mixed, children = _front_end_numpy(seg)
    assert mixed.size > 2
    with pytest.raises(builder.BuilderError):                                    # a mixed parent missing from the list
        builder.build_from_level1(dims, ids, level1, mixed[1:], children[1:])
    with pytest.raises(builder.BuilderError):                                    # the same parent twice
        builder.build_from_level1(dims, ids, level1, np.r_[mixed, mixed[:1]], np.r_[children, children[:1]])
    bad = children.copy()
    bad[0, 0] = ids.size                                                         # leaf out of range
    with pytest.raises(builder.BuilderError):
        builder.build_from_level1(dims, ids, level1, mixed, bad)
    with pytest.raises(builder.BuilderError):                                    # IDs not increasing
        builder.build_from_level1(dims, ids[::-1], level1, mixed, children)
    with pytest.raises(ValueError):
        builder.build_from_level1(dims, ids, level1[:-1], mixed, children)


def _levels_front_numpy(seg, level_done):
    """Plain numpy / oracle statement of what mg_mipmap_levels_build hands to the host: the distinct reduced mixtures of
    the levels 1 .. level_done (the oracle's exact integer histograms divided by their common power of two) in a
    scrambled order, each with its first occurrence level << 40 | voxel, the handles of every level and the non-zeros."""
    ids, l0 = oracle.leaf_index(seg)
    H = oracle.histogram_mipmap(l0, ids.size)
    table, first, handles, nnz = {}, [], [], 0
    for l in range(1, level_done + 1):
        flat = H[l].reshape(-1, ids.size)
        hl = np.zeros(flat.shape[0], dtype=np.uint32)
        for v, row in enumerate(flat):
            leaves = np.flatnonzero(row)
            nnz += leaves.size
            if leaves.size == 1:
                hl[v] = leaves[0]
                continue
            counts = row[leaves].astype(np.uint64)
            tz = min(int(c & -c).bit_length() - 1 for c in counts.tolist())
            key = (tuple(leaves.tolist()), tuple((counts >> np.uint64(tz)).tolist()), 3 * l - tz)
            if key not in table:
                table[key] = len(first)
                first.append((l << 40) | v)
            hl[v] = 0x80000000 | table[key]
        handles.append(hl)
    keys = list(table)
    order = np.argsort(synth.u64(63, 2, np.arange(len(keys), dtype=np.uint64)))      # creation order on the device is arbitrary
    new_of_old = np.empty(len(keys), dtype=np.int64)
    new_of_old[order] = np.arange(len(keys))
    mix = dict(offset=[], k=[], tlog=[], first_pos=[], leaf=[], count=[])
    for q in order:
        leaves, counts, tlog = keys[q]
        mix["offset"].append(len(mix["leaf"])); mix["k"].append(len(leaves)); mix["tlog"].append(tlog); mix["first_pos"].append(first[q])
        mix["leaf"] += leaves; mix["count"] += counts
    dt = dict(offset=np.uint64, k=np.uint32, tlog=np.uint32, first_pos=np.uint64, leaf=np.uint32, count=np.uint64)
    mix = {k: np.array(v, dtype=dt[k]) for k, v in mix.items()}
    for hl in handles:
        m = hl >= 0x80000000
        hl[m] = (0x80000000 | new_of_old[hl[m] & 0x7FFFFFFF]).astype(np.uint32)
    return ids, l0, handles, mix, nnz


@pytest.mark.parametrize("dims,n_seg,bits", [((16, 16, 16), 7, 9), ((13, 11, 9), 6, 9), ((5, 1, 9), 4, 0)])
def test_build_from_levels_is_identical_to_build(dims, n_seg, bits):
    """mgb_build_from_levels continues Eq. 4 above ANY finished level and reproduces mgb_build: same graph, same node of
    every listed mixture, same node indices from the finished level on."""
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, n_seg, 64))
    a = builder.build(seg, quant_bits=bits)
    ga = a.graph()
    n_lv = a.info.n_mip_levels
    for level_done in sorted({1, 2, n_lv - 1}):
        ids, l0, handles, mix, nnz = _levels_front_numpy(seg, level_done)
        b, nodes = builder.build_from_levels(dims, ids, level_done, handles[-1], mix, nnz, quant_bits=bits)
        gb = b.graph()
        for k in ("child_a", "child_b", "weight", "weight_exact", "weight_sigma", "level_offsets", "leaf_segment_id"):
            assert np.array_equal(ga[k], gb[k]), (level_done, k)
        for f in ("n_nodes", "n_leaves", "depth", "n_mip_levels", "n_voxels_total", "n_distinct_mixtures", "nnz_total"):
            assert getattr(a.info, f) == getattr(b.info, f), (level_done, f)
        for l in range(1, n_lv):
            want = a.node_idx(l).reshape(-1)
            if l < level_done:                                     # not stored: they follow from the caller's handles
                with pytest.raises(builder.BuilderError):
                    b.node_idx(l)
            else:
                assert np.array_equal(b.node_idx(l).reshape(-1), want), (level_done, l)
            if l <= level_done:
                h = handles[l - 1]
                got = np.where(h >= 0x80000000, nodes[h & 0x7FFFFFFF] if nodes.size else 0, h)
                assert np.array_equal(got, want), (level_done, l)
        b.close()
    a.close()


def test_build_from_levels_rejects_malformed_input():
    dims = (8, 8, 8)
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, 5, 65))
    ids, l0, handles, mix, nnz = _levels_front_numpy(seg, 1)
    assert mix["k"].size > 2
    bad = dict(mix, count=mix["count"] * np.uint64(2))                             # totals are no longer 2^tlog
    with pytest.raises(builder.BuilderError):
        builder.build_from_levels(dims, ids, 1, handles[0], bad, nnz)
    h = handles[0].copy()
    h[np.flatnonzero(h >= 0x80000000)[0]] = 0x80000000 | mix["k"].size              # names no listed mixture
    with pytest.raises(builder.BuilderError):
        builder.build_from_levels(dims, ids, 1, h, mix, nnz)
    with pytest.raises(builder.BuilderError):                                      # level_done beyond the chain
        builder.build_from_levels(dims, ids, 9, handles[0], mix, nnz)
    # corrupt descriptors must be refused before they size or shift anything
    def with_(key, q, value):
        m = {k: v.copy() for k, v in mix.items()}
        m[key][q] = value
        return m
    for bad in (with_("tlog", 1, 64), with_("tlog", 0, 0xFFFFFFFF),                # a shift by >= 64 bits
                with_("k", 1, 0xFFFFFFF0),                                         # 4 G entries for one mixture
                with_("offset", 2, mix["leaf"].size),                              # starts behind the entries
                with_("offset", 0, 2 ** 64 - 1),                                   # offset + k wraps around
                with_("k", 0, 1), with_("first_pos", 0, 5), with_("first_pos", 1, (2 << 40) | 1)):   # k < 2; level 0 / 2 of a level-1 front
        with pytest.raises(builder.BuilderError) as ei:
            builder.build_from_levels(dims, ids, 1, handles[0], bad, nnz)
        assert "malformed" in str(ei.value)
    b, _ = builder.build_from_levels(dims, ids, 1, handles[0], mix, nnz)           # (the untouched input is accepted)
    b.close()
