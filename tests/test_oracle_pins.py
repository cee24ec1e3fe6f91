"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

Every oracle function is tied to something other than itself: printed values (tests/golden/),
closed forms, hand-derived small cases, brute force, or a numpy library routine.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle
from paper_2009_02702_b200 import synth


# ------------------------------------------------------------------------------------------ O-1
def test_mip_dims_reproduce_table2(golden_dir):
    """Table 2 (L291-L293): voxel totals over all mip levels and the number of levels."""
    rows = [l.split() for l in open(os.path.join(golden_dir, "table2_mip.txt")) if l[0] != "#"]
    assert len(rows) == 3
    for name, X, Y, Z, printed, decimals, levels in rows:
        dims = oracle.mip_dims((int(X), int(Y), int(Z)))
        total = sum(x * y * z for x, y, z in dims)
        assert len(dims) == int(levels), name
        assert dims[-1] == (1, 1, 1)
        # the paper prints millions, truncated ("1,195" for 1,195.4) or to one decimal (404.7)
        q = 10 ** int(decimals)
        assert int(total / 1e6 * q) / q == float(printed), (name, total)


def test_mip_dims_small_cases():
    assert oracle.mip_dims((1, 1, 1)) == [(1, 1, 1)]
    d = oracle.mip_dims((64, 64, 64))
    assert len(d) == 7 and sum(x * y * z for x, y, z in d) == 299593
    assert oracle.mip_dims((5, 3, 2)) == [(5, 3, 2), (3, 2, 1), (2, 1, 1), (1, 1, 1)]


# ------------------------------------------------------------------------------------------ O-2/O-3
def _random_labels(shape_zyx, n_seg, seed):
    n = int(np.prod(shape_zyx))
    lab = (synth.u64(seed, 77, np.arange(n, dtype=np.uint64)) % np.uint64(n_seg)).astype(np.uint32)
    return lab.reshape(shape_zyx)


def test_hist_hand_derived_border_case():
    """Eq. 4 with N = number of existing children (L80; reading Q2), derived by hand for a
    3x1x1 volume with labels [0,1,2]: level 1 = {(1/2,1/2,0), (0,0,1)}, root = (1/4,1/4,1/2)
    -- NOT the finest-voxel average (1/3,1/3,1/3)."""
    S = np.array([[[0, 1, 2]]], dtype=np.uint32)
    H = oracle.histogram_mipmap(S, 3)
    assert [h.shape for h in H] == [(1, 1, 3, 3), (1, 1, 2, 3), (1, 1, 1, 3)]
    assert H[1][0, 0].tolist() == [[4, 4, 0], [0, 0, 8]]          # scaled to 8^1
    assert H[2][0, 0, 0].tolist() == [16, 16, 32]                # scaled to 8^2


def test_hist_counts_sum_to_8_pow_l_non_pow2():
    S = _random_labels((7, 9, 13), 5, 3)
    for l, h in enumerate(oracle.histogram_mipmap(S, 5)):
        assert (h.sum(axis=-1) == 8 ** l).all()


def test_hist_recursion_equals_brute_force_every_voxel():
    """O-2 (recursive, integer) against O-3 (unrolled Eq. 4, floating weights) on every voxel of
    every level of a non-power-of-two volume."""
    S = _random_labels((7, 9, 13), 5, 4)
    H = oracle.histogram_mipmap(S, 5)
    for l, h in enumerate(H):
        Z, Y, X, _ = h.shape
        for k in range(Z):
            for j in range(Y):
                for i in range(X):
                    bf = oracle.brute_force_histogram(S, 5, l, i, j, k)
                    np.testing.assert_allclose(h[k, j, i] / 8.0 ** l, bf, rtol=0, atol=1e-15)


def test_brute_force_weights_exact_fractions():
    """O-3's axis weights, re-derived with exact rationals in Python for one border voxel:
    5x1x1 volume, root (l = 3): sizes 5 -> 3 -> 2 -> 1."""
    S = np.array([[[0, 1, 2, 3, 4]]], dtype=np.uint32)
    # level1: [avg(0,1), avg(2,3), (4)] ; level2: [avg(l1_0,l1_1), l1_2] ; root: avg of both
    half = Fraction(1, 2)
    expect = [half * half * half] * 4 + [half]
    got = oracle.brute_force_histogram(S, 5, 3, 0, 0, 0)
    assert got.tolist() == [float(f) for f in expect]
    H = oracle.histogram_mipmap(S, 5)
    assert (H[3][0, 0, 0] / 8.0 ** 3).tolist() == [float(f) for f in expect]


def test_hist_pow2_is_textbook_box_filter_and_root_is_global_histogram():
    """Power-of-two volume: H(.,l) = box count / 8^l (numpy reshape-sum), and the 1^3 root is
    "the dense, normalized histogram of all segment IDs in the volume" (L86)."""
    n_seg = 6
    S = _random_labels((16, 16, 16), n_seg, 5)
    H = oracle.histogram_mipmap(S, n_seg)
    onehot = (S[..., None] == np.arange(n_seg)).astype(np.uint64)
    for l in range(5):
        b = 1 << l
        box = onehot.reshape(16 // b, b, 16 // b, b, 16 // b, b, n_seg).sum(axis=(1, 3, 5))
        assert (H[l] == box).all()                      # counts sum to 8^l = b^3: same scaling
    assert (H[4][0, 0, 0] == np.bincount(S.reshape(-1), minlength=n_seg)).all()


def test_brute_force_level_is_the_per_voxel_brute_force_and_the_box_filter():
    """brute_force_level (one pass over the finest voxels, all voxels of a level) against what fixes it: the per-voxel
    unrolled Eq. 4 and the integer recursion on a ragged volume; numpy's reshape-sum box count / 8^l on a
    power-of-two one; exact fractions on the 5x1x1 border case."""
    S = _random_labels((7, 9, 13), 5, 14)
    H = oracle.histogram_mipmap(S, 5)
    for l in range(len(H)):
        lvl = oracle.brute_force_level(S, 5, l)
        assert lvl.shape == H[l].shape
        np.testing.assert_allclose(lvl.sum(axis=-1), 1.0, rtol=0, atol=1e-15)
        np.testing.assert_allclose(lvl, H[l] / 8.0 ** l, rtol=0, atol=1e-15)
        Z, Y, X, _ = lvl.shape
        for (i, j, k) in {(0, 0, 0), (X - 1, Y - 1, Z - 1), (X // 2, Y - 1, 0), (X - 1, 0, Z // 2)}:
            np.testing.assert_allclose(lvl[k, j, i], oracle.brute_force_histogram(S, 5, l, i, j, k), rtol=0, atol=1e-16)
    n_seg = 6
    S = _random_labels((16, 16, 16), n_seg, 15)
    onehot = (S[..., None] == np.arange(n_seg)).astype(np.float64)
    for l in range(5):
        b = 1 << l
        box = onehot.reshape(16 // b, b, 16 // b, b, 16 // b, b, n_seg).sum(axis=(1, 3, 5))
        assert np.array_equal(oracle.brute_force_level(S, n_seg, l), box / b ** 3)
    S = np.array([[[0, 1, 2, 3, 4]]], dtype=np.uint32)
    assert oracle.brute_force_level(S, 5, 3)[0, 0, 0].tolist() == [0.125] * 4 + [0.5]
    assert oracle.brute_force_level(S, 5, 1)[0, 0].tolist() == [[.5, .5, 0, 0, 0], [0, 0, .5, .5, 0], [0, 0, 0, 0, 1]]


def test_direct_colour_level_is_the_scalar_product_with_the_histogram():
    """direct_colour_level (O-3c: the colour of every voxel of a level accumulated over its finest voxels, no histogram
    table) against what fixes it: <H, TF> with the recursion's exact integer histograms (O-2, Eq. 4) on a ragged
    7 x 9 x 13 volume, whole levels and z-slab by z-slab; numpy's box mean of TF[S] on a power-of-two volume; exact
    fractions on the 5 x 1 x 1 border case (N = 1 parents, Q2); level 0 is TF[S] itself."""
    S = _random_labels((7, 9, 13), 5, 14)
    tf = np.random.default_rng(3).random((5, 4))
    H = oracle.histogram_mipmap(S, 5)
    for l in range(len(H)):
        want = oracle.direct_colour(H[l], l, tf).reshape(H[l].shape[:3] + (4,))
        got = oracle.direct_colour_level(S, tf, l)
        assert got.shape == want.shape
        np.testing.assert_allclose(got, want, rtol=0, atol=1e-13)     # (up to 819 terms in another order)
        zl = want.shape[0]
        for k0, k1 in [(0, 1), (zl - 1, zl), (zl // 2, zl), (1, 1)]:
            if k0 <= k1 <= zl:
                np.testing.assert_array_equal(oracle.direct_colour_level(S, tf, l, k0, k1), got[k0:k1])
    assert np.array_equal(oracle.direct_colour_level(S, tf, 0), tf[S])
    S = _random_labels((16, 16, 16), 6, 15)
    tf = np.random.default_rng(4).random((6, 4))
    for l in range(5):
        b = 1 << l
        box = tf[S].reshape(16 // b, b, 16 // b, b, 16 // b, b, 4).mean(axis=(1, 3, 5))
        np.testing.assert_allclose(oracle.direct_colour_level(S, tf, l), box, rtol=0, atol=1e-15)
    S = np.array([[[0, 1, 2, 3, 4]]], dtype=np.uint32)
    tf = np.zeros((5, 4))
    tf[:, 0] = [1, 2, 4, 8, 16]
    tf[:, 3] = 1
    assert oracle.direct_colour_level(S, tf, 1)[0, 0, :, 0].tolist() == [1.5, 6.0, 16.0]          # (1+2)/2, (4+8)/2, 16
    assert oracle.direct_colour_level(S, tf, 2)[0, 0, :, 0].tolist() == [3.75, 16.0]              # (1.5+6)/2, 16
    assert oracle.direct_colour_level(S, tf, 3)[0, 0, 0].tolist() == [9.875, 0, 0, 1.0]           # (3.75+16)/2; alpha stays 1
    # a transposed axis or a dropped weight shows: anisotropic ragged volume, one voxel of another segment in a corner
    #   x axis 5 -> 3 -> 2 -> 1: voxel 4 is an only child twice (1, 1), then one of two (1/2)        -> 1/2
    #   y axis 2 -> 1 -> 1 -> 1: voxel 1 is one of two (1/2), then an only child twice                -> 1/2
    #   z axis 3 -> 2 -> 1 -> 1: voxel 2 is an only child (1), one of two (1/2), an only child (1)    -> 1/2
    S = np.zeros((3, 2, 5), dtype=np.uint32)
    S[2, 1, 4] = 1
    tf = np.array([[0, 0, 0, 0], [1, 0, 0, 0.]])
    top = oracle.direct_colour_level(S, tf, 3)
    assert top.shape == (1, 1, 1, 4) and top[0, 0, 0, 0] == 0.125
    assert oracle.direct_colour_level(S, tf, 1)[1, 0, :, 0].tolist() == [0.0, 0.0, 0.5]   # level 1 is 2 x 1 x 3: only y halves there


def test_level0_is_lossless_unit_vector():
    """L223: the finest level holds exactly one ID per voxel."""
    S = _random_labels((4, 5, 6), 7, 6)
    H0 = oracle.histogram_mipmap(S, 7)[0]
    assert (H0.argmax(-1) == S).all() and (H0.sum(-1) == 1).all()


def test_leaf_index_sparse_ids_background_is_a_segment():
    S = np.array([[[0, 40, 40], [7, 0, 1000000]]], dtype=np.uint32)
    ids, idx = oracle.leaf_index(S)
    assert ids.tolist() == [0, 7, 40, 1000000]
    assert idx.tolist() == [[[0, 2, 2], [1, 0, 3]]]


def test_direct_colour_matches_matmul_and_identity_tf():
    S = _random_labels((5, 6, 7), 4, 8)
    H = oracle.histogram_mipmap(S, 4)
    tf = synth.random_tf(4, 9).astype(np.float64)
    eye = np.eye(4)
    for l, h in enumerate(H):
        np.testing.assert_allclose(oracle.direct_colour(h, l, tf), (h / 8.0 ** l) @ tf, rtol=0, atol=1e-15)
        # TF = unit vectors -> the colour IS the histogram (RGBA <- segments 0..3)
        assert (oracle.direct_colour(h, l, eye) == h / 8.0 ** l).all()


# ------------------------------------------------------------------------------------------ O-4
def _load_fig2(golden_dir):
    nodes, mix = {}, {}
    for line in open(os.path.join(golden_dir, "fig2_factorisation.txt")):
        t = line.split()
        if not t or t[0].startswith("#"):
            continue
        if t[0] in ("m", "mprime"):
            mix[t[0]] = [float(v) for v in t[1:]]
        else:
            nodes[int(t[0])] = (int(t[1]), int(t[2]), Fraction(int(t[3]), int(t[4])))
    return nodes, mix


def _graph_from_fig(nodes, last):
    """0-based SoA arrays for leaves 1..4 and nodes 5..last of the figure (1-based in the paper)."""
    a = np.zeros(last, dtype=np.uint32)
    b = np.zeros(last, dtype=np.uint32)
    w = np.zeros(last, dtype=np.float64)
    for n in range(5, last + 1):
        i, j, f = nodes[n]
        a[n - 1], b[n - 1], w[n - 1] = i - 1, j - 1, float(f)
    return a, b, w


def test_fig2_worked_example(golden_dir):
    """Fig. 2 (L103-L118): root lambda_7 must reproduce m = (0.1, 0.2, 0.3, 0.4) -- on colours
    (O-4) and symbolically (O-5); intermediate lambdas as printed."""
    nodes, mix = _load_fig2(golden_dir)
    a, b, w = _graph_from_fig(nodes, 7)
    tf = synth.random_tf(4, 11).astype(np.float64)
    c = oracle.graph_eval(a, b, w, 4, tf)
    np.testing.assert_allclose(c[6], np.array(mix["m"]) @ tf, rtol=0, atol=1e-15)
    mu = oracle.symbolic_eval(a, b, w, 4)
    np.testing.assert_allclose(mu[4], [1 / 3, 2 / 3, 0, 0], atol=1e-16)          # lambda_5
    np.testing.assert_allclose(mu[5], [1 / 6, 2 / 6, 1 / 2, 0], atol=1e-16)      # lambda_6 expanded
    np.testing.assert_allclose(mu[6], mix["m"], atol=1e-16)
    assert (c[:4] == tf).all()                                                   # I1


def test_fig4_node_reuse(golden_dir):
    """Fig. 4 (L172, L144): m' = (0.2, 0.4, 0.1, 0.3) re-uses lambda_5 -- a DAG with a shared node."""
    nodes, mix = _load_fig2(golden_dir)
    a, b, w = _graph_from_fig(nodes, 9)
    mu = oracle.symbolic_eval(a, b, w, 4)
    np.testing.assert_allclose(mu[6], mix["m"], atol=1e-16)
    np.testing.assert_allclose(mu[8], mix["mprime"], atol=1e-16)
    tf = synth.random_tf(4, 12).astype(np.float64)
    c = oracle.graph_eval(a, b, w, 4, tf)
    np.testing.assert_allclose(c[8], np.array(mix["mprime"]) @ tf, rtol=0, atol=1e-15)


def test_weight_multiplies_second_child():
    """L259: (i, j, w) = (1 - w) s_i + w s_j."""
    a = np.array([0, 0, 0], dtype=np.uint32)
    b = np.array([0, 0, 1], dtype=np.uint32)
    w = np.array([0, 0, 0.25])
    tf = np.array([[1.0, 0, 0, 8], [0, 1.0, 0, 16]])
    c = oracle.graph_eval(a, b, w, 2, tf)
    assert c[2].tolist() == [0.75, 0.25, 0.0, 10.0]


def test_chain_closed_form():
    """Chain n_k = lerp(n_{k-1}, leaf1, w): c_k = (1-w)^k T0 + (1 - (1-w)^k) T1 (geometric series)."""
    K, wv = 40, 0.3
    a = np.zeros(K + 2, dtype=np.uint32)
    b = np.zeros(K + 2, dtype=np.uint32)
    w = np.zeros(K + 2)
    for k in range(1, K + 1):
        n = k + 1
        a[n] = 0 if k == 1 else n - 1
        b[n] = 1
        w[n] = wv
    tf = np.array([[0.2, 0.9, 0.5, 1.0], [0.7, 0.1, 0.5, 0.0]])
    c = oracle.graph_eval(a, b, w, 2, tf)
    for k in (1, 2, 17, K):
        g = (1 - wv) ** k
        np.testing.assert_allclose(c[k + 1], g * tf[0] + (1 - g) * tf[1], rtol=0, atol=1e-15)
    lev, depth = oracle.topo_levels(a, b, 2)
    assert depth == K and lev[-1] == K


def _small_dag(seed=21, n_nodes=3000, n_levels=9, n_leaves=37):
    a, b, w, off = synth.random_dag(n_nodes, n_levels, n_leaves, seed)
    return a, b, w, off, n_leaves


def test_symbolic_eval_ties_graph_eval_to_matmul():
    """O-5 vs O-4: c[n] == mu[n] . TF (numpy matmul); I3: rows of mu are mixtures."""
    a, b, w, off, nl = _small_dag()
    tf = synth.random_tf(nl, 22).astype(np.float64)
    c = oracle.graph_eval(a, b, w, nl, tf)
    mu = oracle.symbolic_eval(a, b, w, nl)
    np.testing.assert_allclose(mu.sum(axis=1), 1.0, rtol=0, atol=1e-12)
    assert (mu >= 0).all()
    np.testing.assert_allclose(c, mu @ tf, rtol=0, atol=1e-13)


def test_symbolic_eval_sparse_fig2_fig4_and_dense(golden_dir):
    """The sparse level-by-level O-5 (used on full-size graphs) reproduces Fig. 2 / Fig. 4's printed mixtures, equals
    the dense node-by-node table on a random DAG with shared nodes, and mu . TF is the O-4 colour."""
    nodes, mix = _load_fig2(golden_dir)
    a, b, w = _graph_from_fig(nodes, 9)
    mu = oracle.symbolic_eval_sparse(a, b, w, 4).toarray()
    np.testing.assert_allclose(mu[4], [1 / 3, 2 / 3, 0, 0], atol=1e-16)
    np.testing.assert_allclose(mu[6], mix["m"], atol=1e-16)
    np.testing.assert_allclose(mu[8], mix["mprime"], atol=1e-16)
    a, b, w, off, nl = _small_dag(seed=23)
    sp_mu = oracle.symbolic_eval_sparse(a, b, w, nl)
    assert sp_mu.shape == (a.size, nl)
    np.testing.assert_allclose(sp_mu.toarray(), oracle.symbolic_eval(a, b, w, nl), rtol=0, atol=1e-15)
    tf = synth.random_tf(nl, 24).astype(np.float64)
    np.testing.assert_allclose(sp_mu @ tf, oracle.graph_eval(a, b, w, nl, tf), rtol=0, atol=1e-13)
    np.testing.assert_allclose(np.asarray(sp_mu.sum(axis=1)).reshape(-1), 1.0, rtol=0, atol=1e-12)


def test_constant_tf_and_linearity():
    """I6 (convexity) and I7 (Eq. 5-7 are linear)."""
    a, b, w, off, nl = _small_dag(seed=23)
    const = np.tile(np.array([0.25, 0.5, 0.75, 1.0]), (nl, 1))
    np.testing.assert_allclose(oracle.graph_eval(a, b, w, nl, const), np.tile(const[0], (a.size, 1)),
                               rtol=0, atol=1e-15)
    t1 = synth.random_tf(nl, 24).astype(np.float64)
    t2 = synth.random_tf(nl, 25).astype(np.float64)
    lhs = oracle.graph_eval(a, b, w, nl, 0.3 * t1 - 1.7 * t2)
    rhs = 0.3 * oracle.graph_eval(a, b, w, nl, t1) - 1.7 * oracle.graph_eval(a, b, w, nl, t2)
    np.testing.assert_allclose(lhs, rhs, rtol=0, atol=1e-13)


def test_graph_eval_attr_fig2_chain_and_matmul(golden_dir):
    """NEXT-1 (L269 "any kind of numeric segmentation attribute", L271, L277): for every channel
    count the root of Fig. 2 is m . attr, a chain follows the geometric closed form, and on a random
    DAG the result is the numpy matmul mu @ attr with mu from the (separately pinned) symbolic
    evaluation -- a transposed operand, a dropped (1 - w) or a wrong channel stride fails one."""
    nodes, mix = _load_fig2(golden_dir)
    a, b, w = _graph_from_fig(nodes, 7)
    for n_ch in (1, 2, 3, 4, 7, 16):
        attr = (synth.uniform01(31, n_ch, np.arange(4 * n_ch, dtype=np.uint64)).reshape(4, n_ch) * 3.0 - 1.0)
        c = oracle.graph_eval_attr(a, b, w, 4, attr)
        assert c.shape == (7, n_ch) and (c[:4] == attr).all()
        np.testing.assert_allclose(c[6], np.array(mix["m"]) @ attr, rtol=0, atol=1e-15)
    # chain closed form, 5 channels with distinct values per channel
    K, wv = 25, 0.125
    ca = np.zeros(K + 2, dtype=np.uint32); cb = np.zeros(K + 2, dtype=np.uint32); cw = np.zeros(K + 2)
    for k in range(1, K + 1):
        ca[k + 1], cb[k + 1], cw[k + 1] = (0 if k == 1 else k), 1, wv
    attr = np.array([[1.0, -2.0, 0.5, 8.0, 0.0], [0.0, 4.0, 0.25, -8.0, 1.0]])
    c = oracle.graph_eval_attr(ca, cb, cw, 2, attr)
    for k in (1, 3, K):
        g = (1 - wv) ** k
        np.testing.assert_allclose(c[k + 1], g * attr[0] + (1 - g) * attr[1], rtol=0, atol=1e-14)
    # random DAG: library matmul with the mixture lookup table
    a, b, w, off, nl = _small_dag(seed=26)
    mu = oracle.symbolic_eval(a, b, w, nl)
    for n_ch in (1, 6):
        attr = synth.uniform01(32, n_ch, np.arange(nl * n_ch, dtype=np.uint64)).reshape(nl, n_ch)
        np.testing.assert_allclose(oracle.graph_eval_attr(a, b, w, nl, attr), mu @ attr, rtol=0, atol=1e-13)


def test_topo_levels_definition():
    """L211: sources 0, node = max(v1, v2) + 1; Fig. 2 graph has levels 1, 2, 3."""
    a = np.array([0, 0, 0, 0, 0, 2, 3], dtype=np.uint32)
    b = np.array([0, 0, 0, 0, 1, 4, 5], dtype=np.uint32)
    lev, depth = oracle.topo_levels(a, b, 4)
    assert lev.tolist() == [0, 0, 0, 0, 1, 2, 3] and depth == 3
    # a node whose children are a leaf and a deep node sits one above the DEEPER one (max, Q9)
    a2 = np.array([0, 0, 0, 2, 0], dtype=np.uint32)
    b2 = np.array([0, 0, 1, 1, 3], dtype=np.uint32)
    assert oracle.topo_levels(a2, b2, 2)[0].tolist() == [0, 0, 1, 2, 3]
    # synthetic DAG: child_a in level L-1 makes the level exactly L
    ra, rb, rw, off, nl = _small_dag(seed=26)
    lev, depth = oracle.topo_levels(ra, rb, nl)
    assert depth == len(off) - 2
    for L in range(len(off) - 1):
        assert (lev[int(off[L]):int(off[L + 1])] == L).all()
    with pytest.raises(ValueError):
        oracle.topo_levels(np.array([0, 2, 0], dtype=np.uint32), np.array([0, 0, 0], dtype=np.uint32), 1)


def test_level_synchronous_eval_is_bit_identical_to_index_order():
    a, b, w, off, nl = _small_dag(seed=27, n_nodes=20000, n_levels=12, n_leaves=100)
    # shuffle-free check on a graph whose index order is NOT level order: append cross-level nodes
    tf = synth.random_tf(nl, 28).astype(np.float64)
    ref = oracle.graph_eval(a, b, w, nl, tf)
    for threads in (1, 3):
        got, used = oracle.graph_eval_levels(a, b, w, nl, tf, n_threads=threads)
        assert used == threads
        assert (got == ref).all()


def test_lookup_is_fancy_indexing():
    c = synth.random_tf(50, 30).astype(np.float64)
    idx = (synth.u64(31, 0, np.arange(4 * 5 * 6, dtype=np.uint64)) % np.uint64(50)).astype(np.uint32).reshape(4, 5, 6)
    assert (oracle.lookup(idx, c) == c[idx]).all()


# ------------------------------------------------------------------------------------------ Q13
def test_rgba8_known_values_round_half_even_and_clamp():
    # 0.5 * 255 = 127.5 -> 128 (even); 2.5/255 -> 2 (even) ; 3.5/255 -> 4
    vals = np.array([[0.0, 1.0, 0.5, -0.25], [1.5, 1 / 255, 254.4 / 255, 254.6 / 255],
                     [np.float32(2.5) / np.float32(255), np.float32(3.5) / np.float32(255), np.nan, 0.2]])
    out = oracle.to_rgba8(vals)
    assert out[0].tolist() == [0, 255, 128, 0]
    assert out[1].tolist() == [255, 1, 254, 255]
    p = (np.float32(np.float32(2.5) / np.float32(255)) * np.float32(255))
    assert out[2, 0] == int(np.rint(p)) and out[2, 2] == 0 and out[2, 3] == 51
    # exhaustive: every code k/255 maps back to k
    k = np.arange(256, dtype=np.float64)
    assert (oracle.to_rgba8((k / 255.0).reshape(64, 4)).reshape(-1) == k).all()
    c = oracle.colourise_rgba8(np.array([1, 0], dtype=np.uint32), vals[:2])[0]
    assert (c == out[[1, 0]]).all()


def test_rgba16f_is_round_to_nearest():
    v = np.array([[0.1, 1 / 3, 1.0, 65504.0]])
    assert (oracle.to_rgba16f(v) == v.astype(np.float16)).all()
    assert oracle.to_rgba16f(v).dtype == np.float16


# ------------------------------------------------------------------------------------------ NEXT-3
def _golden_packed(golden_dir):
    for line in open(os.path.join(golden_dir, "packed_bits.txt")):
        if line.startswith("#") or not line.strip():
            continue
        head, ids, hexbytes = [p.strip() for p in line.split("|")]
        i_min, r = (int(x) for x in head.split())
        yield i_min, r, [int(x) for x in ids.split()], bytes(int(x, 16) for x in hexbytes.split())


def test_pack_level_reproduces_hand_worked_streams(golden_dir):
    """Table 1 row (A) with the Q18 bit order: streams worked by hand (tests/golden/packed_bits.txt)."""
    n = 0
    for i_min, r, ids, stream in _golden_packed(golden_dir):
        got = oracle.pack_level(ids, i_min, r)
        assert got.tobytes() == stream[:got.size], (i_min, r, ids)
        assert all(b == 0 for b in stream[got.size:])
        assert oracle.unpack_level(np.frombuffer(stream, dtype=np.uint8) if stream else np.zeros(0, np.uint8),
                                   len(ids), i_min, r).tolist() == ids
        n += 1
    assert n == 4


def test_bits_per_voxel_is_the_minimal_sufficient_bitrate():
    """Eq. 16 (L205): r = ceil(log2(range)) <=> 2^r >= range > 2^(r-1); printed-size anchors."""
    assert oracle.bits_per_voxel(0, 1181) == 11          # 1,182 sources -> 11 bits (config 3, level 0)
    assert oracle.bits_per_voxel(0, 352) == 9            # 353 sources
    assert oracle.bits_per_voxel(0, 15917) == 14         # 15,918 leaves
    assert oracle.bits_per_voxel(7, 7) == 0 and oracle.bits_per_voxel(7, 8) == 1
    assert oracle.bits_per_voxel(0, 2 ** 32 - 1) == 32
    for rng in list(range(1, 70)) + [255, 256, 257, 2 ** 20, 2 ** 20 + 1, 2 ** 31, 2 ** 31 + 1]:
        for i_min in (0, 5, 1000):
            r = oracle.bits_per_voxel(i_min, i_min + rng - 1)
            assert 2 ** r >= rng and (r == 0 or 2 ** (r - 1) < rng)


@pytest.mark.parametrize("r", [0, 1, 3, 7, 8, 11, 13, 16, 21, 31, 32])
def test_pack_unpack_round_trip_and_numpy_bit_view(r):
    """Round trip, stream length ceil(n r / 8), and an independent decode through numpy's unpackbits."""
    n = 1013
    i_min = 12345 if r < 32 else 0
    span = np.uint64(1) << np.uint64(r)
    vals = (synth.u64(3, 70 + r, np.arange(n, dtype=np.uint64)) % span).astype(np.uint64)
    ids = (vals + np.uint64(i_min)).astype(np.uint32)
    stream = oracle.pack_level(ids, i_min, r)
    assert stream.size == (n * r + 7) // 8
    assert np.array_equal(oracle.unpack_level(stream, n, i_min, r), ids)
    if r:
        bits = np.unpackbits(stream, bitorder="little")[:n * r].reshape(n, r).astype(np.uint64)
        dec = (bits << np.arange(r, dtype=np.uint64)).sum(axis=1)
        assert np.array_equal(dec, vals)
    lo, hi = oracle.index_range(ids)
    assert lo == int(ids.min()) and hi == int(ids.max()) and oracle.bits_per_voxel(lo, hi) <= r
