"""NEXT-4 (second half): the device front end of the histogram mipmap (mg_mipmap_leaf_index,
mg_mipmap_front_level1) against the oracle's definitions, and the whole device-assisted assembly
(workload.from_volume_device) against the host builder: bit-exact, everything here is integer work."""
import numpy as np
import pytest

import oracle
from paper_2009_02702_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

NONE = 0xFFFFFFFF


@pytest.fixture(scope="module")
def libs():
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2009_02702_b200 import mg, workload
    torch.cuda.set_device(0)
    return mg, workload


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a).view(np.int32)).cuda()


def _front(mg, seg, capacity=None, in_place=False):
    Z, Y, X = seg.shape
    d_seg = _dev(seg)
    d_l0 = d_seg if in_place else torch.full_like(d_seg, -1)
    ids = mg.mipmap_leaf_index(d_seg, seg.size, d_l0)
    pz, py, px = -(-Z // 2), -(-Y // 2), -(-X // 2)
    n1 = pz * py * px
    cap = n1 if capacity is None else capacity
    d_l1 = torch.full((n1,), 7, dtype=torch.int32, device="cuda")
    mv = torch.full((max(cap, 1),), -1, dtype=torch.int32, device="cuda")
    mc = torch.full((max(cap, 1), 8), -1, dtype=torch.int32, device="cuda")
    n_mixed = mg.mipmap_front_level1(d_l0, (X, Y, Z), d_l1, mv, mc, cap)
    u = lambda t: t.cpu().numpy().view(np.uint32)
    return ids, u(d_l0).reshape(Z, Y, X), u(d_l1).reshape(pz, py, px), u(mv), u(mc), n_mixed


@pytest.mark.parametrize("dims,n_seg", [((32, 32, 32), 9), ((37, 29, 23), 12), ((5, 1, 9), 4), ((1, 1, 1), 1), ((2, 1, 1), 2),
                                        ((130, 67, 3), 40)])
def test_front_end_matches_the_definition(libs, dims, n_seg):
    mg, _ = libs
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, n_seg, 71)) * np.uint32(7) + np.uint32(3)    # sparse IDs (Q14)
    ids, l0, l1, mv, mc, n_mixed = _front(mg, seg)
    ref_ids, ref_l0 = oracle.leaf_index(seg)
    assert np.array_equal(ids, ref_ids) and np.array_equal(l0, ref_l0)
    # level 1 against the oracle's exact histograms (O-2): pure <=> one non-zero count
    H = oracle.histogram_mipmap(ref_l0, ref_ids.size)
    if len(H) > 1:
        h1 = H[1]
        nnz = (h1 != 0).sum(axis=-1)
        leaf = h1.argmax(axis=-1).astype(np.uint32)
        assert np.array_equal(l1 == NONE, nnz > 1)
        assert np.array_equal(l1[nnz == 1], leaf[nnz == 1])
        assert n_mixed == int((nnz > 1).sum())
        order = np.argsort(mv[:n_mixed])
        assert np.array_equal(mv[:n_mixed][order], np.flatnonzero((nnz > 1).reshape(-1)))        # each listed once
        Z, Y, X = seg.shape
        for q in order[:: max(1, n_mixed // 300)]:                                             # children of sampled parents
            v = int(mv[q])
            i, j, k = v % l1.shape[2], (v // l1.shape[2]) % l1.shape[1], v // (l1.shape[2] * l1.shape[1])
            for t in range(8):
                x, y, z = 2 * i + (t & 1), 2 * j + ((t >> 1) & 1), 2 * k + (t >> 2)
                want = ref_l0[z, y, x] if (x < X and y < Y and z < Z) else NONE
                assert mc[q, t] == want
    else:
        assert n_mixed == 0


def test_front_end_in_place_and_small_capacity(libs):
    mg, _ = libs
    dims = (37, 29, 23)
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, 12, 72))
    ids, l0, l1, mv, mc, n_mixed = _front(mg, seg)
    ids2, l0b, l1b, mv2, mc2, n2 = _front(mg, seg, capacity=5, in_place=True)                 # level0 written over seg
    assert np.array_equal(ids, ids2) and np.array_equal(l0, l0b) and np.array_equal(l1, l1b)
    assert n2 == n_mixed > 5                                                                   # the true count is reported
    assert set(mv2[:5].tolist()) <= set(mv[:n_mixed].tolist())
    with pytest.raises(mg.MgError):
        mg.mipmap_leaf_index(_dev(seg), seg.size, torch.zeros(seg.size, dtype=torch.int32, device="cuda"), capacity=3)
    big = seg.copy()
    big[0, 0, 0] = 1 << 28
    with pytest.raises(mg.MgError):
        mg.mipmap_leaf_index(_dev(big), big.size, torch.zeros(big.size, dtype=torch.int32, device="cuda"))


@pytest.mark.parametrize("dims", [(24, 10, 9), (23, 10, 9), (6, 1, 1)])
@pytest.mark.parametrize("off_in,off_out", [(0, 0), (1, 1), (2, 2), (3, 3), (1, 0), (0, 3), (2, 1)])
def test_front_end_at_any_alignment(libs, dims, off_in, off_out):
    """The kernels take 16-byte (leaf index) and 8-byte (level 1) loads where the pointers allow it: every offset of
    the volume and of level 0 from a 16-byte boundary, equal or not, even and odd X, gives the aligned result."""
    mg, _ = libs
    X, Y, Z = dims
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, min(11, X * Y * Z // 2), 73)) * np.uint32(5) + np.uint32(1)
    ref_ids, ref_l0 = oracle.leaf_index(seg)
    n = seg.size
    buf_in = torch.full((n + 8,), -1, dtype=torch.int32, device="cuda")
    buf_out = torch.full((n + 8,), -2, dtype=torch.int32, device="cuda")
    buf_in[off_in:off_in + n] = _dev(seg).reshape(-1)
    d_l0 = buf_out[off_out:off_out + n]
    ids = mg.mipmap_leaf_index(buf_in[off_in:off_in + n], n, d_l0)
    assert np.array_equal(ids, ref_ids)
    out = buf_out.cpu().numpy()
    assert np.array_equal(out[off_out:off_out + n].view(np.uint32), ref_l0.reshape(-1))
    assert (out[:off_out] == -2).all() and (out[off_out + n:] == -2).all()                    # nothing outside is written
    assert (buf_in.cpu().numpy()[:off_in] == -1).all()
    # level 1 from the (mis)aligned level 0 == level 1 from an aligned copy
    pz, py, px = -(-Z // 2), -(-Y // 2), -(-X // 2)
    n1 = pz * py * px
    res = []
    for l0 in (d_l0, d_l0.clone()):
        d_l1 = torch.full((n1,), 7, dtype=torch.int32, device="cuda")
        mv = torch.full((n1,), -1, dtype=torch.int32, device="cuda")
        mc = torch.full((n1, 8), -1, dtype=torch.int32, device="cuda")
        nm = mg.mipmap_front_level1(l0, (X, Y, Z), d_l1, mv, mc, n1)
        order = torch.argsort(mv[:nm])
        res.append((nm, d_l1.cpu(), mv[:nm][order].cpu(), mc[:nm][order].cpu()))
    assert res[0][0] == res[1][0] and all(torch.equal(a, b) for a, b in zip(res[0][1:], res[1][1:]))
    H = oracle.histogram_mipmap(ref_l0, ref_ids.size)
    if len(H) > 1:
        assert np.array_equal(res[0][1].numpy().view(np.uint32).reshape(pz, py, px) == NONE, (H[1] != 0).sum(axis=-1) > 1)


@pytest.mark.parametrize("cfg_id,scale", [(3, 0.08), (2, 0.06), (4, 0.12), (1, 1.0)])
def test_device_assisted_assembly_equals_the_host_builder(libs, cfg_id, scale):
    """workload.make(device_mipmap=True) vs the host path: same graph, same device mipmap, same stats."""
    mg, workload = libs
    a = workload.make(cfg_id, scale)
    b = workload.make(cfg_id, scale, device_mipmap=True)
    try:
        for k in ("child_a", "child_b", "weight", "weight_sigma", "level_offsets", "leaf_segment_id"):
            assert np.array_equal(a.host_graph[k], b.host_graph[k]), k
        assert a.mip_dims == b.mip_dims and a.level_start == b.level_start and a.n_voxels == b.n_voxels
        assert torch.equal(a.d_idx, b.d_idx)
        assert b.host_idx[0] is None and np.array_equal(b.host_level(0), a.host_level(0))
        for k in ("n_nodes", "depth", "n_distinct_mixtures"):
            assert a.stats[k] == b.stats[k], k
        assert abs(a.stats["nnz_per_voxel"] - b.stats["nnz_per_voxel"]) < 1e-15
    finally:
        a.close()
        b.close()


def _same_assembly(a, b):
    for k in ("child_a", "child_b", "weight", "weight_sigma", "level_offsets", "leaf_segment_id"):
        assert np.array_equal(a.host_graph[k], b.host_graph[k]), k
    assert a.mip_dims == b.mip_dims and a.level_start == b.level_start and a.n_voxels == b.n_voxels
    assert torch.equal(a.d_idx, b.d_idx)                              # the node index of every voxel of every level
    for k in ("n_nodes", "depth", "n_distinct_mixtures"):
        assert a.stats[k] == b.stats[k], k
    assert abs(a.stats["nnz_per_voxel"] - b.stats["nnz_per_voxel"]) < 1e-15


@pytest.mark.parametrize("cfg_id,scale", [(3, 0.08), (2, 0.06), (4, 0.12), (1, 1.0)])
def test_device_levels_assembly_equals_the_host_builder(libs, cfg_id, scale):
    """workload.make(device_mipmap="levels"): the levels >= 1 merged and hash-consed on the device
    (mg_mipmap_levels_build), the host continuing above (mgb_build_from_levels): same graph, same device mipmap."""
    mg, workload = libs
    a = workload.make(cfg_id, scale)
    b = workload.make(cfg_id, scale, device_mipmap="levels")
    try:
        _same_assembly(a, b)
        assert b.stats["device_levels_done"] >= 1 and b.host_idx[0] is None
        print(f"cfg{cfg_id} x{scale}: device built levels 1 .. {b.stats['device_levels_done']} of {len(b.mip_dims) - 1}, "
              f"{b.stats['n_device_mixtures']} of {b.stats['n_distinct_mixtures']} distinct mixtures")
    finally:
        a.close()
        b.close()


@pytest.mark.parametrize("dims,n_seg", [((24, 24, 24), 400), ((37, 29, 23), 12), ((9, 1, 5), 4), ((2, 2, 2), 3), ((64, 48, 3), 900)])
def test_device_levels_ragged_and_crowded_volumes(libs, dims, n_seg):
    """Ragged ceil-halving chains (N = 1, 2, 4 children at the borders, Q2) and label noise with hundreds of segments, where
    the mixtures outgrow the 256 entries a warp merges and the device hands the upper levels to the host early."""
    mg, workload = libs
    X, Y, Z = dims
    seg = (synth.u64(71, 3, np.arange(X * Y * Z, dtype=np.uint64)) % np.uint64(n_seg)).astype(np.uint32).reshape(Z, Y, X) * 3 + 5
    a = workload.from_volume(seg, name="noise")
    b = workload.from_volume_device_levels(_dev(seg).view(Z, Y, X), name="noise")
    try:
        _same_assembly(a, b)
        if n_seg >= 400:
            assert 1 <= b.stats["device_levels_done"] < len(b.mip_dims) - 1     # abandoned before the top
    finally:
        a.close()
        b.close()


@pytest.mark.parametrize("upsampled,cap,done", [(True, (100, 800), 1), (True, (0, 300), 1), (False, (64, 0), 0)])
def test_device_levels_store_overflow_goes_to_the_host(libs, upsampled, cap, done):
    """A level whose mixtures do not fit the device store is handed to the host with the levels above it, not reported as
    an error.  The case that reaches this with the default sizing is a nearest-neighbour 2x-upsampled volume: level 1 is
    pure throughout (no merge to size the stores from) and level 2 holds every merge; small explicit capacities
    (mg_mipmap_levels_build_ex) bring it to a size a test can afford -- too few mixtures, too few entries, and a noise
    volume whose level 1 already overflows (nothing built on the device).  Same graph and indices as the host builder."""
    mg, workload = libs
    n = 20
    small = (synth.u64(72, 3, np.arange(n ** 3, dtype=np.uint64)) % np.uint64(150)).astype(np.uint32).reshape(n, n, n) * 2 + 1
    seg = np.repeat(np.repeat(np.repeat(small, 2, 0), 2, 1), 2, 2) if upsampled else small
    if upsampled:
        ids, l0 = oracle.leaf_index(seg)
        H = oracle.histogram_mipmap(l0, ids.size)
        assert ((H[1] != 0).sum(axis=-1) == 1).all() and ((H[2] != 0).sum(axis=-1) > 1).mean() > 0.99
    a = workload.from_volume(seg, name="overflow")
    b = workload.from_volume_device_levels(_dev(seg).view(*seg.shape), name="overflow", store_capacity=cap)
    try:
        _same_assembly(a, b)
        assert b.stats.get("device_levels_done", 0) == done
    finally:
        a.close()
        b.close()


def test_mixture_table_matches_the_oracle_histograms(libs):
    """mg_mipmap_levels_build against the definition, not against the host builder: every handle of every finished level
    expands to the oracle's exact integer histogram of that voxel (Eq. 4, O-2) divided by its common power of two; equal
    mixtures share one number; first occurrences are the scanline minimum."""
    mg, workload = libs
    dims = (21, 18, 14)
    X, Y, Z = dims
    seg = synth.voronoi_volume(dims, synth.voronoi_seeds(dims, 9, 72))
    ids, l0 = oracle.leaf_index(seg)
    H = oracle.histogram_mipmap(l0, ids.size)
    sizes = [h.shape[0] * h.shape[1] * h.shape[2] for h in H]
    start = np.concatenate([[0], np.cumsum(sizes)[:-1]]).astype(np.uint64)
    buf = torch.zeros(int(sum(sizes)), dtype=torch.int32, device="cuda")
    buf[:sizes[0]] = _dev(l0.reshape(-1))
    t = mg.MixtureTable(buf, dims, ids.size, buf, start)
    assert t.info.levels_done == len(H) - 1 and t.info.n_leaves == ids.size
    m = t.export()
    hb = buf.cpu().numpy().view(np.uint32)
    seen, nnz = {}, 0
    for l in range(1, len(H)):
        flat = H[l].reshape(-1, ids.size)
        for v in range(flat.shape[0]):
            h = int(hb[int(start[l]) + v])
            leaves = np.flatnonzero(flat[v])
            nnz += leaves.size
            if leaves.size == 1:
                assert h == leaves[0]
                continue
            assert h & 0x80000000
            q = h & 0x7FFFFFFF
            o, k = int(m["offset"][q]), int(m["k"][q])
            counts = flat[v][leaves]
            tz = min(int(c & -c).bit_length() - 1 for c in counts.tolist())
            assert np.array_equal(m["leaf"][o:o + k], leaves) and np.array_equal(m["count"][o:o + k], counts >> np.uint64(tz))
            assert int(m["tlog"][q]) == 3 * l - tz
            seen.setdefault(q, (l << 40) | v)
    assert len(seen) == t.info.n_mixtures and nnz == t.info.nnz_levels
    for q, pos in seen.items():
        assert int(m["first_pos"][q]) == pos
    keys = {(tuple(m["leaf"][int(o):int(o) + int(k)]), tuple(m["count"][int(o):int(o) + int(k)])) for o, k in zip(m["offset"], m["k"])}
    assert len(keys) == t.info.n_mixtures                            # hash-consed: no mixture twice
    t.close()


def test_levels_build_error_paths(libs):
    mg, workload = libs
    l0 = _dev(np.zeros(8 * 8 * 8, np.uint32))
    buf = torch.zeros(8 * 8 * 8 + 64 + 8 + 1, dtype=torch.int32, device="cuda")
    start = np.array([0, 512, 576, 584], dtype=np.uint64)
    with pytest.raises(mg.MgError):                                   # 8^3 has 4 levels, not 3
        mg.MixtureTable(l0, (8, 8, 8), 1, buf, start[:3])
    with pytest.raises(mg.MgError):                                   # no leaves
        mg.MixtureTable(l0, (8, 8, 8), 0, buf, start)
    t = mg.MixtureTable(l0, (8, 8, 8), 1, buf, start)                 # one segment: every level pure, no mixture at all
    assert t.info.levels_done == 3 and t.info.n_mixtures == 0 and t.info.nnz_levels == 64 + 8 + 1
    assert not buf.cpu().numpy().any()
    assert all(v.size == 0 for v in t.export().values())
    t.close()
    # a pure 2 x 2 x 2 volume: two levels, so no level ever reads the device counters back -- the table is still empty
    buf2 = torch.full((8 + 1,), 5, dtype=torch.int32, device="cuda")
    t = mg.MixtureTable(l0, (2, 2, 2), 1, buf2, np.array([0, 8], dtype=np.uint64))
    assert t.info.levels_done == 1 and t.info.n_mixtures == 0 and t.info.n_entries == 0 and t.info.nnz_levels == 1
    assert int(buf2[8]) == 0 and all(v.size == 0 for v in t.export().values())
    t.close()
