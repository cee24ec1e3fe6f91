"""NEXT-3 parity: bit-packed node-ID volumes (Table 1 rows (8), (9), (A); Eq. 15-16) through the C ABI.

The device packer must produce the oracle's stream bit for bit; mg_colorize_packed must produce exactly
what the oracle's unpack + lookup + conversion gives (and what mg_colorize gives on the unpacked indices).
"""
import numpy as np
import pytest

import oracle
from paper_2009_02702_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mg():
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2009_02702_b200 import mg as _mg
    torch.cuda.set_device(0)
    return _mg


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _ids(n, i_min, span, seed):
    return ((synth.u64(seed, 80, np.arange(n, dtype=np.uint64)) % np.uint64(span)) + np.uint64(i_min)).astype(np.uint32)


@pytest.mark.parametrize("n,i_min,span", [(1, 5, 1), (7, 0, 2), (2049, 100, 1182), (100003, 0, 1 << 21), (4097, 3, (1 << 32) - 3),
                                          (65536, 0, 1 << 16), (999, 77, 1)])
def test_index_range_and_pack_match_oracle(mg, n, i_min, span):
    ids = _ids(n, i_min, span, 31)
    d = _dev(ids)
    lo, hi = mg.index_range(d, n)
    assert (lo, hi) == oracle.index_range(ids)
    r = mg.bits_per_voxel(lo, hi)
    assert r == oracle.bits_per_voxel(lo, hi)
    nbytes = mg.packed_stream_bytes(n, r)
    assert nbytes % 16 == 0 and nbytes >= (n * r + 7) // 8 + 16
    packed = torch.full((nbytes,), 0xEE, dtype=torch.uint8, device="cuda")
    mg.pack_indices(d, n, lo, r, packed)
    torch.cuda.synchronize()
    got = packed.cpu().numpy()
    ref = oracle.pack_level(ids, lo, r)
    assert np.array_equal(got[:ref.size], ref)                 # bit-exact stream
    assert not got[ref.size:].any()                            # zero padding, fully written
    assert np.array_equal(oracle.unpack_level(got, n, lo, r), ids)


@pytest.mark.parametrize("off", [0, 1, 2, 3])
@pytest.mark.parametrize("n", [1, 2, 3, 6, 9, 1000, 4099])
def test_index_range_and_pack_at_any_alignment(mg, off, n):
    """mg_index_range reads 16 bytes at a time between the 16-byte boundaries: the extremes placed in the first and the
    last element (the ones taken one by one) at every offset of the level from a boundary; the packer from the same view."""
    ids = _ids(n, 1000, 5000, 32 + off)
    for first, last in ((7, 900000), (900000, 7)):
        ids[0], ids[-1] = first, last
        if n == 1:
            first = last
        buf = torch.zeros(n + 8, dtype=torch.int32, device="cuda")                         # zeros outside: must not be read
        buf[off:off + n] = _dev(ids.view(np.int32))
        d = buf[off:off + n]
        lo, hi = mg.index_range(d, n)
        assert (lo, hi) == oracle.index_range(ids) == (min(first, last), max(first, last))
        r = mg.bits_per_voxel(lo, hi)
        packed = torch.zeros(mg.packed_stream_bytes(n, r), dtype=torch.uint8, device="cuda")
        mg.pack_indices(d, n, lo, r, packed)
        ref = oracle.pack_level(ids, lo, r)
        assert np.array_equal(packed.cpu().numpy()[:ref.size], ref)


def _graph(mg, sizes, seed):
    a, b, w, off = synth.random_dag_levels(sizes, seed=seed)
    tf = synth.random_tf(sizes[0], seed + 1)
    g = mg.Graph(a, b, w, sizes[0], level_offsets=off)
    nodes = torch.zeros((sum(sizes), 4), dtype=torch.float32, device="cuda")
    g.propagate(_dev(tf), nodes)
    torch.cuda.synchronize()
    ref_nodes = oracle.graph_eval(a, b, w, sizes[0], tf.astype(np.float64))
    return g, nodes, ref_nodes


@pytest.mark.parametrize("fmt_name", ["RGBA8", "RGBA16F", "BOTH"])
def test_colorize_packed_multi_level_matches_oracle_and_unpacked_path(mg, fmt_name):
    sizes = [353, 50001, 20002, 9003, 4001, 1200, 333, 77, 20, 6, 2, 1]
    g, nodes, ref_nodes = _graph(mg, sizes, 33)
    n_nodes = sum(sizes)
    # levels: (n voxels, i_min, span): leaf-only level (few bits), wide level, ragged tiny levels, r = 0 level
    spec = [(300007, 0, 353), (40001, 10, n_nodes - 10), (2048, 353, 50001), (2047, 5, 1 << 16), (5, 70000, 3), (1, 84998, 1), (3, 7, 1)]
    levels, streams, all_ids, pos, out_pos = [], [], [], 0, 0
    for k, (n, i_min, span) in enumerate(spec):
        ids = _ids(n, i_min, span, 40 + k)
        lo, hi = oracle.index_range(ids)
        r = oracle.bits_per_voxel(lo, hi)
        st = oracle.pack_level(ids, lo, r)
        nbytes = mg.packed_stream_bytes(n, r)
        buf = np.zeros(nbytes, dtype=np.uint8)
        buf[:st.size] = st
        levels.append(dict(n_voxels=n, out_offset=out_pos, byte_offset=pos, bits=r, i_min=lo))
        streams.append(buf)
        all_ids.append((out_pos, ids))
        pos += nbytes
        out_pos += -(-n // 64) * 64
    d_packed = _dev(np.concatenate(streams))
    out8 = torch.full((out_pos, 4), 7, dtype=torch.uint8, device="cuda")
    out16 = torch.full((out_pos, 4), 7, dtype=torch.float16, device="cuda")
    fmt = getattr(mg, "MG_" + fmt_name)
    if fmt_name == "RGBA8":
        g.colorize_packed(d_packed, levels, nodes, out8, fmt=fmt)
    elif fmt_name == "RGBA16F":
        g.colorize_packed(d_packed, levels, nodes, out16, fmt=fmt)
    else:
        g.colorize_packed(d_packed, levels, nodes, out8, out16, fmt=fmt)
    torch.cuda.synchronize()
    got8, got16 = out8.cpu().numpy(), out16.cpu().numpy()
    code8 = oracle.to_rgba8(ref_nodes)
    # the unpacked path on the same indices must agree bit for bit
    for (o, ids), lv in zip(all_ids, levels):
        n = ids.size
        ref8 = np.zeros((n, 4), np.uint8)
        u8 = torch.zeros((n, 4), dtype=torch.uint8, device="cuda")
        u16 = torch.zeros((n, 4), dtype=torch.float16, device="cuda")
        g.colorize(_dev(ids), n, nodes, u8, u16, fmt=mg.MG_BOTH)
        torch.cuda.synchronize()
        if fmt_name in ("RGBA8", "BOTH"):
            assert np.array_equal(got8[o:o + n], u8.cpu().numpy())
            diff = np.abs(got8[o:o + n].astype(np.int64) - code8[ids].astype(np.int64))
            assert diff.max() <= 1 and (diff != 0).mean() < 1e-3          # fp32 vs fp64 palette: rare +-1 at boundaries
            end = -(-n // 64) * 64
            assert (got8[o + n:o + end] == 7).all()                        # padding untouched
        if fmt_name in ("RGBA16F", "BOTH"):
            assert np.array_equal(got16[o:o + n].view(np.uint16), u16.cpu().numpy().view(np.uint16))
            ref16 = oracle.to_rgba16f(ref_nodes[ids])
            assert (np.abs(got16[o:o + n].view(np.int16).astype(np.int64) - ref16.view(np.int16).astype(np.int64)) <= 1).all()
        del ref8


def test_colorize_packed_error_paths(mg):
    g, nodes, _ = _graph(mg, [8, 100, 10], 35)
    d = torch.zeros(64, dtype=torch.uint8, device="cuda")
    out = torch.zeros((64, 4), dtype=torch.uint8, device="cuda")
    lv = [dict(n_voxels=4, out_offset=2, byte_offset=0, bits=3, i_min=0)]          # out_offset not a multiple of 4
    with pytest.raises(mg.MgError):
        g.colorize_packed(d, lv, nodes, out)
    lv = [dict(n_voxels=4, out_offset=0, byte_offset=0, bits=33, i_min=0)]
    with pytest.raises(mg.MgError):
        g.colorize_packed(d, lv, nodes, out)
    other = torch.rand_like(nodes)
    lv = [dict(n_voxels=4, out_offset=0, byte_offset=0, bits=3, i_min=0)]
    with pytest.raises(mg.MgError):                                                # not the propagated buffer: no reuse
        g.colorize_packed(d, lv, other, out, from_last_propagate=True)
    g.colorize_packed(d, lv, nodes, out, from_last_propagate=True)                 # valid: the palettes of mg_propagate
    torch.cuda.synchronize()
    first = out.cpu().numpy()[:4].copy()
    g.colorize_packed(d, lv, other, out)                                           # default: derived from what is passed
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy()[:4], oracle.to_rgba8(other.cpu().numpy().astype(np.float64))[[0, 0, 0, 0]])
    with pytest.raises(mg.MgError):                                                # ... after which reuse is refused
        g.colorize_packed(d, lv, nodes, out, from_last_propagate=True)
    g.colorize_packed(d, lv, nodes, out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy()[:4], first)
    lv = [dict(n_voxels=4, out_offset=0, byte_offset=0, bits=3, i_min=10 ** 6)]    # i_min beyond the graph
    with pytest.raises(mg.MgError):
        g.colorize_packed(d, lv, nodes, out)


def test_stale_index_range_cannot_corrupt_or_overrun(mg):
    """An (i_min, r) pair that does not cover the data (a stale mg_index_range result): the packer reduces the
    offending value modulo 2^r instead of spilling into its neighbours' bits, and the colouriser clamps unpacked
    indices to the last node instead of gathering out of bounds."""
    g, nodes, ref_nodes = _graph(mg, [8, 100, 10], 36)
    n_nodes = nodes.shape[0]
    ids = np.array([5, 6, 7, 5 + 8 + 3, 6, 5, 4, 7], dtype=np.uint32)             # one value >= i_min + 2^r, one < i_min
    i_min, r = 5, 2
    d = torch.zeros(mg.packed_stream_bytes(ids.size, r), dtype=torch.uint8, device="cuda")
    mg.pack_indices(_dev(ids), ids.size, i_min, r, d)
    torch.cuda.synchronize()
    want = ((ids.astype(np.int64) - i_min) % (1 << r)).astype(np.uint32)
    assert np.array_equal(d.cpu().numpy()[:2], oracle.pack_level(want + i_min, i_min, r)[:2])     # 8 values x 2 bits
    out = torch.zeros((8, 4), dtype=torch.uint8, device="cuda")
    lv = [dict(n_voxels=8, out_offset=0, byte_offset=0, bits=r, i_min=n_nodes - 2)]   # i_min + 3 > last node
    g.colorize_packed(d, lv, nodes, out)
    torch.cuda.synchronize()
    code = oracle.to_rgba8(nodes.cpu().numpy().astype(np.float64))
    assert np.array_equal(out.cpu().numpy(), code[np.minimum(n_nodes - 2 + want, n_nodes - 1)])
