"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element.

Tolerances (BASELINE.json north_star): leaves bit-exact; fp32 node colours max-abs <= 1e-5 against
the same-graph oracle; RGBA8 equal to the oracle's code except where the oracle value lies within
255 * 1e-5 of a rounding boundary (then +-1 LSB); fp16 within 1 fp16 ulp of RN(oracle).
"""
import numpy as np
import pytest

import oracle
from paper_2009_02702_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-5


@pytest.fixture(scope="module")
def mg():
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2009_02702_b200 import mg as _mg
    torch.cuda.set_device(0)
    return _mg


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _propagate(mg, a, b, w, off, n_leaves, tf, flags=0, host_tf=False):
    g = mg.Graph(a, b, w, n_leaves, level_offsets=off, flags=flags)
    n = g.info.n_nodes
    out = torch.full((n, 4), float("nan"), dtype=torch.float32, device="cuda")
    if host_tf:
        g.propagate_host(np.ascontiguousarray(tf, dtype=np.float32), out)
    else:
        g.propagate(_dev(tf.astype(np.float32)), out)
    torch.cuda.synchronize()
    return g, out


def _check_nodes(got, a, b, w, n_leaves, tf, perm=None):
    ref = oracle.graph_eval(a, b, w, n_leaves, tf.astype(np.float64))
    got = got.cpu().numpy()
    if perm is not None:
        got = got[perm]                       # got_in_old_numbering[old] = got[new_of_old[old]]
    assert np.array_equal(got[:n_leaves].view(np.uint32), tf.astype(np.float32).view(np.uint32)), "leaves not bit-exact"
    err = np.abs(got.astype(np.float64) - ref).max()
    assert err <= TOL, err
    return ref


# level-size profiles: all-tail, big levels only, big then a long small tail, ragged (non multiple
# of 4) sizes, tail exceeding the shared-memory mirror
PROFILES = {
    "tiny_all_tail": [16, 40, 20, 9, 3, 1],
    "fig_like_single_level": [4, 3],
    "big_levels": [1000, 30001, 20003, 9001],
    "big_then_tail": [353, 50001, 20002, 9003, 4001, 1200, 333, 77, 20, 6, 2, 1],
    "tail_over_smem": [64, 20000, 8000, 7000, 6000, 3000, 10],
    "ragged_starts": [3, 8193, 8195, 8197, 9001],
}


@pytest.mark.parametrize("name", list(PROFILES))
def test_propagate_matches_oracle(mg, name):
    sizes = PROFILES[name]
    a, b, w, off = synth.random_dag_levels(sizes, seed=list(PROFILES).index(name) + 7)
    tf = synth.random_tf(sizes[0], 40)
    g, out = _propagate(mg, a, b, w, off, sizes[0], tf)
    info = g.info
    assert info.depth == len(sizes) - 1 and info.n_nodes == sum(sizes)
    _check_nodes(out, a, b, w, sizes[0], tf)
    g.close()


def test_propagate_leaves_only_graph(mg):
    a = np.zeros(5, dtype=np.uint32)
    tf = synth.random_tf(5, 41)
    g, out = _propagate(mg, a, a, np.zeros(5, dtype=np.float32), [0, 5], 5, tf)
    assert np.array_equal(out.cpu().numpy(), tf)


def test_fig2_graph_on_gpu(mg, golden_dir):
    """Fig. 2 (L103-L118) through the CUDA path: root = 0.1 T1 + 0.2 T2 + 0.3 T3 + 0.4 T4."""
    a = np.array([0, 0, 0, 0, 0, 2, 3], dtype=np.uint32)
    b = np.array([0, 0, 0, 0, 1, 4, 5], dtype=np.uint32)
    w = np.array([0, 0, 0, 0, 2 / 3, 1 / 2, 3 / 5], dtype=np.float32)
    tf = synth.random_tf(4, 42)
    g, out = _propagate(mg, a, b, w, [0, 4, 5, 6, 7], 4, tf)
    root = out.cpu().numpy()[6].astype(np.float64)
    assert np.abs(root - np.array([0.1, 0.2, 0.3, 0.4]) @ tf.astype(np.float64)).max() < 1e-6


def test_propagate_host_tf_and_repeat_updates(mg):
    sizes = PROFILES["big_then_tail"]
    a, b, w, off = synth.random_dag_levels(sizes, seed=3)
    g = mg.Graph(a, b, w, sizes[0], level_offsets=off)
    out = torch.zeros((sum(sizes), 4), dtype=torch.float32, device="cuda")
    for upd in range(3):                                     # consecutive TF updates (config 2 style)
        tf = synth.random_tf(sizes[0], 43, update=upd)
        pinned = torch.from_numpy(tf).pin_memory()
        g.propagate_host(pinned, out)
        torch.cuda.synchronize()
        _check_nodes(out, a, b, w, sizes[0], tf)


def test_relabel_flag_permutes_and_preserves_values(mg):
    """A children-before-parents graph whose levels are interleaved (builder order): MG_RELABEL must
    produce a bijection that keeps leaves, makes levels contiguous and preserves every node value."""
    sizes = [37, 9000, 30000, 5000, 700, 90, 11, 2]
    a, b, w, off = synth.random_dag_levels(sizes, seed=9)
    n = a.size
    nl = sizes[0]
    # interleave the levels: sort by level + noise in [0, 0.999) -- a parent (level >= child's + 1)
    # still sorts after both of its children
    lev = np.repeat(np.arange(len(sizes)), sizes)
    key = lev[nl:] + synth.uniform01(9, 50, np.arange(n - nl, dtype=np.uint64)).astype(np.float64) * 0.999
    order = np.concatenate([np.arange(nl), nl + np.argsort(key, kind="stable")])   # new position -> orig id
    pos = np.empty(n, dtype=np.int64)
    pos[order] = np.arange(n)
    a2 = pos[a[order]].astype(np.uint32)
    b2 = pos[b[order]].astype(np.uint32)
    w2 = w[order]
    a2[:nl] = 0
    b2[:nl] = 0
    assert (a2[nl:] < np.arange(nl, n)).all() and (b2[nl:] < np.arange(nl, n)).all()
    tf = synth.random_tf(nl, 44)
    g, out = _propagate(mg, a2, b2, w2, None, nl, tf, flags=mg.MG_RELABEL)
    perm = g.node_permutation().astype(np.int64)
    assert np.array_equal(np.sort(perm), np.arange(n)) and np.array_equal(perm[:nl], np.arange(nl))
    offs = g.level_offsets()
    olev, depth = oracle.topo_levels(a2, b2, nl)
    assert g.info.depth == depth and g.info.relabelled == 1
    new_lev = np.searchsorted(offs, perm, side="right") - 1
    assert np.array_equal(new_lev, olev)                     # levels contiguous in the new numbering
    _check_nodes(out, a2, b2, w2, nl, tf, perm=perm)
    # device-side index relabelling
    idx = synth.random_node_idx(10007, n, 45)
    d = _dev(idx)
    g.relabel_indices(d, idx.size)
    torch.cuda.synchronize()
    assert np.array_equal(d.cpu().numpy(), perm[idx].astype(np.uint32))


def _rgba8_ok(got_u8, ref_c):
    """Equal to the oracle's code, or +-1 where the oracle value is within 255e-5 of a boundary."""
    code = oracle.to_rgba8(ref_c).astype(np.int64)
    got = got_u8.astype(np.int64)
    diff = got - code
    if not diff.any():
        return True
    scaled = np.clip(ref_c, 0.0, 1.0) * 255.0
    near = np.abs(scaled - np.floor(scaled) - 0.5) <= 255 * TOL + 1e-4   # + fp32 product rounding
    return bool(((diff == 0) | ((np.abs(diff) == 1) & near)).all())


def _f16_ok(got_f16, ref_c):
    ref = oracle.to_rgba16f(ref_c)
    gi = got_f16.view(np.int16).astype(np.int64)
    ri = ref.view(np.int16).astype(np.int64)
    return bool((np.abs(gi - ri) <= 1).all())                # non-negative values: ulp = bit distance


@pytest.mark.parametrize("reuse", [False, True], ids=["derive", "from_last_propagate"])
@pytest.mark.parametrize("n_vox", [0, 1, 3, 5, 2048, 2049, 123457, 1 << 21])
@pytest.mark.parametrize("fmt_name", ["RGBA8", "RGBA16F", "BOTH"])
def test_colorize_matches_oracle(mg, n_vox, fmt_name, reuse):
    sizes = PROFILES["big_then_tail"]
    a, b, w, off = synth.random_dag_levels(sizes, seed=5)
    tf = synth.random_tf(sizes[0], 46)
    g, nodes = _propagate(mg, a, b, w, off, sizes[0], tf)
    ref_nodes = oracle.graph_eval(a, b, w, sizes[0], tf.astype(np.float64))
    idx = synth.random_node_idx(max(n_vox, 1), a.size, 47)[:n_vox]
    d_idx = _dev(idx) if n_vox else torch.zeros(1, dtype=torch.int32, device="cuda")
    ref = oracle.lookup(idx, ref_nodes) if n_vox else np.zeros((0, 4))
    fmt = getattr(mg, "MG_" + fmt_name)
    out8 = torch.full((max(n_vox, 1), 4), 7, dtype=torch.uint8, device="cuda")
    out16 = torch.full((max(n_vox, 1), 4), 7, dtype=torch.float16, device="cuda")
    launches0 = mg.kernel_launch_count()
    if fmt_name == "RGBA8":
        g.colorize(d_idx, n_vox, nodes, out8, fmt=fmt, mip_level=0, from_last_propagate=reuse)
    elif fmt_name == "RGBA16F":
        g.colorize(d_idx, n_vox, nodes, out16, fmt=fmt, mip_level=0, from_last_propagate=reuse)
    else:
        g.colorize(d_idx, n_vox, nodes, out8, out16, fmt=fmt, mip_level=0, from_last_propagate=reuse)
    torch.cuda.synchronize()
    if n_vox and n_vox % 4 == 0:                             # aligned body only: the flag saves exactly the conversion kernel
        assert mg.kernel_launch_count() - launches0 == (1 if reuse else 2)
    if n_vox == 0:
        return
    if fmt_name in ("RGBA8", "BOTH"):
        assert _rgba8_ok(out8.cpu().numpy()[:n_vox], ref)
    if fmt_name in ("RGBA16F", "BOTH"):
        assert _f16_ok(out16.cpu().numpy()[:n_vox], ref)


@pytest.mark.parametrize("fmt_name", ["RGBA8", "RGBA16F", "BOTH"])
@pytest.mark.parametrize("tile_bytes", [40000, 90000, 200000, 333333])
def test_colorize_tiled_palette_matches_oracle(mg, fmt_name, tile_bytes, monkeypatch):
    """An RGBA8 palette larger than the L2 serves is gathered tile by tile, one sweep over the indices per tile
    (include/mg.h, mg_colorize).  MG_COLORIZE_TILE_BYTES shrinks the tile so that an 84,999-node palette (340 KB)
    takes 4, 2 and 2 sweeps (and, at 40,000 B, the single sweep again: more than 4 tiles); ragged head / tail, an
    output pre-filled with garbage, every voxel against the oracle.  fp16 always takes one sweep."""
    monkeypatch.setenv("MG_COLORIZE_TILE_BYTES", str(tile_bytes))
    sizes = PROFILES["big_then_tail"]
    a, b, w, off = synth.random_dag_levels(sizes, seed=5)
    tf = synth.random_tf(sizes[0], 46)
    g, nodes = _propagate(mg, a, b, w, off, sizes[0], tf)
    ref_nodes = oracle.graph_eval(a, b, w, sizes[0], tf.astype(np.float64))
    n_vox = 400003
    idx = synth.random_node_idx(n_vox + 3, a.size, 147)
    idx[3:40] = np.arange(37) * (a.size // 37)                # one vector per combination of tiles, more or less
    d_idx = _dev(idx)
    ref = oracle.lookup(idx[3:], ref_nodes)
    out8 = torch.full((n_vox + 3, 4), 0xCD, dtype=torch.uint8, device="cuda")
    out16 = torch.full((n_vox + 3, 4), float("nan"), dtype=torch.float16, device="cuda")
    fmt = getattr(mg, "MG_" + fmt_name)
    launches0 = mg.kernel_launch_count()
    args = {"RGBA8": (out8[3:],), "RGBA16F": (out16[3:],), "BOTH": (out8[3:], out16[3:])}[fmt_name]
    g.colorize(d_idx[3:], n_vox, nodes, *args, fmt=fmt, from_last_propagate=True)
    torch.cuda.synchronize()
    n_sweeps = mg.kernel_launch_count() - launches0 - 2      # head + tail scalar launches
    t8 = -(-a.size * 4 // tile_bytes)
    t8 = t8 if 2 <= t8 <= 4 else 1
    want = {"RGBA8": t8, "RGBA16F": 1, "BOTH": 1 if t8 == 1 else t8 + 1}[fmt_name]
    assert n_sweeps == want, (n_sweeps, want)
    if fmt_name in ("RGBA8", "BOTH"):
        assert _rgba8_ok(out8.cpu().numpy()[3:], ref) and (out8.cpu().numpy()[:3] == 0xCD).all()
    if fmt_name in ("RGBA16F", "BOTH"):
        assert _f16_ok(out16.cpu().numpy()[3:], ref)
    g.close()


@pytest.mark.parametrize("shift_idx,shift_out", [(1, 1), (3, 3), (2, 0), (1, 2)])
def test_colorize_unaligned_views(mg, shift_idx, shift_out):
    """Per-level sub-buffers of a concatenated mipmap start at arbitrary voxels: same shift -> vector
    body with ragged head/tail; different shifts -> scalar path.  Neighbouring voxels are untouched."""
    sizes = [50, 9000, 100, 5]
    a, b, w, off = synth.random_dag_levels(sizes, seed=6)
    tf = synth.random_tf(50, 48)
    g, nodes = _propagate(mg, a, b, w, off, 50, tf)
    ref_nodes = oracle.graph_eval(a, b, w, 50, tf.astype(np.float64))
    n = 10001
    idx = synth.random_node_idx(n + 8, a.size, 49)
    d_idx = _dev(idx)
    out8 = torch.full((n + 8, 4), 9, dtype=torch.uint8, device="cuda")
    g.colorize(d_idx[shift_idx:], n, nodes, out8[shift_out:], fmt=mg.MG_RGBA8, mip_level=3)
    torch.cuda.synchronize()
    got = out8.cpu().numpy()
    assert _rgba8_ok(got[shift_out:shift_out + n], oracle.lookup(idx[shift_idx:shift_idx + n], ref_nodes))
    assert (got[:shift_out] == 9).all() and (got[shift_out + n:] == 9).all()


def test_colorize_foreign_palette_and_force_convert(mg):
    """node_rgba that did not come from mg_propagate (or was edited) is converted by the call itself: that is the
    default; MG_FORCE_CONVERT (the pre-contract spelling) is still accepted and means the same."""
    sizes = [8, 100, 10]
    a, b, w, off = synth.random_dag_levels(sizes, seed=8)
    g = mg.Graph(a, b, w, 8, level_offsets=off)
    n = sum(sizes)
    pal = synth.random_tf(n, 51) * 1.4 - 0.2                  # includes values outside [0,1] -> clamp
    pal[3] = [np.nan, 2.0, -1.0, 0.5]
    d_pal = _dev(pal)
    idx = synth.random_node_idx(5000, n, 52)
    idx[:4] = 3
    out8 = torch.zeros((5000, 4), dtype=torch.uint8, device="cuda")
    g.colorize(_dev(idx), 5000, d_pal, out8, fmt=mg.MG_RGBA8)
    torch.cuda.synchronize()
    ref = oracle.to_rgba8(pal.astype(np.float64))[idx]        # same fp32 values: exact equality
    assert np.array_equal(out8.cpu().numpy(), ref)
    assert out8.cpu().numpy()[0].tolist() == [0, 255, 0, 128]
    d_pal[5] = 0.25                                           # edit in place, same pointer
    pal[5] = 0.25
    for extra in (0, mg.MG_FORCE_CONVERT):
        out8.zero_()
        g.colorize(_dev(idx), 5000, d_pal, out8, fmt=mg.MG_RGBA8 | extra)
        torch.cuda.synchronize()
        assert np.array_equal(out8.cpu().numpy(), oracle.to_rgba8(pal.astype(np.float64))[idx])
    with pytest.raises(mg.MgError) as e:                      # never propagated into: nothing to reuse
        g.colorize(_dev(idx), 5000, d_pal, out8, fmt=mg.MG_RGBA8, from_last_propagate=True)
    assert e.value.code == mg.MG_ERR_INVALID_ARG


def test_palette_contract(mg):
    """include/mg.h, mg_colorize: the default derives the palettes from node_rgba as it is on the stream; the 8/16-bit
    palettes of the last mg_propagate are gathered only under MG_PALETTE_FROM_LAST_PROPAGATE, which the library
    refuses whenever it can see that they no longer mirror node_rgba (the vec4 entry per node is THE
    palette)."""
    sizes = PROFILES["big_then_tail"]
    a, b, w, off = synth.random_dag_levels(sizes, seed=31)
    nl, n = sizes[0], sum(sizes)
    g = mg.Graph(a, b, w, nl, level_offsets=off)
    idx = synth.random_node_idx(40000, n, 70)
    d_idx = _dev(idx)
    out8 = torch.zeros((idx.size, 4), dtype=torch.uint8, device="cuda")
    X = torch.zeros((n, 4), dtype=torch.float32, device="cuda")
    tf1, tf2 = synth.random_tf(nl, 71), synth.random_tf(nl, 72)
    ref1 = oracle.graph_eval(a, b, w, nl, tf1.astype(np.float64))
    ref2 = oracle.graph_eval_attr(a, b, w, nl, tf2.astype(np.float64))

    def col(**kw):
        out8.zero_()
        g.colorize(d_idx, idx.size, X, out8, fmt=mg.MG_RGBA8, **kw)
        torch.cuda.synchronize()
        return out8.cpu().numpy()

    # (1) propagate(X) -> propagate_attr(X, C = 4) -> colorize(X): the colours of the SECOND call
    g.propagate(_dev(tf1), X)
    assert _rgba8_ok(col(from_last_propagate=True), oracle.lookup(idx, ref1))
    g.propagate_attr(_dev(tf2), X, 4)
    assert _rgba8_ok(col(), oracle.lookup(idx, ref2))
    with pytest.raises(mg.MgError) as e:                      # the library saw the write: reuse refused
        col(from_last_propagate=True)
    assert e.value.code == mg.MG_ERR_INVALID_ARG
    # (2) an attr write that only overlaps the palette buffer (other base pointer) is seen too
    g.propagate(_dev(tf1), X)
    g.propagate_attr(_dev(tf2[:, :1].copy()), X.view(-1)[8:8 + n], 1)
    with pytest.raises(mg.MgError):
        col(from_last_propagate=True)
    # (3) an unflagged colourise re-derives the palettes from whatever it is given: reuse refused afterwards
    g.propagate(_dev(tf1), X)
    other = _dev(np.ascontiguousarray(ref2, dtype=np.float32))
    out8.zero_()
    g.colorize(d_idx, idx.size, other, out8, fmt=mg.MG_RGBA8)
    torch.cuda.synchronize()
    assert _rgba8_ok(out8.cpu().numpy(), oracle.lookup(idx, ref2))
    with pytest.raises(mg.MgError):
        col(from_last_propagate=True)
    # (4) a foreign pointer is refused; so is the flag together with MG_FORCE_CONVERT
    g.propagate(_dev(tf1), X)
    with pytest.raises(mg.MgError):
        g.colorize(d_idx, idx.size, other, out8, fmt=mg.MG_RGBA8, from_last_propagate=True)
    with pytest.raises(mg.MgError):
        g.colorize(d_idx, idx.size, X, out8, fmt=mg.MG_RGBA8 | mg.MG_FORCE_CONVERT, from_last_propagate=True)
    # (5) the caller's own in-place edit: the default shows it; the flag is the caller's statement that there
    # was none, so it shows the propagated colours (documented behaviour, not an error the library can detect)
    g.propagate(_dev(tf1), X)
    X[idx[0]] = torch.tensor([1.0, 0.0, 1.0, 0.0], device="cuda")
    assert col()[0].tolist() == [255, 0, 255, 0]
    g.propagate(_dev(tf1), X)
    X[idx[0]] = torch.tensor([1.0, 0.0, 1.0, 0.0], device="cuda")
    assert _rgba8_ok(col(from_last_propagate=True), oracle.lookup(idx, ref1))
    g.close()


def test_no_palettes_graph(mg):
    """MG_NO_PALETTES: mg_propagate writes node_rgba only; colourise derives its palettes; the reuse flag is refused."""
    sizes = PROFILES["big_then_tail"]
    a, b, w, off = synth.random_dag_levels(sizes, seed=32)
    tf = synth.random_tf(sizes[0], 73)
    g, nodes = _propagate(mg, a, b, w, off, sizes[0], tf, flags=mg.MG_NO_PALETTES)
    ref = _check_nodes(nodes, a, b, w, sizes[0], tf)
    idx = synth.random_node_idx(30001, a.size, 74)
    out8 = torch.zeros((idx.size, 4), dtype=torch.uint8, device="cuda")
    out16 = torch.zeros((idx.size, 4), dtype=torch.float16, device="cuda")
    g.colorize(_dev(idx), idx.size, nodes, out8, out16, fmt=mg.MG_BOTH)
    torch.cuda.synchronize()
    assert _rgba8_ok(out8.cpu().numpy(), oracle.lookup(idx, ref)) and _f16_ok(out16.cpu().numpy(), oracle.lookup(idx, ref))
    with pytest.raises(mg.MgError):
        g.colorize(_dev(idx), idx.size, nodes, out8, fmt=mg.MG_RGBA8, from_last_propagate=True)
    nodes2 = torch.zeros_like(nodes)
    out_dev = torch.zeros((idx.size, 4), dtype=torch.uint8, device="cuda")
    g.tf_update_host(torch.from_numpy(tf).pin_memory(), nodes2, _dev(idx), idx.size, out_dev, None, fmt=mg.MG_RGBA8)
    torch.cuda.synchronize()
    assert _rgba8_ok(out_dev.cpu().numpy(), oracle.lookup(idx, ref))
    g.close()


def test_tf_update_host_end_to_end(mg):
    sizes = PROFILES["big_then_tail"]
    a, b, w, off = synth.random_dag_levels(sizes, seed=10)
    g = mg.Graph(a, b, w, sizes[0], level_offsets=off)
    n = sum(sizes)
    n_vox = 300001
    idx = synth.random_node_idx(n_vox, n, 53)
    d_idx = _dev(idx)
    nodes = torch.zeros((n, 4), dtype=torch.float32, device="cuda")
    out_dev = torch.zeros((n_vox, 4), dtype=torch.uint8, device="cuda")
    out_host = torch.zeros((n_vox, 4), dtype=torch.uint8).pin_memory()
    tf = synth.random_tf(sizes[0], 54)
    tf_host = torch.from_numpy(tf).pin_memory()
    g.tf_update_host(tf_host, nodes, d_idx, n_vox, out_dev, out_host, fmt=mg.MG_RGBA8)
    torch.cuda.synchronize()
    ref_nodes = _check_nodes(nodes, a, b, w, sizes[0], tf)
    assert _rgba8_ok(out_host.numpy(), oracle.lookup(idx, ref_nodes))
    assert np.array_equal(out_host.numpy(), out_dev.cpu().numpy())


def test_check_indices_counts_out_of_range_entries(mg):
    a, b, w, off = synth.random_dag_levels([4, 6, 2], seed=12)
    g = mg.Graph(a, b, w, 4, level_offsets=off)
    idx = synth.random_node_idx(100003, 12, 81)
    assert g.check_indices(_dev(idx), idx.size) == 0
    idx[[0, 5, 100002]] = [12, 0xFFFFFFFF, 4000]
    assert g.check_indices(_dev(idx), idx.size) == 3
    assert g.check_indices(_dev(idx)[1:], idx.size - 1) == 2 and g.check_indices(_dev(idx), 0) == 0


def test_error_paths(mg):
    a, b, w, off = synth.random_dag_levels([4, 6, 2], seed=11)
    g = mg.Graph(a, b, w, 4, level_offsets=off)
    nodes = torch.zeros((12, 4), dtype=torch.float32, device="cuda")
    tf = torch.zeros((4, 4), dtype=torch.float32, device="cuda")
    with pytest.raises(mg.MgError) as e:
        g.propagate(tf, nodes.view(-1)[1:].data_ptr())        # misaligned node_rgba
    assert e.value.code == mg.MG_ERR_INVALID_ARG
    with pytest.raises(mg.MgError):
        g.colorize(tf, 4, nodes, tf, fmt=0)
    with pytest.raises(mg.MgError) as e:                      # level not max+1
        mg.Graph(a, b, w, 4, level_offsets=[0, 4, 5, 12])
    assert e.value.code == mg.MG_ERR_INVALID_GRAPH
    bad = a.copy()
    bad[5] = b[5]
    with pytest.raises(mg.MgError):
        mg.Graph(bad, b, w, 4, level_offsets=off)
    assert mg.kernel_launch_count() > 0


@pytest.mark.parametrize("reuse", [True, False], ids=["from_last_propagate", "derive"])
@pytest.mark.parametrize("profile,n_vox", [("big_then_tail", 200003), ("big_levels", 3000001), ("tiny_all_tail", 4099)])
def test_back_to_back_updates_without_sync(mg, profile, n_vox, reuse):
    """Programmatic dependent launch lets a kernel become resident before its predecessor has finished
    (griddepcontrol.wait orders them).  Many TF updates enqueued back to back, each with its own TF and
    its own output buffers, no host synchronisation in between: every update must see exactly its own
    palette (no stale cached colours from the previous update, no early reads)."""
    sizes = PROFILES[profile]
    a, b, w, off = synth.random_dag_levels(sizes, seed=21)
    g = mg.Graph(a, b, w, sizes[0], level_offsets=off)
    n = sum(sizes)
    n_upd = 12
    idx = synth.random_node_idx(n_vox, n, 60)
    d_idx = _dev(idx)
    tfs = [synth.random_tf(sizes[0], 61, update=u) for u in range(n_upd)]
    d_tfs = [_dev(t) for t in tfs]
    nodes = torch.zeros((n, 4), dtype=torch.float32, device="cuda")          # ONE palette buffer, reused
    outs = [torch.zeros((n_vox, 4), dtype=torch.uint8, device="cuda") for _ in range(n_upd)]
    snaps = [torch.zeros((n, 4), dtype=torch.float32, device="cuda") for _ in range(n_upd)]
    st = torch.cuda.current_stream().cuda_stream
    for u in range(n_upd):
        g.propagate(d_tfs[u], nodes, st)
        g.colorize(d_idx, n_vox, nodes, outs[u], fmt=mg.MG_RGBA8, stream=st, from_last_propagate=reuse)
        snaps[u].copy_(nodes)                                                 # stream-ordered snapshot
    torch.cuda.synchronize()
    for u in range(n_upd):
        ref = oracle.graph_eval(a, b, w, sizes[0], tfs[u].astype(np.float64))
        got = snaps[u].cpu().numpy()
        assert np.array_equal(got[:sizes[0]], tfs[u])
        assert np.abs(got - ref).max() <= TOL, u
        assert _rgba8_ok(outs[u].cpu().numpy(), oracle.lookup(idx, ref)), u


def test_tail_plan_limits(mg):
    """The single-CTA tail takes the longest suffix of levels that fits its shared-memory budget."""
    sizes = [500, 30000, 9000, 8000, 3000, 900, 200, 40, 8, 1]
    a, b, w, off = synth.random_dag_levels(sizes, seed=22)
    tf = synth.random_tf(sizes[0], 62)
    g, out = _propagate(mg, a, b, w, off, sizes[0], tf)
    info = g.info
    assert 2 <= info.first_fused_level <= 5 and info.n_launches_propagate == info.first_fused_level
    _check_nodes(out, a, b, w, sizes[0], tf)
