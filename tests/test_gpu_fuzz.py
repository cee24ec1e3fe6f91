"""Seeded random differential test of the whole device API against the oracle: random DAG shapes (level counts and
sizes chosen so that the per-level kernels, the single-CTA tail and their boundaries all occur), random leaf
attributes, random colourise sizes, the mixture table and the bit-packed path.  Tolerances as in the specific tests."""
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


def _rand(seed, stream, n, lo, hi):
    return (lo + synth.u64(seed, stream, np.arange(n, dtype=np.uint64)) % np.uint64(hi - lo + 1)).astype(np.int64)


def _shape(seed):
    depth = int(_rand(seed, 1, 1, 1, 14)[0])
    kind = int(_rand(seed, 2, 1, 0, 3)[0])
    n_leaves = int(_rand(seed, 3, 1, 2, 600)[0])
    sizes = [n_leaves]
    for L in range(depth):
        r = int(_rand(seed, 10 + L, 1, 0, 10 ** 6)[0])
        if kind == 0:
            s = 1 + r % 40                                                   # everything in the tail
        elif kind == 1:
            s = 8000 + r % 9000 if L < depth // 2 else 1 + r % 300          # big levels, then a tail
        elif kind == 2:
            s = 8185 + r % 16                                                # around the tail's 8192-node level limit
        else:
            s = 1 + r % 20000                                                # anything
        sizes.append(s)
    return sizes


@pytest.mark.parametrize("seed", range(24))
def test_random_graph_all_calls(mg, seed):
    sizes = _shape(1000 + seed)
    a, b, w, off = synth.random_dag_levels(sizes, seed=2000 + seed)
    nl, n = sizes[0], int(sum(sizes))
    g = mg.Graph(a, b, w, nl, level_offsets=off)
    dev = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()

    # propagate (a4, a5)
    tf = synth.random_tf(nl, 3000 + seed)
    nodes = torch.full((n, 4), float("nan"), dtype=torch.float32, device="cuda")
    g.propagate(dev(tf), nodes)
    ref = oracle.graph_eval(a, b, w, nl, tf.astype(np.float64))
    got = nodes.cpu().numpy()
    assert np.array_equal(got[:nl].view(np.uint32), tf.view(np.uint32))
    assert np.abs(got - ref).max() <= 1e-5

    # colourise (a6), uint32 and bit-packed, a random ragged size
    nv = int(_rand(seed, 40, 1, 1, 70000)[0])
    idx = synth.random_node_idx(nv, n, 4000 + seed)
    d_idx = dev(idx.view(np.int32))
    out = torch.zeros((nv, 4), dtype=torch.uint8, device="cuda")
    g.colorize(d_idx, nv, nodes, out)
    code = oracle.to_rgba8(ref)[idx].astype(np.int64)
    diff = np.abs(out.cpu().numpy().astype(np.int64) - code)
    assert diff.max() <= 1 and (diff != 0).mean() < 2e-3
    i_min, i_max = mg.index_range(d_idx, nv)
    assert (i_min, i_max) == oracle.index_range(idx)
    bits = mg.bits_per_voxel(i_min, i_max)
    assert bits == oracle.bits_per_voxel(i_min, i_max)
    packed = torch.zeros(mg.packed_stream_bytes(nv, bits), dtype=torch.uint8, device="cuda")
    mg.pack_indices(d_idx, nv, i_min, bits, packed)
    ref_stream = oracle.pack_level(idx, i_min, bits)
    assert np.array_equal(packed.cpu().numpy()[:ref_stream.size], ref_stream)
    out_p = torch.zeros_like(out)
    g.colorize_packed(packed, [dict(n_voxels=nv, out_offset=0, byte_offset=0, bits=bits, i_min=i_min)], nodes, out_p)
    assert torch.equal(out, out_p)

    # attributes (NEXT-1)
    C_ = int(_rand(seed, 41, 1, 1, 9)[0])
    attr = synth.random_attr(nl, C_, seed=5000 + seed, lo=-1.0, hi=2.0)
    xa = torch.full((n, C_), float("nan"), dtype=torch.float32, device="cuda")
    g.propagate_attr(dev(attr), xa, C_)
    refa = oracle.graph_eval_attr(a, b, w, nl, attr.astype(np.float64))
    assert np.abs(xa.cpu().numpy() - refa).max() <= 3e-5

    # mixture table (NEXT-4) on the smaller graphs (the oracle's table is dense)
    if n * nl <= 4_000_000:
        sg = (0.02 * synth.random_attr(n, 1, seed=6000 + seed).reshape(-1)).astype(np.float32)
        lut = g.mixture_lut(sg)
        rp, leaf, mu, dmu = lut.export()
        omu, odmu = oracle.mixture_lut(a, b, w.astype(np.float64), sg.astype(np.float64), nl)
        rows = np.repeat(np.arange(n), np.diff(rp).astype(np.int64))
        M, D = np.zeros_like(omu), np.zeros_like(odmu)
        M[rows, leaf] = mu
        D[rows, leaf] = dmu
        np.testing.assert_allclose(M, omu, rtol=1e-12)
        np.testing.assert_allclose(D, odmu, rtol=1e-12, atol=1e-300)
        lut.close()
    g.close()
