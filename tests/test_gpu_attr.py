"""NEXT-1: mg_propagate_attr (any numeric attribute, C channels) against the CPU oracle.

Tolerance: the same as mg_propagate (same per-channel fp32 arithmetic): leaves bit-exact, max-abs
<= 1e-5 * max|attr| against oracle.graph_eval_attr on the same graph.
"""
import numpy as np
import pytest

import oracle
from paper_2009_02702_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-5

PROFILES = {
    "all_tail": [16, 40, 20, 9, 3, 1],
    "single_level": [4, 3],
    "big_levels_only": [1000, 30001, 20003, 9001],
    "big_then_tail": [353, 50001, 20002, 9003, 4001, 1200, 333, 77, 20, 6, 2, 1],
    "ragged": [3, 8193, 8195, 4097, 9001, 5],
}


@pytest.fixture(scope="module")
def mg():
    if not torch.cuda.is_available():
        pytest.fail("the gpu-marked tests need a CUDA device (no CPU fallback exists)")
    from paper_2009_02702_b200 import mg as _mg
    torch.cuda.set_device(0)
    return _mg


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("name", list(PROFILES))
@pytest.mark.parametrize("n_ch", [1, 2, 3, 4, 6, 8, 16, 64])
def test_propagate_attr_matches_oracle(mg, name, n_ch):
    sizes = PROFILES[name]
    a, b, w, off = synth.random_dag_levels(sizes, seed=50 + list(PROFILES).index(name))
    attr = synth.random_attr(sizes[0], n_ch, seed=60, lo=-2.0, hi=3.0)
    g = mg.Graph(a, b, w, sizes[0], level_offsets=off)
    n = sum(sizes)
    out = torch.full((n, n_ch), float("nan"), dtype=torch.float32, device="cuda")
    g.propagate_attr(_dev(attr), out, n_ch)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    ref = oracle.graph_eval_attr(a, b, w, sizes[0], attr.astype(np.float64))
    assert np.array_equal(got[:sizes[0]].view(np.uint32), attr.view(np.uint32)), "leaves not bit-exact"
    err = np.abs(got.astype(np.float64) - ref).max()
    assert err <= TOL * 3.0, err
    g.close()


def test_attr_4_channels_equals_mg_propagate_bit_for_bit(mg):
    """C = 4 is the RGBA path: same arithmetic, so the two kernels agree bit for bit."""
    sizes = PROFILES["big_then_tail"]
    a, b, w, off = synth.random_dag_levels(sizes, seed=70)
    tf = synth.random_tf(sizes[0], 71)
    g = mg.Graph(a, b, w, sizes[0], level_offsets=off)
    n = sum(sizes)
    c1 = torch.empty((n, 4), dtype=torch.float32, device="cuda")
    c2 = torch.empty((n, 4), dtype=torch.float32, device="cuda")
    d_tf = _dev(tf)
    g.propagate(d_tf, c1)
    g.propagate_attr(d_tf, c2, 4)
    torch.cuda.synchronize()
    assert torch.equal(c1.view(torch.int32), c2.view(torch.int32))
    g.close()


def test_opacity_only_equals_alpha_channel_of_rgba(mg):
    """L271 (i)-(ii): propagating the TF's opacity alone gives the A channel of the RGBA palette."""
    sizes = PROFILES["big_then_tail"]
    a, b, w, off = synth.random_dag_levels(sizes, seed=72)
    tf = synth.random_tf(sizes[0], 73, alpha_zero_frac=0.3)
    g = mg.Graph(a, b, w, sizes[0], level_offsets=off)
    n = sum(sizes)
    rgba = torch.empty((n, 4), dtype=torch.float32, device="cuda")
    alpha = torch.empty((n, 1), dtype=torch.float32, device="cuda")
    g.propagate(_dev(tf), rgba)
    g.propagate_attr(_dev(tf[:, 3:4].copy()), alpha, 1)
    torch.cuda.synchronize()
    assert torch.equal(rgba[:, 3].contiguous().view(torch.int32), alpha[:, 0].contiguous().view(torch.int32))
    g.close()


def test_batched_tfs_and_relabelled_graph(mg):
    """K = 3 transfer functions as 12 channels on a graph loaded with MG_RELABEL (library numbering)."""
    sizes = [37, 6000, 5000, 900, 100, 10, 1]
    a, b, w, off = synth.random_dag_levels(sizes, seed=74)
    g = mg.Graph(a, b, w, sizes[0], flags=mg.MG_RELABEL)
    perm = g.node_permutation().astype(np.int64)
    tfs = [synth.random_tf(sizes[0], 75, update=k) for k in range(3)]
    attr = np.concatenate(tfs, axis=1)
    n = sum(sizes)
    out = torch.empty((n, 12), dtype=torch.float32, device="cuda")
    g.propagate_attr(_dev(attr), out, 12)
    torch.cuda.synchronize()
    got = out.cpu().numpy()[perm]
    for k in range(3):
        ref = oracle.graph_eval(a, b, w, sizes[0], tfs[k].astype(np.float64))
        assert np.abs(got[:, 4 * k:4 * k + 4] - ref).max() <= TOL
    g.close()


def test_attr_unaligned_views_and_repeat_without_sync(mg):
    """Buffers offset by 4 bytes take the scalar path; two updates enqueued back to back (PDL chain)
    must each see their own leaf values."""
    sizes = PROFILES["big_then_tail"]
    a, b, w, off = synth.random_dag_levels(sizes, seed=76)
    g = mg.Graph(a, b, w, sizes[0], level_offsets=off)
    n = sum(sizes)
    n_ch = 4
    base_leaf = torch.empty(sizes[0] * n_ch + 1, dtype=torch.float32, device="cuda")
    base_out = torch.empty(n * n_ch + 1, dtype=torch.float32, device="cuda")
    leaf = base_leaf[1:].view(sizes[0], n_ch)
    out = base_out[1:].view(n, n_ch)
    at0 = synth.random_attr(sizes[0], n_ch, seed=77)
    at1 = synth.random_attr(sizes[0], n_ch, seed=78)
    leaf.copy_(_dev(at0))
    g.propagate_attr(leaf, out, n_ch)
    snap = out.clone()
    leaf.copy_(_dev(at1))
    g.propagate_attr(leaf, out, n_ch)
    torch.cuda.synchronize()
    for at, got in ((at0, snap), (at1, out)):
        ref = oracle.graph_eval_attr(a, b, w, sizes[0], at.astype(np.float64))
        assert np.abs(got.cpu().numpy() - ref).max() <= TOL
    g.close()


def test_attr_error_paths(mg):
    a, b, w, off = synth.random_dag_levels([4, 3], seed=79)
    g = mg.Graph(a, b, w, 4, level_offsets=off)
    leaf = torch.zeros((4, 4), dtype=torch.float32, device="cuda")
    out = torch.zeros((7, 4), dtype=torch.float32, device="cuda")
    for args in ((None, out, 4), (leaf, None, 4), (leaf, out, 0), (leaf, out, mg.MG_MAX_ATTR_CHANNELS + 1), (out, out, 4)):
        with pytest.raises(mg.MgError) as e:
            g.propagate_attr(*args)
        assert e.value.code == mg.MG_ERR_INVALID_ARG
    g.close()
