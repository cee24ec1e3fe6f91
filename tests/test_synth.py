"""The seeded input generators: determinism, ranges and the structure DESIGN.md states."""
import numpy as np

from paper_2009_02702_b200 import synth


def test_splitmix64_published_vector():
    # first outputs of splitmix64 seeded with 0 (widely published test vector)
    s = np.uint64(0)
    assert int(synth.splitmix64(s)) == 0xE220A8397B1DCDAF
    assert int(synth.splitmix64(np.uint64(0x9E3779B97F4A7C15))) == 0x6E789E6AA1B965F4


def test_uniform01_range_and_exactness():
    u = synth.uniform01(7, 0, np.arange(100000, dtype=np.uint64))
    assert u.dtype == np.float32 and u.min() >= 0.0 and u.max() < 1.0
    assert ((u * (1 << 24)) % 1 == 0).all()
    assert abs(float(u.mean()) - 0.5) < 0.01


def test_tf_configs():
    tf = synth.random_tf(1182, 3, alpha_zero_frac=0.3)
    assert tf.shape == (1182, 4) and tf.dtype == np.float32
    frac = float((tf[:, 3] == 0).mean())
    assert 0.25 < frac < 0.35 and (tf[:, :3] > 0).mean() > 0.99      # only A is zeroed
    assert not np.array_equal(synth.random_tf(16, 1, update=0), synth.random_tf(16, 1, update=1))
    t0 = synth.random_tf(100, 4)
    t1 = synth.single_segment_update(t0, 4, 5)
    assert (t0 != t1).any(axis=1).sum() == 1


def test_config_tf_sequences_are_the_ones_baseline_names():
    """Config 2: 100 consecutive random TFs; config 4: update u is update u - 1 with one random segment re-drawn
    (BASELINE.json configs[1], configs[3]); Workload.tf(u) is that sequence, whatever order it is asked in."""
    from paper_2009_02702_b200.workload import Workload
    for cid, n_leaves in ((2, 353), (4, 15918)):
        w = Workload("t")
        w.cfg = dict(synth.CONFIGS[cid])
        w.n_leaves = n_leaves
        assert w.n_updates == 100
        last = w.tf(99)
        tfs = [w.tf(u) for u in range(100)]
        assert np.array_equal(tfs[99], last) and all(t.shape == (n_leaves, 4) and t.dtype == np.float32 for t in tfs)
        changed = [int((tfs[u] != tfs[u - 1]).any(axis=1).sum()) for u in range(1, 100)]
        if cid == 4:
            assert max(changed) == 1 and sum(changed) >= 95
            assert np.array_equal(tfs[7], synth.single_segment_update(tfs[6], 4, 7))
            tfs[3][0, 0] = 9.0                                                 # callers get copies
            assert w.tf(3)[0, 0] != 9.0
        else:
            assert min(changed) == n_leaves and len({t.tobytes() for t in tfs}) == 100
            assert np.array_equal(tfs[5], synth.random_tf(353, 2, update=5))


def test_config1_volume():
    c = synth.CONFIGS[1]
    S = synth.make_volume(c)
    assert S.shape == (64, 64, 64) and S.dtype == np.uint32
    assert np.unique(S).tolist() == list(range(16))
    seeds = synth.voronoi_seeds(c["dims"], 16, 1)
    assert len({tuple(p) for p in seeds.tolist()}) == 16
    for k, (x, y, z) in enumerate(seeds.tolist()):
        assert S[z, y, x] == k                                          # a seed owns its own voxel
    # crop evaluation equals the full volume
    crop = synth.make_volume(c, region=(10, 14, 20, 25, 30, 37))
    assert (crop == S[10:14, 20:25, 30:37]).all()


def test_voronoi_anisotropy_and_jitter():
    c = synth.scaled_config(3, 1 / 32)
    S = synth.make_volume(c)
    assert S.shape == (9, 64, 64)
    # z-neighbours differ more often than x-neighbours (cells are 7x thinner in z, L277)
    assert (S[1:] != S[:-1]).mean() > 2 * (S[:, :, 1:] != S[:, :, :-1]).mean()
    c2 = synth.scaled_config(2, 1 / 24)
    Sj = synth.make_volume(c2)
    c2n = dict(c2, jitter=0)
    Sn = synth.make_volume(c2n)
    diff = (Sj != Sn).mean()
    assert 0.0 < diff < 0.5                                              # jitter roughens boundaries only


def test_cylinders_exact_and_background():
    c = synth.scaled_config(4, 1 / 8)
    p = synth.cylinder_params(c["dims"], 40, c["seed"])
    assert ((p[:, 6] >= 32) & (p[:, 6] <= 80) & (p[:, 7] >= 20) & (p[:, 7] <= 200)).all()
    n2 = (p[:, 3:6] ** 2).sum(axis=1)
    assert ((n2 > 0) & (n2 <= 1024 * 1024)).all()
    S = synth.cylinder_volume(c["dims"], p)
    assert S.max() <= 40 and (S == 0).mean() > 0.3
    crop = synth.cylinder_volume(c["dims"], p, region=(5, 30, 10, 50, 3, 40))
    assert (crop == S[5:30, 10:50, 3:40]).all()


def test_random_dag_structure():
    a, b, w, off = synth.random_dag(5000, 8, 64, 5)
    assert off[0] == 0 and off[1] == 64 and off[-1] == 5000
    for L in range(1, 8):
        lo, hi = int(off[L]), int(off[L + 1])
        assert (a[lo:hi] >= off[L - 1]).all() and (a[lo:hi] < lo).all()
        assert (b[lo:hi] < lo).all() and (a[lo:hi] != b[lo:hi]).all()
        assert (w[lo:hi] > 0).all() and (w[lo:hi] < 1).all()
    idx = synth.random_node_idx(1000, 5000, 5)
    assert idx.max() < 5000 and idx.dtype == np.uint32
